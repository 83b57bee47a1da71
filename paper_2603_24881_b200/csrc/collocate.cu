// Collocation kernel (Eq. 3; the work of Alg. 1, re-decomposed for B200).
//
// One warp per work item = one 4x4x4 grid block and a range of its visit list.  The warp is eight groups
// of four lanes; a group evaluates one (pair, block) visit at a time and a lane owns the slab of 4x4 grid
// points at its own n1, so the polynomial collapse in u1 and the Gaussian set-up are paid once per 16
// points (gpw_math.cuh, colloc_slab).  Every lane keeps its rho values (and, for DERIV, the gradient in
// grid-index components) in registers for the whole list; the eight groups are summed by a shuffle
// reduce-scatter and the block is written once (the theoretical minimum the paper aims at),
// with no per-point cross-thread reduction (the bottleneck of Alg. 1 l.11).  The next
// visit's pair record and polynomial are copied to shared memory with cp.async while the current visit
// is evaluated (two slots per group).
#include "gpw_kernels.cuh"

namespace gpw {
namespace {

constexpr int NGRP = 8;   // groups of 4 lanes per warp
constexpr int NWARP = 4;  // warps (work items) per CTA

// Shared-memory slot of one visit: the pair record (8 doubles) followed by the pair polynomial.
GPW_CX int slot_doubles(int lmax) { return 8 + ncoef_pad(lmax); }
// A group's two slots, padded so that consecutive groups start 16 bytes apart modulo the 128-byte bank
// row: the eight groups' broadcast reads of the same coefficient then hit eight different bank pairs.
GPW_CX int group_stride(int lmax) {
    int n = 2 * slot_doubles(lmax);
    while (n % 16 != 2) n += 2;
    return n;
}

struct ColCtx {
    const TaskK *tasks;
    const Visit *visits;   // already offset to the block's list
    const double *work;    // pair polynomials
    const double *gm;      // the level's metric Gm (constant bank)
    const long long *coef_base;   // the level's class offsets into the workspace (constant bank)
    double *slot;          // the group's two shared-memory slots
    int n1, n2, n3;        // stored index of the lane's slab corner
    int N0, N1, N2;
    int x;                 // lane within the group
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// The group's four lanes copy the pair record and polynomial of `task` (class L) into a slot (16 bytes per
// lane and trip).
__device__ __forceinline__ void stage_visit(const ColCtx &c, int L, int task, double *slot) {
    const int npad = ncoef_pad(L);
    const int nch = 4 + npad / 2;   // 16-byte chunks
    const char *src_k = reinterpret_cast<const char *>(c.tasks + task);
    const char *src_c = reinterpret_cast<const char *>(c.work + c.coef_base[L] + (long long)task * npad);
    for (int k = c.x; k < nch; k += 4)
        cp_async16(reinterpret_cast<char *>(slot) + 16 * k, k < 4 ? src_k + 16 * k : src_c + 16 * (k - 4));
    cp_async_commit();
}

// The item's visits in chunks of NGRP that never straddle an L segment (so the code path is warp-uniform).
// Lane l holds seg[l & 7] of the block; all lanes advance together.
struct ChunkIt {
    int L;
    unsigned base, hi;   // the chunk is [base, min(base + NGRP, hi)); hi = end of the segment inside the item
};
template <int LMAX>
__device__ __forceinline__ bool next_chunk(ChunkIt &it, unsigned it_lo, unsigned it_hi, unsigned myseg) {
    it.base += NGRP;
    while (it.L < 0 || it.base >= it.hi) {
        it.L++;
        if (it.L > LMAX) return false;
        it.base = max(it_lo, __shfl_sync(0xffffffffu, myseg, it.L));
        it.hi = min(it_hi, __shfl_sync(0xffffffffu, myseg, it.L + 1));
    }
    return true;
}

template <int L, int DERIV, bool ORTHO>
__device__ __forceinline__ void colloc_visit(const ColCtx &c, const Visit vi, const double *s, double (*acc)[16]) {
    const double ap = s[3];
    double q[6];
#pragma unroll
    for (int k = 0; k < 6; k++) q[k] = ap * c.gm[k];
    const double u1 = (double)(c.n1 + vi.s[0] * c.N0) - s[0];
    const double u20 = (double)(c.n2 + vi.s[1] * c.N1) - s[1];
    const double u30 = (double)(c.n3 + vi.s[2] * c.N2) - s[2];
    colloc_slab<L, DERIV, ORTHO>(s + 8, q, s[4], s[5], s[6], u1, u20, u30, acc);
}

// Sum an N-vector over the eight groups (lane bits 4, 8, 16); afterwards the lane holds N/8 sums,
// a[0 .. N/8) = total[off .. off + N/8).
template <int N>
__device__ __forceinline__ int group_reduce_scatter(double *a, int lane) {
    int off = 0;
#pragma unroll
    for (int step = 0; step < 3; step++) {
        const int bit = 16 >> step;
        const int half = N >> (step + 1);
        const bool up = lane & bit;
#pragma unroll
        for (int i = 0; i < half; i++) {
            const double send = up ? a[i] : a[i + half];
            const double keep = up ? a[i + half] : a[i];
            a[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
        off += up ? half : 0;
    }
    return off;
}

template <int DERIV, int LMAX, bool ORTHO>
__global__ void __launch_bounds__(128, DERIV ? 2 : 3) k_collocate(const __grid_constant__ GridParams P,
                                                                   const TaskK *__restrict__ tasks,
                                                                   const Visit *__restrict__ visits,
                                                                   const Item *__restrict__ items, int nitem,
                                                                   const double *__restrict__ coef) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int SLOT = slot_doubles(LMAX);
    constexpr int GSTRIDE = group_stride(LMAX);
    extern __shared__ __align__(16) double sm[];   // [NWARP][NGRP] x (two slots, padded to GSTRIDE)
    const int w = blockIdx.x * NWARP + (threadIdx.x >> 5);
    if (w >= nitem) return;
    const Item it = items[w];
    const LevelGeom &g = P.lev[it.level];
    const int lane = threadIdx.x & 31, grp = lane >> 2, x = lane & 3;
    const int T2 = g.T[2], T1 = g.T[1];
    const int b3 = it.tile % T2, b2 = (it.tile / T2) % T1, b1 = it.tile / (T2 * T1);
    ColCtx c;
    c.tasks = tasks;
    c.visits = visits + P.tile_base[it.level][it.tile];
    c.work = coef;
    c.gm = g.Gm;
    c.coef_base = P.coef_base[it.level];
    c.slot = sm + (size_t)((threadIdx.x >> 5) * NGRP + grp) * GSTRIDE;
    c.x = x;
    c.n1 = 4 * b1 + x; c.n2 = 4 * b2; c.n3 = 4 * b3;
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];
    const unsigned myseg = P.seg[it.level][(size_t)it.tile * 8 + (lane & 7)];

    double acc[NCOMP][16];
#pragma unroll
    for (int k = 0; k < NCOMP; k++)
#pragma unroll
        for (int i = 0; i < 16; i++) acc[k][i] = 0.0;

    // Software pipeline over the chunks, across L segments: the visit records of chunk k+2 are loaded and
    // the pair record + polynomial of chunk k+1 are copied to shared memory (cp.async) while chunk k is
    // evaluated.
    ChunkIt c0{-1, 0u, 0u};
    bool h0 = next_chunk<LMAX>(c0, it.lo, it.hi, myseg);
    ChunkIt c1 = c0;
    bool h1 = h0 && next_chunk<LMAX>(c1, it.lo, it.hi, myseg);
    Visit v0, v1;
    v0.task = 0; v0.s[0] = v0.s[1] = v0.s[2] = 0; v0.pad = 0;
    v1 = v0;
    if (h0 && c0.base + grp < c0.hi) { v0 = c.visits[c0.base + grp]; stage_visit(c, c0.L, v0.task, c.slot); }
    if (h1 && c1.base + grp < c1.hi) v1 = c.visits[c1.base + grp];
    int cur = 0;
    while (h0) {
        ChunkIt c2 = c1;
        const bool h2 = h1 && next_chunk<LMAX>(c2, it.lo, it.hi, myseg);
        Visit v2 = v1;
        if (h2 && c2.base + grp < c2.hi) v2 = c.visits[c2.base + grp];
        cp_async_wait_all();
        __syncwarp();   // the slot is complete, and every lane has left the slot refilled next
        if (h1 && c1.base + grp < c1.hi) stage_visit(c, c1.L, v1.task, c.slot + (cur ^ 1) * SLOT);
        if (c0.base + grp < c0.hi) {
            const double *s = c.slot + cur * SLOT;
            switch (c0.L) {
                case 0: colloc_visit<0, DERIV, ORTHO>(c, v0, s, acc); break;
                case 1: colloc_visit<1, DERIV, ORTHO>(c, v0, s, acc); break;
                case 2: colloc_visit<2, DERIV, ORTHO>(c, v0, s, acc); break;
                case 3: if constexpr (LMAX >= 3) colloc_visit<3, DERIV, ORTHO>(c, v0, s, acc); break;
                case 4: if constexpr (LMAX >= 4) colloc_visit<4, DERIV, ORTHO>(c, v0, s, acc); break;
                case 5: if constexpr (LMAX >= 5) colloc_visit<5, DERIV, ORTHO>(c, v0, s, acc); break;
                default: if constexpr (LMAX >= 6) colloc_visit<6, DERIV, ORTHO>(c, v0, s, acc); break;
            }
        }
        c0 = c1; h0 = h1; v0 = v1;
        c1 = c2; h1 = h2; v1 = v2;
        cur ^= 1;
    }
    __syncwarp();
    // gradient: grid-index components -> Cartesian, d/dX_c = sum_i Hinv[i][c] d/du_i (linear: before the sum)
    if constexpr (DERIV != 0) {
#pragma unroll
        for (int i = 0; i < 16; i++) {
            const double d1 = acc[1][i], d2 = acc[2][i], d3 = acc[3][i];
#pragma unroll
            for (int k = 0; k < 3; k++)
                acc[1 + k][i] = g.Hinv[0 * 3 + k] * d1 + g.Hinv[1 * 3 + k] * d2 + g.Hinv[2 * 3 + k] * d3;
        }
    }
    // the eight groups worked on different visits of the same block
    double *flat = &acc[0][0];
    const int off = group_reduce_scatter<NCOMP * 16>(flat, lane);
    const size_t ng = (size_t)g.N[0] * g.N[1] * g.N[2];
    constexpr int PER = NCOMP * 16 / 8;            // 8 (two rows of one component) or 2 (half a row)
    const int comp = off >> 4, j = (off & 15) >> 2, t0 = off & 3;
    double *out = P.grid[it.level] + comp * ng + ((size_t)c.n1 * g.N[1] + c.n2 + j) * g.N[2] + c.n3 + t0;
    if (it.single) {
#pragma unroll
        for (int i = 0; i < PER; i += 2) {
            double *o = out + (i >> 2) * g.N[2] + (i & 3);
            *reinterpret_cast<double2 *>(o) = make_double2(flat[i], flat[i + 1]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < PER; i++) atomicAdd(out + (i >> 2) * g.N[2] + (i & 3), flat[i]);
    }
}

template <int DERIV, int LMAX, bool ORTHO>
cudaError_t launch(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items, int nitem,
                   const double *coef, cudaStream_t st) {
    constexpr int smem = NWARP * NGRP * group_stride(LMAX) * (int)sizeof(double);
    static bool configured = false;   // per instantiation
    if (!configured) {
        const cudaError_t e = cudaFuncSetAttribute(k_collocate<DERIV, LMAX, ORTHO>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k_collocate<DERIV, LMAX, ORTHO><<<(nitem + NWARP - 1) / NWARP, NWARP * 32, smem, st>>>(P, tasks, visits, items, nitem, coef);
    return cudaGetLastError();
}

template <int DERIV, bool ORTHO>
cudaError_t launch_l(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items, int nitem,
                     const double *coef, int max_L, cudaStream_t st) {
    if (max_L <= 2) return launch<DERIV, 2, ORTHO>(P, tasks, visits, items, nitem, coef, st);
    if (max_L <= 4) return launch<DERIV, 4, ORTHO>(P, tasks, visits, items, nitem, coef, st);
    return launch<DERIV, 6, ORTHO>(P, tasks, visits, items, nitem, coef, st);
}

}  // namespace

cudaError_t launch_collocate(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items,
                             int nitem, const double *coef, int deriv, int max_L, bool ortho, cudaStream_t st) {
    if (deriv) return ortho ? launch_l<1, true>(P, tasks, visits, items, nitem, coef, max_L, st)
                            : launch_l<1, false>(P, tasks, visits, items, nitem, coef, max_L, st);
    return ortho ? launch_l<0, true>(P, tasks, visits, items, nitem, coef, max_L, st)
                 : launch_l<0, false>(P, tasks, visits, items, nitem, coef, max_L, st);
}

}  // namespace gpw
