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
    unsigned gmask;        // the group's lanes
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// The group's four lanes copy the pair record and polynomial of `task` into a slot (16 bytes per lane and trip).
template <int L>
__device__ __forceinline__ void stage_visit(const ColCtx &c, int task, double *slot) {
    constexpr int NCH = 4 + ncoef_pad(L) / 2;   // 16-byte chunks
    const char *src_k = reinterpret_cast<const char *>(c.tasks + task);
    const char *src_c = reinterpret_cast<const char *>(c.work + c.coef_base[L] + (long long)task * ncoef_pad(L));
#pragma unroll
    for (int k0 = 0; k0 < NCH; k0 += 4) {
        const int k = k0 + c.x;
        if (k < NCH) cp_async16(reinterpret_cast<char *>(slot) + 16 * k, k < 4 ? src_k + 16 * k : src_c + 16 * (k - 4));
    }
    cp_async_commit();
}

template <int L, int DERIV, int SLOT>
__device__ __forceinline__ void colloc_segment(const ColCtx &c, unsigned lo, unsigned hi, int grp,
                                               double (*acc)[16]) {
    unsigned v = lo + grp;
    if (v >= hi) return;
    Visit vi = c.visits[v];
    stage_visit<L>(c, vi.task, c.slot);
    Visit vin = vi;
    if (v + NGRP < hi) vin = c.visits[v + NGRP];
    int cur = 0;
    for (;;) {
        const unsigned vn = v + NGRP;
        const bool more = vn < hi;
        cp_async_wait_all();
        __syncwarp(c.gmask);   // the slot is complete, and every lane has left the slot refilled next
        Visit vinn = vin;
        if (more) {
            stage_visit<L>(c, vin.task, c.slot + (cur ^ 1) * SLOT);   // in flight while this visit is evaluated
            if (vn + NGRP < hi) vinn = c.visits[vn + NGRP];
        }
        const double *s = c.slot + cur * SLOT;
        const double ap = s[3];
        double q[6];
#pragma unroll
        for (int k = 0; k < 6; k++) q[k] = ap * c.gm[k];
        const double u1 = (double)(c.n1 + vi.s[0] * c.N0) - s[0];
        const double u20 = (double)(c.n2 + vi.s[1] * c.N1) - s[1];
        const double u30 = (double)(c.n3 + vi.s[2] * c.N2) - s[2];
        colloc_slab<L, DERIV>(s + 8, q, s[4], s[5], s[6], u1, u20, u30, acc);
        if (!more) break;
        vi = vin; vin = vinn;
        v = vn;
        cur ^= 1;
    }
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

template <int DERIV, int LMAX>
__global__ void __launch_bounds__(128, DERIV ? 2 : 3) k_collocate(const __grid_constant__ GridParams P,
                                                                   const TaskK *__restrict__ tasks,
                                                                   const Visit *__restrict__ visits,
                                                                   const Item *__restrict__ items, int nitem,
                                                                   const double *__restrict__ coef) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int SLOT = slot_doubles(LMAX);
    extern __shared__ __align__(16) double sm[];   // [NWARP][NGRP][2][SLOT]
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
    c.slot = sm + (size_t)((threadIdx.x >> 5) * NGRP + grp) * 2 * SLOT;
    c.x = x;
    c.gmask = 0xFu << (grp * 4);
    c.n1 = 4 * b1 + x; c.n2 = 4 * b2; c.n3 = 4 * b3;
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];
    const unsigned *seg = P.seg[it.level] + (size_t)it.tile * 8;

    double acc[NCOMP][16];
#pragma unroll
    for (int k = 0; k < NCOMP; k++)
#pragma unroll
        for (int i = 0; i < 16; i++) acc[k][i] = 0.0;

#pragma unroll 1
    for (int L = 0; L <= LMAX; L++) {
        const unsigned lo = max(it.lo, seg[L]), hi = min(it.hi, seg[L + 1]);
        if (lo >= hi) continue;
        switch (L) {
            case 0: colloc_segment<0, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            case 1: colloc_segment<1, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            case 2: colloc_segment<2, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            case 3: if constexpr (LMAX >= 3) colloc_segment<3, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            case 4: if constexpr (LMAX >= 4) colloc_segment<4, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            case 5: if constexpr (LMAX >= 5) colloc_segment<5, DERIV, SLOT>(c, lo, hi, grp, acc); break;
            default: if constexpr (LMAX >= 6) colloc_segment<6, DERIV, SLOT>(c, lo, hi, grp, acc); break;
        }
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

template <int DERIV, int LMAX>
cudaError_t launch(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items, int nitem,
                   const double *coef, cudaStream_t st) {
    constexpr int smem = NWARP * NGRP * 2 * slot_doubles(LMAX) * (int)sizeof(double);
    static bool configured = false;   // per instantiation
    if (!configured) {
        const cudaError_t e = cudaFuncSetAttribute(k_collocate<DERIV, LMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k_collocate<DERIV, LMAX><<<(nitem + NWARP - 1) / NWARP, NWARP * 32, smem, st>>>(P, tasks, visits, items, nitem, coef);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_collocate(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items,
                             int nitem, const double *coef, int deriv, int max_L, cudaStream_t st) {
    if (deriv) {
        if (max_L <= 2) return launch<1, 2>(P, tasks, visits, items, nitem, coef, st);
        if (max_L <= 4) return launch<1, 4>(P, tasks, visits, items, nitem, coef, st);
        return launch<1, 6>(P, tasks, visits, items, nitem, coef, st);
    }
    if (max_L <= 2) return launch<0, 2>(P, tasks, visits, items, nitem, coef, st);
    if (max_L <= 4) return launch<0, 4>(P, tasks, visits, items, nitem, coef, st);
    return launch<0, 6>(P, tasks, visits, items, nitem, coef, st);
}

}  // namespace gpw
