// Collocation kernel (Eq. 3; the work of Alg. 1, re-decomposed for B200).
//
// One warp per work item = one 4x4x4 grid block and a range of its visit list.  The warp is eight groups
// of four lanes; a group evaluates one (pair, block) visit at a time and a lane owns the slab of 4x4 grid
// points at its own n1, so the polynomial collapse in u1 and the Gaussian set-up are paid once per 16
// points (gpw_math.cuh, colloc_slab).  Every lane keeps its rho values (and, for DERIV, the gradient in
// grid-index components) in registers for the whole list; the eight groups are summed by a shuffle
// reduce-scatter and the block is written once (the theoretical minimum the paper aims at),
// with no per-point cross-thread reduction (the bottleneck of Alg. 1 l.11).
//
// Data movement: the item's visits are cut into chunks of eight (one per group) that never straddle an L
// segment; the chunk table is built once per item in shared memory.  A pair's record and polynomial are
// one contiguous block of the workspace (8 + ncoef_pad(L) doubles) and reach the group's shared-memory
// slot by cp.async (16 bytes per lane and trip) issued two chunks ahead; the item's visit records are copied
// to shared memory once, so that no prefetched value waits in registers (the accumulators take 128 of the
// 255 registers of the GGA variant; a bulk-copy version was measured slower: cp.async.bulk is a
// warp-uniform instruction, eight different sources per chunk serialise).
#include "gpw_kernels.cuh"

namespace gpw {
namespace {

constexpr int NGRP = 8;     // groups of 4 lanes per warp
constexpr int NWARP = 4;    // warps (work items) per CTA
constexpr int NSLOT = 3;    // shared-memory slots per group (copy issued two chunks ahead)
constexpr int MAXCH = 64;   // chunks per item: ITEM_MAX / NGRP full ones + one ragged chunk per L segment
constexpr int MAXVIS = 384; // visits per item (ITEM_MAX of plan.cpp)

// Shared-memory slot of one visit: the pair record (8 doubles) followed by the pair polynomial.
GPW_CX int slot_doubles(int lmax) { return 8 + ncoef_pad(lmax); }
// A group's slots, padded to an odd number of 16-byte units: the eight groups' broadcast reads of the same
// coefficient then hit eight different bank pairs.
GPW_CX int group_stride(int lmax) {
    int n = NSLOT * slot_doubles(lmax);
    while (n % 4 != 2) n += 2;
    return n;
}
// per warp: the groups' slots, the chunk table, the item's visit records
GPW_CX int warp_doubles(int lmax) { return NGRP * group_stride(lmax) + MAXCH + MAXVIS; }

struct ColCtx {
    const double *rec;     // per-pair records: header (8 doubles) + polynomial
    const double *gm;      // the level's metric Gm (constant bank)
    const long long *coef_base;   // the level's class offsets (constant bank): record of pair i of class L
                                  // starts at coef_base[L] + i * (8 + ncoef_pad(L))
    double *slot;          // the group's shared-memory slots
    int n1, n2, n3;        // stored index of the lane's slab corner
    int N0, N1, N2;
    int x;                 // lane within the group
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(unsigned smem, const void *gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(unsigned smem, const void *gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// A visit record is its raw 8 bytes: task in the low word, the three signed wrap counts in bytes 4..6.
__device__ __forceinline__ int visit_task(unsigned long long r) { return (int)(unsigned)r; }
__device__ __forceinline__ int visit_wrap(unsigned long long r, int axis) {
    return (int)(signed char)(unsigned char)(r >> (32 + 8 * axis));
}

// The group's four lanes copy the record of `task` (class L) into a slot, 16 bytes per lane and trip.
template <int LMAX>
__device__ __forceinline__ void stage_visit(const ColCtx &c, int L, int task, double *slot) {
    const int nrec = 8 + ncoef_pad(L);          // doubles, even
    const char *src = reinterpret_cast<const char *>(c.rec + c.coef_base[L] + (long long)task * nrec) + 16 * c.x;
    const unsigned dst = smem_u32(slot) + 16 * c.x;
    const int n16 = nrec / 2 - c.x;             // 16-byte units left for this lane, stride 4
    constexpr int TRIPS = (slot_doubles(LMAX) / 2 + 3) / 4;
#pragma unroll
    for (int t = 0; t < TRIPS; t++)
        if (4 * t < n16) cp_async16(dst + 64 * t, src + 64 * t);
}

template <int L, int DERIV, bool ORTHO>
__device__ __forceinline__ void colloc_visit(const ColCtx &c, unsigned long long vi, const double *s, double (*acc)[16]) {
    const double ap = s[3];
    double q[6];
#pragma unroll
    for (int k = 0; k < 6; k++) q[k] = ap * c.gm[k];
    const double u1 = (double)(c.n1 + visit_wrap(vi, 0) * c.N0) - s[0];
    const double u20 = (double)(c.n2 + visit_wrap(vi, 1) * c.N1) - s[1];
    const double u30 = (double)(c.n3 + visit_wrap(vi, 2) * c.N2) - s[2];
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
                                                                   const Visit *__restrict__ visits,
                                                                   const Item *__restrict__ items, int nitem,
                                                                   const double *__restrict__ rec) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int SLOT = slot_doubles(LMAX);
    constexpr int GSTRIDE = group_stride(LMAX);
    extern __shared__ __align__(16) double sm[];
    const int warp = threadIdx.x >> 5;
    const int w = blockIdx.x * NWARP + warp;
    if (w >= nitem) return;
    const Item it = items[w];
    const LevelGeom &g = P.lev[it.level];
    const int lane = threadIdx.x & 31, grp = lane >> 2, x = lane & 3;
    double *wsm = sm + (size_t)warp * warp_doubles(LMAX);
    uint2 *tab = reinterpret_cast<uint2 *>(wsm + NGRP * GSTRIDE);
    unsigned long long *vis = reinterpret_cast<unsigned long long *>(wsm + NGRP * GSTRIDE + MAXCH);

    // ---- the item's visit records -> shared memory (first cp.async group) ----
    {
        const Visit *src = visits + P.tile_base[it.level][it.tile] + it.lo;
        const int n = min((int)(it.hi - it.lo), MAXVIS);   // cannot bind: items have at most MAXVIS visits
        for (int i = lane; i < n; i += 32) cp_async8(smem_u32(vis + i), src + i);
        cp_async_commit();
    }
    // ---- chunk table: entry = (first visit relative to it.lo, L | visits << 8) ----
    const unsigned myseg = P.seg[it.level][(size_t)it.tile * 8 + (lane & 7)];
    int nch = 0;
#pragma unroll 1
    for (int L = 0; L <= LMAX; L++) {
        const unsigned lo = max(it.lo, __shfl_sync(0xffffffffu, myseg, L));
        const unsigned hi = min(it.hi, __shfl_sync(0xffffffffu, myseg, L + 1));
        if (lo >= hi) continue;
        const int n = (int)((hi - lo + NGRP - 1) / NGRP);
        for (int k = lane; k < n; k += 32) {
            const unsigned base = lo + NGRP * k;
            if (nch + k < MAXCH) tab[nch + k] = make_uint2(base - it.lo, (unsigned)L | (min(hi - base, (unsigned)NGRP) << 8));
        }
        nch += n;
    }
    nch = min(nch, MAXCH);   // cannot bind: at most MAXVIS / NGRP full chunks + one ragged chunk per L segment

    ColCtx c;
    c.rec = rec;
    c.gm = g.Gm;
    c.coef_base = P.coef_base[it.level];
    c.slot = wsm + (size_t)grp * GSTRIDE;
    c.x = x;
    {
        const int T2 = g.T[2], T1 = g.T[1];
        const int b3 = it.tile % T2, b2 = (it.tile / T2) % T1, b1 = it.tile / (T2 * T1);
        c.n1 = 4 * b1 + x; c.n2 = 4 * b2; c.n3 = 4 * b3;
    }
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];

    double acc[NCOMP][16];
#pragma unroll
    for (int k = 0; k < NCOMP; k++)
#pragma unroll
        for (int i = 0; i < 16; i++) acc[k][i] = 0.0;

    cp_async_wait<0>();
    __syncwarp();   // visit records and chunk table complete

    // ---- software pipeline over the chunks: the records of chunk k+2 are in flight while chunk k is evaluated;
    //      one commit group per chunk (empty past the end), so "all but the newest" = chunks <= k complete ----
    auto stage_chunk = [&](int k, int slot) {
        if (k < nch) {
            const uint2 e = tab[k];
            if ((unsigned)grp < (e.y >> 8))
                stage_visit<LMAX>(c, (int)(e.y & 0xffu), visit_task(vis[e.x + grp]), c.slot + slot * SLOT);
        }
        cp_async_commit();
    };
    stage_chunk(0, 0);
    stage_chunk(1, 1);
    int slot = 0;
#pragma unroll 1
    for (int k = 0; k < nch; k++) {
        cp_async_wait<1>();   // chunk k has landed (chunk k+1 may still be in flight)
        __syncwarp();         // ... for all four lanes of the group; and every lane has left the slot refilled next
        stage_chunk(k + 2, slot >= 1 ? slot - 1 : slot + 2);
        const uint2 e = tab[k];
        if ((unsigned)grp < (e.y >> 8)) {
            const unsigned long long v0 = vis[e.x + grp];
            const double *s = c.slot + slot * SLOT;
            switch ((int)(e.y & 0xffu)) {
                case 0: colloc_visit<0, DERIV, ORTHO>(c, v0, s, acc); break;
                case 1: colloc_visit<1, DERIV, ORTHO>(c, v0, s, acc); break;
                case 2: colloc_visit<2, DERIV, ORTHO>(c, v0, s, acc); break;
                case 3: if constexpr (LMAX >= 3) colloc_visit<3, DERIV, ORTHO>(c, v0, s, acc); break;
                case 4: if constexpr (LMAX >= 4) colloc_visit<4, DERIV, ORTHO>(c, v0, s, acc); break;
                case 5: if constexpr (LMAX >= 5) colloc_visit<5, DERIV, ORTHO>(c, v0, s, acc); break;
                default: if constexpr (LMAX >= 6) colloc_visit<6, DERIV, ORTHO>(c, v0, s, acc); break;
            }
        }
        if (++slot == NSLOT) slot = 0;
    }
    cp_async_wait<0>();
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
cudaError_t launch(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                   const double *rec, cudaStream_t st) {
    constexpr int smem = NWARP * warp_doubles(LMAX) * (int)sizeof(double);
    static bool configured = false;   // per instantiation
    if (!configured) {
        const cudaError_t e = cudaFuncSetAttribute(k_collocate<DERIV, LMAX, ORTHO>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k_collocate<DERIV, LMAX, ORTHO><<<(nitem + NWARP - 1) / NWARP, NWARP * 32, smem, st>>>(P, visits, items, nitem, rec);
    return cudaGetLastError();
}

template <int DERIV, bool ORTHO>
cudaError_t launch_l(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                     const double *rec, int max_L, cudaStream_t st) {
    if (max_L <= 2) return launch<DERIV, 2, ORTHO>(P, visits, items, nitem, rec, st);
    if (max_L <= 4) return launch<DERIV, 4, ORTHO>(P, visits, items, nitem, rec, st);
    return launch<DERIV, 6, ORTHO>(P, visits, items, nitem, rec, st);
}

}  // namespace

cudaError_t launch_collocate(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                             const double *rec, int deriv, int max_L, bool ortho, cudaStream_t st) {
    if (deriv) return ortho ? launch_l<1, true>(P, visits, items, nitem, rec, max_L, st)
                            : launch_l<1, false>(P, visits, items, nitem, rec, max_L, st);
    return ortho ? launch_l<0, true>(P, visits, items, nitem, rec, max_L, st)
                 : launch_l<0, false>(P, visits, items, nitem, rec, max_L, st);
}

}  // namespace gpw
