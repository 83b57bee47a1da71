// Collocation kernel (Eq. 3; the work of Alg. 1, re-decomposed for B200).
//
// One warp (= one CTA) per work item = one 4x4x4 grid block and a range of its visit list: eight groups
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
#include <type_traits>

#include "gpw_kernels.cuh"

namespace gpw {
namespace {

constexpr int NGRP = 8;     // groups of 4 lanes per warp
// warps (work items) per CTA.  One: a warp's registers and shared memory go to the next item the moment it
// finishes, instead of waiting for the slowest of four items (measured: cfg2 k_collocate 3.58 -> 3.47 ms,
// cfg4 30.8 -> 29.6 ms; two warps per CTA: no gain)
constexpr int NWARP = 1;
// Shared-memory slots per group: three (copy issued two chunks ahead), except where the slots are what limits the
// resident warps -- value-only launches with polynomials of degree >= 5 (168 registers or fewer allow twelve warps per
// SM, three slots of 100-186 doubles per group only nine, or five for the degree-8 polynomials of tau): two there, the
// copy one chunk ahead.
#ifndef GPW_NSLOT_SMALL
#define GPW_NSLOT_SMALL 2
#endif
GPW_CX int nslot(int deriv, int dmax) { return (deriv == 0 && dmax >= 5) ? GPW_NSLOT_SMALL : 3; }
constexpr int MAXCH = 64;   // chunks per item: ITEM_MAX / NGRP full ones + one ragged chunk per L segment
constexpr int MAXVIS = 384; // visits per item (ITEM_MAX of plan.cpp)

// Per-visit Gaussian values (k_visit_gauss, computed once per plan: they depend on the geometry only): the
// Gaussian at the corner of each of the four lanes' slabs and the first-step ratios along n2 and n3, which for
// orthogonal lattice vectors are the same for the four slabs.
GPW_CX int vg_doubles(bool ortho) { return ortho ? 6 : 12; }
// Shared-memory slot of one visit: the pair record (8 doubles), the pair polynomial, the visit's Gaussian values.
GPW_CX int slot_vg(int lmax) { return 8 + ncoef_pad(lmax); }
GPW_CX int slot_doubles(int lmax, bool ortho) { return slot_vg(lmax) + vg_doubles(ortho); }
// A group's slots, padded to an odd number of 16-byte units: the eight groups' broadcast reads of the same
// coefficient then hit eight different bank pairs.
GPW_CX int group_stride(int lmax, bool ortho, int ns) {
    int n = ns * slot_doubles(lmax, ortho);
    while (n % 4 != 2) n += 2;
    return n;
}
// per warp: the groups' slots, the chunk table, the item's visit records
GPW_CX int warp_doubles(int lmax, bool ortho, int ns) { return NGRP * group_stride(lmax, ortho, ns) + MAXCH + MAXVIS; }

struct ColCtx {
    const double *rec;     // per-pair records: header (8 doubles) + polynomial
    const double *vg;      // Gaussian values of the item's visits (vg_doubles per visit)
    const double *gm;      // the level's metric Gm (constant bank)
    const long long *coef_base;   // the level's class offsets (constant bank): record of pair i of class L
                                  // starts at coef_base[L] + i * (8 + ncoef_pad(L))
    double *slot;          // the group's shared-memory slots
    int n1, n2, n3;        // stored index of the lane's slab corner
    int N0, N1, N2;
    int x;                 // lane within the group
};

// A visit record is its raw 8 bytes: task in the low word, the three signed wrap counts in bytes 4..6.
__device__ __forceinline__ int visit_task(unsigned long long r) { return (int)(unsigned)r; }
__device__ __forceinline__ int visit_wrap(unsigned long long r, int axis) {
    return (int)(signed char)(unsigned char)(r >> (32 + 8 * axis));
}

// The group's four lanes copy the record of `task` (class L) into a slot, 16 bytes per lane and trip.
// ... and the visit's Gaussian values (visit index iv relative to the item's first visit).
// LMAX here is the largest polynomial degree of the instantiation, deg the degree of this pair's polynomial (the
// pair's L plus the degree offset of the launch), L the pair's own la + lb (its class in coef_base).
template <int LMAX, bool ORTHO>
__device__ __forceinline__ void stage_visit(const ColCtx &c, int L, int deg, int task, unsigned iv, double *slot) {
    const int nrec = 8 + ncoef_pad(deg);        // doubles, even
    const char *src = reinterpret_cast<const char *>(c.rec + c.coef_base[L] + (long long)task * nrec) + 16 * c.x;
    const unsigned dst = smem_u32(slot) + 16 * c.x;
    const int n16 = nrec / 2 - c.x;             // 16-byte units left for this lane, stride 4
    constexpr int TRIPS = (slot_vg(LMAX) / 2 + 3) / 4;
#pragma unroll
    for (int t = 0; t < TRIPS; t++)
        if (4 * t < n16) cp_async16(dst + 64 * t, src + 64 * t);
    constexpr int VG = vg_doubles(ORTHO);
    const char *gsrc = reinterpret_cast<const char *>(c.vg + (size_t)iv * VG) + 16 * c.x;
    const unsigned gdst = smem_u32(slot + slot_vg(LMAX)) + 16 * c.x;
    if (c.x < VG / 2) cp_async16(gdst, gsrc);
    if constexpr (VG / 2 > 4) { if (c.x + 4 < VG / 2) cp_async16(gdst + 64, gsrc + 64); }
}

template <int L, int LMAX, int DERIV, bool ORTHO>
__device__ __forceinline__ void colloc_visit(const ColCtx &c, unsigned long long vi, const double *s, bool valid,
                                             double (*acc)[16]) {
    const double ap = s[3];
    double q[6];
#pragma unroll
    for (int k = 0; k < 6; k++) q[k] = ap * c.gm[k];
    const double u1 = (double)(c.n1 + visit_wrap(vi, 0) * c.N0) - s[0];
    const double u20 = (double)(c.n2 + visit_wrap(vi, 1) * c.N1) - s[1];
    const double u30 = (double)(c.n3 + visit_wrap(vi, 2) * c.N2) - s[2];
    const double *gv = s + slot_vg(LMAX);
    SlabGauss SG;
    SG.g0 = valid ? gv[c.x] : 0.0;   // a group without a visit of its own adds zeros (see the chunk loop)
    SG.r2 = ORTHO ? gv[4] : gv[4 + c.x];
    SG.r3 = ORTHO ? gv[5] : gv[8 + c.x];
    colloc_slab<L, DERIV, ORTHO>(s + 8, q, s[4], s[5], s[6], SG, u1, u20, u30, acc);
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

// LMAX: largest la + lb of the plan's pairs held by the instantiation.  LOFF: degree offset -- the polynomial of a pair
// of class L has degree L + LOFF (0: density and gradient; 2: kinetic-energy density, Eq. 15, whose pair product is
// again a polynomial times the same Gaussian, of degree L + 2).
// LLO, ACC: a launch evaluates the visits of the classes LLO <= L <= LMAX only; ACC: it adds to what an earlier launch
// wrote instead of overwriting.  The GGA collocation of plans with f shells runs as two launches -- classes L <= 4
// (the instantiation LMAX = 4: no body that spills, straight-line segment loops, 55 kB of code) and L = 5, 6 (LLO = 5,
// ACC) -- because the single kernel holding all seven bodies stalled on instruction fetch and spilled (profiles/r02.md).
template <int DERIV, int LMAX, bool ORTHO, int LOFF, int LLO = 0, bool ACC = false>
__global__ void __launch_bounds__(NWARP * 32, (DERIV ? 8 : 12) / NWARP) k_collocate(const __grid_constant__ GridParams P,
                                                                   const Visit *__restrict__ visits,
                                                                   const Item *__restrict__ items, int nitem,
                                                                   const double *__restrict__ rec,
                                                                   const double *__restrict__ vg) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int DMAX = LMAX + LOFF;
    constexpr int SLOT = slot_doubles(DMAX, ORTHO);
    constexpr int NSLOT = nslot(DERIV, DMAX);
    constexpr int GSTRIDE = group_stride(DMAX, ORTHO, NSLOT);
    extern __shared__ __align__(16) double sm[];
    const int warp = threadIdx.x >> 5;
    const int w = blockIdx.x * NWARP + warp;
    if (w >= nitem) return;
    const Item it = items[w];
    const LevelGeom &g = P.lev[it.level];
    {   // sharded plans: only the blocks of this process's n1 slab
        const int b1 = it.tile / (g.T[2] * g.T[1]);
        if (b1 < P.part_lo[it.level] || b1 >= P.part_hi[it.level]) return;
    }
    const int lane = threadIdx.x & 31, grp = lane >> 2, x = lane & 3;
    double *wsm = sm + (size_t)warp * warp_doubles(DMAX, ORTHO, NSLOT);
    uint2 *tab = reinterpret_cast<uint2 *>(wsm + NGRP * GSTRIDE);
    unsigned long long *vis = reinterpret_cast<unsigned long long *>(wsm + NGRP * GSTRIDE + MAXCH);

    // ---- the item's visit records -> shared memory (first cp.async group) ----
    {
        const Visit *src = visits + it.vstart;
        const int n = min((int)(it.hi - it.lo), MAXVIS);   // cannot bind: items have at most MAXVIS visits
        for (int i = lane; i < n; i += 32) cp_async8(smem_u32(vis + i), src + i);
        cp_async_commit();
    }
    // ---- chunk table: entry = (first visit relative to it.lo, L | visits << 8) ----
    const unsigned myseg = P.seg[it.level][(size_t)it.tile * 8 + (lane & 7)];
    int nch = 0;
    int kend[LMAX + 1];      // one past the last chunk of every L segment
#pragma unroll
    for (int L = 0; L < LLO; L++) kend[L] = 0;
#pragma unroll
    for (int L = LLO; L <= LMAX; L++) {
        const unsigned lo = max(it.lo, __shfl_sync(0xffffffffu, myseg, L));
        const unsigned hi = min(it.hi, __shfl_sync(0xffffffffu, myseg, L + 1));
        if (lo < hi) {
            const int n = (int)((hi - lo + NGRP - 1) / NGRP);
            for (int k = lane; k < n; k += 32) {
                const unsigned base = lo + NGRP * k;
                if (nch + k < MAXCH) tab[nch + k] = make_uint2(base - it.lo, (unsigned)L | (min(hi - base, (unsigned)NGRP) << 8));
            }
            nch += n;
        }
        kend[L] = min(nch, MAXCH);
    }
    nch = min(nch, MAXCH);   // cannot bind: at most MAXVIS / NGRP full chunks + one ragged chunk per L segment
    if (nch == 0) {          // no visit of this launch's classes in the item (the memset / the earlier launch stands)
        cp_async_wait<0>();
        return;
    }

    ColCtx c;
    c.rec = rec;
    c.vg = vg + (size_t)it.vstart * vg_doubles(ORTHO);
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
    // Branch-free: past the last chunk the last one is staged again (into a slot nobody reads any more), and a
    // group without a visit of its own copies group 0's record into its own slot.
    auto stage_chunk = [&](int k, int slot) {
        const uint2 e = tab[min(k, nch - 1)];
        const unsigned iv = e.x + ((unsigned)grp < (e.y >> 8) ? grp : 0);
        stage_visit<DMAX, ORTHO>(c, (int)(e.y & 0xffu), (int)(e.y & 0xffu) + LOFF, visit_task(vis[iv]), iv, c.slot + slot * SLOT);
        cp_async_commit();
    };
    stage_chunk(0, 0);
    if constexpr (NSLOT > 2) stage_chunk(1, 1);
    // One loop per L segment, its body straight-line code: a group without a visit of its own in a ragged chunk
    // evaluates group 0's visit with a zero Gaussian instead of branching around the evaluation, so that the
    // control work of the next chunks (table and visit records, cp.async addresses) can be scheduled into the
    // FP64 instruction stream.
    int slot = 0, k = 0;
    // the chunk's table entry and the group's visit record are read one chunk ahead (they are in shared memory
    // from the start), which takes two dependent shared-memory loads off the head of every chunk
    bool valid = (unsigned)grp < (tab[0].y >> 8);
    int gi = valid ? grp : 0;
    unsigned long long v0 = vis[tab[0].x + gi];
    auto run_segment = [&](auto Lc, int k_end) {
        constexpr int L = decltype(Lc)::value;
#pragma unroll 1
        for (; k < k_end; k++) {
            cp_async_wait<NSLOT - 2>();   // chunk k has landed (with three slots chunk k+1 may still be in flight)
            __syncwarp();         // ... for all four lanes of the group; and every lane has left the slot refilled next
            stage_chunk(k + NSLOT - 1, slot >= 1 ? slot - 1 : slot + NSLOT - 1);
            const uint2 en = tab[min(k + 1, nch - 1)];
            const bool valid_n = (unsigned)grp < (en.y >> 8);
            const int gi_n = valid_n ? grp : 0;
            const unsigned long long v_n = vis[en.x + gi_n];
            colloc_visit<L + LOFF, DMAX, DERIV, ORTHO>(c, v0, wsm + (size_t)gi * GSTRIDE + slot * SLOT, valid, acc);
            valid = valid_n; gi = gi_n; v0 = v_n;
            if (++slot == NSLOT) slot = 0;
        }
    };
    if constexpr (LMAX <= 4 || DERIV == 0) {
        if constexpr (LLO <= 0) run_segment(std::integral_constant<int, 0>{}, kend[0]);
        if constexpr (LLO <= 1) run_segment(std::integral_constant<int, 1>{}, kend[1]);
        if constexpr (LLO <= 2) run_segment(std::integral_constant<int, 2>{}, kend[2]);
        if constexpr (LMAX >= 3 && LLO <= 3) run_segment(std::integral_constant<int, 3>{}, kend[3]);
        if constexpr (LMAX >= 4 && LLO <= 4) run_segment(std::integral_constant<int, 4>{}, kend[4]);
        if constexpr (LMAX >= 5 && LLO <= 5) run_segment(std::integral_constant<int, 5>{}, kend[5]);
        if constexpr (LMAX >= 6) run_segment(std::integral_constant<int, 6>{}, kend[6]);
    } else {
        // deriv = 1 with f shells (L up to 6): the straight-line form costs registers the L = 5, 6 bodies do not
        // have (measured on cfg 4: 7 % slower); one loop, the evaluation behind a branch
#pragma unroll 1
        for (; k < nch; k++) {
            cp_async_wait<NSLOT - 2>();
            __syncwarp();
            stage_chunk(k + NSLOT - 1, slot >= 1 ? slot - 1 : slot + NSLOT - 1);
            const uint2 e = tab[k];
            if ((unsigned)grp < (e.y >> 8)) {
                const unsigned long long v0 = vis[e.x + grp];
                const double *s = c.slot + slot * SLOT;
                switch ((int)(e.y & 0xffu)) {
                    case 0: if constexpr (LLO <= 0) colloc_visit<0 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    case 1: if constexpr (LLO <= 1) colloc_visit<1 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    case 2: if constexpr (LLO <= 2) colloc_visit<2 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    case 3: if constexpr (LLO <= 3) colloc_visit<3 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    case 4: if constexpr (LLO <= 4) colloc_visit<4 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    case 5: colloc_visit<5 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                    default: colloc_visit<6 + LOFF, DMAX, DERIV, ORTHO>(c, v0, s, true, acc); break;
                }
            }
            if (++slot == NSLOT) slot = 0;
        }
    }
    cp_async_wait<0>();
    __syncwarp();
    // The eight groups worked on different visits of the same block: sum every component's 16 slab values over
    // the groups; afterwards the lane holds the two points off, off + 1 of its slab (same row), all components.
    int off = 0;
#pragma unroll
    for (int k = 0; k < NCOMP; k++) off = group_reduce_scatter<16>(acc[k], lane);
    // gradient: grid-index components -> Cartesian, d/dX_c = sum_i Hinv[i][c] d/du_i -- after the sum, on the
    // lane's two points instead of the sixteen of the slab
    if constexpr (DERIV != 0) {
#pragma unroll
        for (int i = 0; i < 2; i++) {
            const double d1 = acc[1][i], d2 = acc[2][i], d3 = acc[3][i];
#pragma unroll
            for (int k = 0; k < 3; k++)
                acc[1 + k][i] = g.Hinv[0 * 3 + k] * d1 + g.Hinv[1 * 3 + k] * d2 + g.Hinv[2 * 3 + k] * d3;
        }
    }
    const size_t ng = (size_t)g.N[0] * g.N[1] * g.N[2];
    const int j = off >> 2, t0 = off & 3;
    double *out = P.grid[it.level] + ((size_t)c.n1 * g.N[1] + c.n2 + j) * g.N[2] + c.n3 + t0;
    if (it.single) {
#pragma unroll
        for (int k = 0; k < NCOMP; k++) {
            double2 *o = reinterpret_cast<double2 *>(out + k * ng);
            if constexpr (ACC) { const double2 old = *o; *o = make_double2(old.x + acc[k][0], old.y + acc[k][1]); }
            else *o = make_double2(acc[k][0], acc[k][1]);
        }
    } else {
#pragma unroll
        for (int k = 0; k < NCOMP; k++) {
            atomicAdd(out + k * ng, acc[k][0]);
            atomicAdd(out + k * ng + 1, acc[k][1]);
        }
    }
}

template <int DERIV, int LMAX, bool ORTHO, int LOFF, int LLO = 0, bool ACC = false>
cudaError_t launch(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                   const double *rec, const double *vg, cudaStream_t st) {
    constexpr int smem = NWARP * warp_doubles(LMAX + LOFF, ORTHO, nslot(DERIV, LMAX + LOFF)) * (int)sizeof(double);
    // the attribute is per device (and per instantiation)
    static bool configured_dev[64] = {false};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
    const bool known = dev >= 0 && dev < 64;
    if (!known || !configured_dev[dev]) {
        const cudaError_t e = cudaFuncSetAttribute(k_collocate<DERIV, LMAX, ORTHO, LOFF, LLO, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (known) configured_dev[dev] = true;
    }
    k_collocate<DERIV, LMAX, ORTHO, LOFF, LLO, ACC><<<(nitem + NWARP - 1) / NWARP, NWARP * 32, smem, st>>>(P, visits, items, nitem, rec, vg);
    return cudaGetLastError();
}

template <int DERIV, bool ORTHO>
cudaError_t launch_l(const GridParams &P, const Visit *visits, const Item *items, int nitem, const Item *items_hi, int nitem_hi,
                     const double *rec, const double *vg, int max_L, cudaStream_t st) {
    if (max_L <= 2) return launch<DERIV, 2, ORTHO, 0>(P, visits, items, nitem, rec, vg, st);
    if (max_L <= 4) return launch<DERIV, 4, ORTHO, 0>(P, visits, items, nitem, rec, vg, st);
    if constexpr (DERIV != 0) {   // two launches: classes L <= 4, then L = 5, 6 on top (see k_collocate): cfg4 28.9 -> 24.6 ms
        const cudaError_t e = launch<DERIV, 4, ORTHO, 0>(P, visits, items, nitem, rec, vg, st);
        if (e != cudaSuccess) return e;
        // ... over its own items (the tails L >= 5 of the blocks' lists): on cfg 4 nine items in ten of the full list hold
        // no such visit, and 700 000 warps that only find that out cost more than the work of the others
        if (nitem_hi <= 0) return cudaSuccess;
        return launch<DERIV, 6, ORTHO, 0, 5, true>(P, visits, items_hi, nitem_hi, rec, vg, st);
    } else {
        // (two launches like the above, with the second over its own items, were measured for deriv = 0 too: cfg 3 1.45 -> 1.46 ms)
        return launch<DERIV, 6, ORTHO, 0>(P, visits, items, nitem, rec, vg, st);
    }
}
// kinetic-energy density: value only, polynomials of degree L + 2
template <bool ORTHO>
cudaError_t launch_tau(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                       const double *rec, const double *vg, int max_L, cudaStream_t st) {
    if (max_L <= 4) return launch<0, 4, ORTHO, 2>(P, visits, items, nitem, rec, vg, st);
    return launch<0, 6, ORTHO, 2>(P, visits, items, nitem, rec, vg, st);
}

}  // namespace

cudaError_t launch_collocate(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                             const Item *items_hi, int nitem_hi,
                             const double *rec, const double *vg, int deriv, int off, int max_L, bool ortho, cudaStream_t st) {
    if (off == 2 && deriv == 0)
        return ortho ? launch_tau<true>(P, visits, items, nitem, rec, vg, max_L, st)
                     : launch_tau<false>(P, visits, items, nitem, rec, vg, max_L, st);
    if (off != 0) return cudaErrorInvalidValue;
    if (deriv) return ortho ? launch_l<1, true>(P, visits, items, nitem, items_hi, nitem_hi, rec, vg, max_L, st)
                            : launch_l<1, false>(P, visits, items, nitem, items_hi, nitem_hi, rec, vg, max_L, st);
    return ortho ? launch_l<0, true>(P, visits, items, nitem, items_hi, nitem_hi, rec, vg, max_L, st)
                 : launch_l<0, false>(P, visits, items, nitem, items_hi, nitem_hi, rec, vg, max_L, st);
}

// ---------------------------------------------------------------------------------------- plan-time kernel
// Gaussian values of every (pair, block) visit, in the order of the visit lists: one CTA per stored block.
//   ORTHO:  [G(x = 0..3), r2, r3]      else:  [G(x = 0..3), r2(x = 0..3), r3(x = 0..3)]
// G(x) = exp(-a_p |H u|^2) at the corner (u10 + x, u20, u30) of lane x's slab, r2 / r3 = the ratio to the next
// point along n2 / n3 there (the starting values of the recursion of Eq. 24-25).
namespace {
template <bool ORTHO>
__global__ void __launch_bounds__(128) k_visit_gauss(const __grid_constant__ GridParams P, const TaskK *__restrict__ tasks,
                                                     const Visit *__restrict__ visits, double *__restrict__ vg) {
    constexpr int VG = vg_doubles(ORTHO);
    int tile = blockIdx.x, level = 0;
    while (tile >= P.lev[level].ntile) { tile -= P.lev[level].ntile; level++; }
    const LevelGeom &g = P.lev[level];
    const long long lo = P.tile_base[level][tile], hi = P.tile_base[level][tile + 1];
    const int T2 = g.T[2], T1 = g.T[1];
    const int n3 = 4 * (tile % T2), n2 = 4 * ((tile / T2) % T1), n1 = 4 * (tile / (T2 * T1));
    for (long long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const Visit v = visits[i];
        const TaskK k = tasks[v.task];
        double q[6];
#pragma unroll
        for (int m = 0; m < 6; m++) q[m] = k.ap * g.Gm[m];
        const double u10 = (double)(n1 + v.s[0] * g.N[0]) - k.nP[0];
        const double u20 = (double)(n2 + v.s[1] * g.N[1]) - k.nP[1];
        const double u30 = (double)(n3 + v.s[2] * g.N[2]) - k.nP[2];
        double *o = vg + (size_t)i * VG;
#pragma unroll
        for (int x = 0; x < 4; x++) {
            const double u1 = u10 + x;
            if constexpr (ORTHO) {
                o[x] = exp(-fma(q[0] * u1, u1, fma(q[1] * u20, u20, q[2] * u30 * u30)));
            } else {
                o[x] = exp(-(q[0] * u1 * u1 + q[1] * u20 * u20 + q[2] * u30 * u30 +
                             2.0 * (q[3] * u1 * u20 + (q[4] * u1 + q[5] * u20) * u30)));
                o[4 + x] = exp(-(2.0 * (q[3] * u1 + q[1] * u20 + q[5] * u30) + q[1]));
                o[8 + x] = exp(-(2.0 * (q[4] * u1 + q[5] * u20 + q[2] * u30) + q[2]));
            }
        }
        if constexpr (ORTHO) {
            o[4] = exp(-(q[1] * fma(2.0, u20, 1.0)));
            o[5] = exp(-(q[2] * fma(2.0, u30, 1.0)));
        }
    }
}
}  // namespace

size_t visit_gauss_doubles(bool ortho) { return (size_t)vg_doubles(ortho); }

cudaError_t launch_visit_gauss(const GridParams &P, int ntile_all, const TaskK *tasks, const Visit *visits, double *vg,
                               bool ortho, cudaStream_t st) {
    if (ntile_all <= 0) return cudaSuccess;
    if (ortho) k_visit_gauss<true><<<ntile_all, 128, 0, st>>>(P, tasks, visits, vg);
    else k_visit_gauss<false><<<ntile_all, 128, 0, st>>>(P, tasks, visits, vg);
    return cudaGetLastError();
}

}  // namespace gpw
