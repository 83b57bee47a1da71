// Integration kernel (Eq. 4 with the quadrature of Eq. 29; the work of Alg. 2,
// PAPER.md:240-263, re-decomposed for B200).
//
// One CTA per work item = one brick of 1 x 5 x 5 grid blocks and a range of its entry list; an entry is a
// (pair, lattice image) with the mask of the brick's blocks it visits.  The CTA stages the brick of v in
// shared memory once (for DERIV with the vector field already mapped to grid-index components), laid out
// per block and n1 plane.  A warp is eight groups of four lanes; a group owns one entry at a time and a
// lane owns the n1 plane x of every block, i.e. slabs of 4 x 4 points at a fixed u1.  Over all the
// entry's blocks the lane accumulates the partial moments B0[ky][kz] (and B1 for DERIV) in registers
// (gpw_math.cuh, integ_slab_rows); the expansion in u1, a shuffle reduction over the group's four lanes
// and one FP64 atomic per moment finish the entry.  Alg. 2 instead adds nca*ncb values per (pair, block)
// to global memory; amortising over the brick cuts that traffic by the blocks per
// entry, and the moment form keeps the per-lane state at (L+1)(L+2)/2 doubles instead of nca*ncb.
// Orthogonal cells: the Gaussian separates and the 1-D factor tables of every entry over its brick are
// geometry only -- computed once per plan (k_entry_gauss below, 352 bytes per entry) and staged by cp.async
// with the pair record, so that an entry starts on its first block without exp() or recursion (measured:
// cfg2 k_integrate 4.04 -> 3.58 ms, cfg4 33.4 -> 26.8 ms against building them per entry in the kernel).
#include "gpw_kernels.cuh"

namespace gpw {
namespace {

constexpr int NWARP = 4;
constexpr int NGRP = 8;   // groups of 4 lanes per warp

// Shared-memory brick, general cells: chunk = the 4 x 4 points of one n1 plane of one block, all components,
// plus 16 bytes of padding: the four lanes of a group then read four different bank quarters with their
// 16-byte loads.
GPW_CX int chunk_doubles(int ncomp) { return ncomp * 16 + 2; }
// Shared-memory brick, ORTHO: one 128-byte line per (block, component, row j) = the points t = 0,1 of the four
// n1 planes (64 bytes, 16 banks) followed by the points t = 2,3 of the four planes (the other 16 banks).  A
// 16-byte load instruction is served per quarter warp = two lane groups; even groups read the first half of
// the line first and odd groups the second half (they own their four points in the order 2,3,0,1), so the two
// groups of a quarter warp never meet in a bank, whatever blocks they are working on.
GPW_CX int brick_doubles(int ncomp, bool ortho) {
    return ortho ? BRICK_TILES * ncomp * 4 * 16 : BRICK_TILES * 4 * chunk_doubles(ncomp);
}

// ORTHO: the Gaussian separates, G = gx(u1) gy(u2) gz(u3).  The 1-D factors of every brick entry over the whole
// brick -- gy[4 BR2], gz[4 BR3], gx[4] -- depend on the geometry only: they are computed once per plan
// (k_entry_gauss, EG doubles per entry) and reach one of the group's two shared-memory slots by cp.async one
// chunk ahead; a group's slots are padded so that the eight groups' 16-byte reads start in different banks.
constexpr int GT2 = 4 * BR2, GT3 = 4 * BR3;
constexpr int EG = GT2 + GT3 + 4;
constexpr int GT_STRIDE = 2 * EG + 2;
static_assert(GT2 % 2 == 0 && GT3 % 2 == 0 && EG % 2 == 0 && GT_STRIDE % 2 == 0, "16-byte alignment of the factor tables");

struct BrickCtx {
    unsigned gmask;          // the group's four lanes
    int odd;                 // parity of the group within its warp
    const double *vs;        // shared memory brick: chunk (block, x) at (block*4 + x) * chunk_doubles
    const double *gm;        // the level's metric (constant bank)
    int o1, o2, o3;          // stored grid index of the brick origin
    int N0, N1, N2;
    int x;                   // lane within the group = n1 plane
};

template <int L, int DERIV, bool ORTHO>
__device__ __forceinline__ void integ_entry(const BrickCtx &c, const BEntry en, const double *prs, const double *gt,
                                            bool valid, double *__restrict__ dst) {
    // the pair record (TaskK) staged in the group's shared-memory slot
    PairRec pr;
    pr.nP0 = prs[0]; pr.nP1 = prs[1]; pr.nP2 = prs[2]; pr.ap = prs[3];
    pr.c22 = prs[4]; pr.c23 = prs[5]; pr.c33 = prs[6];
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int CHS = chunk_doubles(NCOMP);
    constexpr int NB = npair2(L), NBX = npair2(L - 1);
    double B0[NB], B1[NBX > 0 ? NBX : 1];
#pragma unroll
    for (int i = 0; i < NB; i++) B0[i] = 0.0;
#pragma unroll
    for (int i = 0; i < (NBX > 0 ? NBX : 1); i++) B1[i] = 0.0;
    double q[6];
#pragma unroll
    for (int k = 0; k < 6; k++) q[k] = pr.ap * c.gm[k];
    const double u1 = (double)(c.o1 + c.x + en.s[0] * c.N0) - pr.nP0;
    const double u2b = (double)(c.o2 + en.s[1] * c.N1) - pr.nP1;
    const double u3b = (double)(c.o3 + en.s[2] * c.N2) - pr.nP2;
    // ORTHO: the entry's 1-D factor tables are in the slot gt; the factor of the lane's own n1 plane
    double gx = 1.0;
    if constexpr (ORTHO) gx = gt[GT2 + GT3 + c.x];
    unsigned mask = valid ? en.mask : 0u;
    while (mask) {   // group-uniform
        const int bit = __ffs(mask) - 1;
        mask &= mask - 1;
        const int t2 = bit / BR3, t3 = bit - t2 * BR3;
        const double *chunk = c.vs + (bit * 4 + c.x) * CHS;
        const double u20 = u2b + 4 * t2, u30 = u3b + 4 * t3;
        auto vrow = [&](int k, int j, double *o) {
            const double2 a = *reinterpret_cast<const double2 *>(chunk + k * 16 + j * 4);
            const double2 b = *reinterpret_cast<const double2 *>(chunk + k * 16 + j * 4 + 2);
            o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
        };
        if constexpr (ORTHO) {
            const int h = c.odd;
            const double *line = c.vs + (size_t)bit * (NCOMP * 64) + 2 * c.x;
            auto vline = [&](int k, int j, double *o) {
                const double *r = line + (k * 4 + j) * 16;
                const double2 a = *reinterpret_cast<const double2 *>(r + 8 * h);
                const double2 b = *reinterpret_cast<const double2 *>(r + 8 * (1 - h));
                o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
            };
            const double2 y0 = *reinterpret_cast<const double2 *>(gt + 4 * t2);
            const double2 y1 = *reinterpret_cast<const double2 *>(gt + 4 * t2 + 2);
            const double2 z0 = *reinterpret_cast<const double2 *>(gt + GT2 + 4 * t3 + 2 * h);
            const double2 z1 = *reinterpret_cast<const double2 *>(gt + GT2 + 4 * t3 + 2 * (1 - h));
            const double rowg[4] = {gx * y0.x, gx * y0.y, gx * y1.x, gx * y1.y};
            const double g3[4] = {z0.x, z0.y, z1.x, z1.y};
            const double t0 = (double)(2 * h), t2o = (double)(2 * (1 - h));
            const double toff[4] = {t0, t0 + 1.0, t2o, t2o + 1.0};
            integ_slab_rows<L, DERIV, true>(vline, q, pr.c22, pr.c23, pr.c33, SlabGauss{0.0, 0.0, 0.0}, u1, u20, u30,
                                            B0, B1, rowg, g3, toff);
        } else {
            const SlabGauss SG = slab_gauss<false>(q, u1, u20, u30);
            integ_slab_rows<L, DERIV, false>(vrow, q, pr.c22, pr.c23, pr.c33, SG, u1, u20, u30, B0, B1);
        }
    }
    __syncwarp();
    // expansion in u1, sum over the group's four lanes (n1 planes), one atomic per moment.  The sum is a reduce-scatter:
    // after the exchange with lane x ^ 1 a lane holds the pair sums of one half of the moments, after the one with lane
    // x ^ 2 the full sums of one quarter, which it adds to the workspace -- 3/4 N shuffles of doubles instead of the 2 N
    // of a butterfly per moment (the shuffles share the shared-memory pipe the block loops are bound by; the entry tails
    // were 12 % of the warp samples of cfg 2).  Same summation tree: (x0 + x1) + (x2 + x3).
    constexpr int N = ncoef(L), N4 = (N + 3) & ~3, HALF = N4 / 2, QUART = N4 / 4;
    double pw1[L + 1];
    pw1[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= L; k++) pw1[k] = pw1[k - 1] * u1;
    if constexpr (N > 84) {
        // degree 7, 8 (the derivative variants of f shells): 120 / 165 moments do not fit a register array; a butterfly per moment
#pragma unroll
        for (int kz = 0; kz <= L; kz++)
#pragma unroll
            for (int ky = 0; ky <= L - kz; ky++)
#pragma unroll
                for (int kx = 0; kx <= L - kz - ky; kx++) {
                    double s = integ_expand_term<L, DERIV>(B0, B1, pw1, kx, ky, kz);
                    s += __shfl_xor_sync(0xffffffffu, s, 1);
                    s += __shfl_xor_sync(0xffffffffu, s, 2);
                    const int k = cidx(L, kx, ky, kz);
                    if (valid && (k & 3) == c.x) atomicAdd(dst + k, s);
                }
        return;
    }
    double sv[N4];
#pragma unroll
    for (int k = N; k < N4; k++) sv[k] = 0.0;
#pragma unroll
    for (int kz = 0; kz <= L; kz++)
#pragma unroll
        for (int ky = 0; ky <= L - kz; ky++)
#pragma unroll
            for (int kx = 0; kx <= L - kz - ky; kx++) sv[cidx(L, kx, ky, kz)] = integ_expand_term<L, DERIV>(B0, B1, pw1, kx, ky, kz);
    const bool up1 = c.x & 1, up2 = c.x & 2;
#pragma unroll
    for (int i = 0; i < HALF; i++) {
        const double send = up1 ? sv[i] : sv[i + HALF];
        const double keep = up1 ? sv[i + HALF] : sv[i];
        sv[i] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
    }
#pragma unroll
    for (int i = 0; i < QUART; i++) {
        const double send = up2 ? sv[i] : sv[i + QUART];
        const double keep = up2 ? sv[i + QUART] : sv[i];
        sv[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
    }
    const int off = (up1 ? HALF : 0) + (up2 ? QUART : 0);
#pragma unroll
    for (int i = 0; i < QUART; i++)
        if (valid && off + i < N) atomicAdd(dst + off + i, sv[i]);
}

// LMAX: largest la + lb held by the instantiation.  LOFF: degree offset -- the moments of a pair of class L are
// accumulated up to degree L + LOFF (0: Eq. 4; 1: nuclear gradient, Alg. 3; 2: kinetic-energy potential, Eq. 16).
// LLO: a launch takes the entries of the classes LLO <= L <= LMAX only (the moments of all launches add up in `mom`).
// Plans with f shells run as two launches, classes L <= 4 (the instantiation LMAX = 4: smaller code, and for deriv = 0
// three CTAs per SM instead of two) and L = 5, 6.
template <int DERIV, int LMAX, bool ORTHO, int LOFF, int LLO = 0>
// deriv = 0 with f shells (L up to 6): three CTAs per SM leave 168 registers and the L = 5, 6 bodies spill; two CTAs
// at 220 registers without spills are faster (cfg3 k_integrate 2.40 -> 2.31 ms)
__global__ void __launch_bounds__(NWARP * 32, (DERIV || LMAX + LOFF > 4) ? 2 : 3) k_integrate(const __grid_constant__ GridParams P,
                                                                          const TaskK *__restrict__ tasks,
                                                                          const BEntry *__restrict__ entries,
                                                                          const BItem *__restrict__ items,
                                                                          const double *__restrict__ eg,
                                                                          double *__restrict__ mom) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int CHS = chunk_doubles(NCOMP);
    extern __shared__ __align__(16) double vs[];   // [BRICK_TILES * 4] chunks
    __shared__ unsigned s_seg[8];
    __shared__ __align__(16) double s_gtab[ORTHO ? NWARP * NGRP * GT_STRIDE : 2];
    __shared__ __align__(16) double s_pair[NWARP * NGRP * 2 * 8];   // per group: two slots of one pair record
    const BItem *itp = items + blockIdx.x;
    const int level = itp->level, brick = itp->brick;
    {   // sharded plans: only the bricks of this process's n1 slab (a brick is one block thick along n1)
        const int k1p = brick / (P.lev[level].B[2] * P.lev[level].B[1]);
        if (k1p < P.part_lo[level] || k1p >= P.part_hi[level]) return;
    }
    const unsigned it_lo = itp->lo, it_hi = itp->hi;
    const long long ebase = itp->base;
    if (threadIdx.x < 8) s_seg[threadIdx.x] = itp->seg[threadIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, grp = lane >> 2;
    const BEntry *ent = entries + ebase;
    __syncthreads();   // s_seg
    {   // nothing of this launch's classes in the item: leave before the brick is staged (uniform over the CTA)
        const unsigned lo = max(it_lo, s_seg[LLO]), hi = min(it_hi, s_seg[LMAX + 1]);
        if (lo >= hi) return;
    }

    // The item's entries in chunks of NGRP that never straddle an L segment (so the code path is
    // warp-uniform); the chunks are dealt to the CTA's warps round robin: warp w takes the chunks w, w + NWARP, ... of
    // the item's chunk sequence and finds each by walking the segments forward (chunk c lies in the segment whose
    // first chunk c0 and chunk count n have c0 <= c < c0 + n).
    int L = LLO - 1, cnext = warp, kc0 = 0, nseg = 0;
    unsigned base = 0, lo = 0, hi = 0;
    auto next_chunk = [&]() -> bool {
        if (L > LMAX) return false;   // past the last segment (the sequence has ended for this warp)
        const int cidx_ = cnext;
        cnext += NWARP;
        while (cidx_ >= kc0 + nseg) {
            kc0 += nseg;
            nseg = 0;
            L++;
            if (L > LMAX) return false;
            lo = max(it_lo, s_seg[L]);
            hi = min(it_hi, s_seg[L + 1]);
            nseg = lo < hi ? (int)((hi - lo + NGRP - 1) / NGRP) : 0;
        }
        base = lo + (unsigned)(NGRP * (cidx_ - kc0));
        return true;
    };
    // Software pipeline over the warp's chunks: the entry records are loaded two chunks ahead (one 16-byte load
    // per group), the pair records, whose address depends on the entry, one chunk ahead.
    struct Chunk { int L; unsigned base, hi; bool ok; };
    auto take = [&]() -> Chunk { const bool ok = next_chunk(); return Chunk{L, base, hi, ok}; };
    const uint4 *ent4 = reinterpret_cast<const uint4 *>(ent);
    auto load_entry = [&](const Chunk &ch) -> uint4 {
        return (ch.ok && ch.base + grp < ch.hi) ? __ldg(ent4 + ch.base + grp) : make_uint4(0u, 0u, 0u, 0u);
    };
    auto decode = [](const uint4 r) -> BEntry {
        BEntry e;
        e.task = (int)r.x;
        e.s[0] = (signed char)(r.y & 0xffu); e.s[1] = (signed char)((r.y >> 8) & 0xffu); e.s[2] = (signed char)((r.y >> 16) & 0xffu);
        e.L = (unsigned char)(r.y >> 24);
        e.mask = r.z; e.pad = r.w;
        return e;
    };
    // the first two chunks' entry records are in flight while the brick is staged
    Chunk c0 = take();
    Chunk c1 = take();
    uint4 e0 = load_entry(c0), e1 = load_entry(c1);

    const LevelGeom &g = P.lev[level];
    const int B2 = g.B[2], B1n = g.B[1];
    const int k3 = brick % B2, k2 = (brick / B2) % B1n, k1 = brick / (B2 * B1n);
    const size_t ng = (size_t)g.N[0] * g.N[1] * g.N[2];
    const double *vin = P.grid[level];
    // ---- stage the brick: one row of 4 points (x NCOMP) per thread and trip; t3 fastest for coalescing ----
    for (int r = threadIdx.x; r < BRICK_TILES * 16; r += NWARP * 32) {
        const int t3 = r % BR3, j = (r / BR3) & 3, t2 = (r / (BR3 * 4)) % BR2, x = r / (BR3 * 4 * BR2);
        const int b1 = k1, b2 = BR2 * k2 + t2, b3 = BR3 * k3 + t3;
        if (b2 >= g.T[1] || b3 >= g.T[2]) continue;   // ragged brick: never referenced
        const double *src = vin + ((size_t)(4 * b1 + x) * g.N[1] + 4 * b2 + j) * g.N[2] + 4 * b3;
        double raw[NCOMP][4];
#pragma unroll
        for (int k = 0; k < NCOMP; k++) {
            const double2 *p2 = reinterpret_cast<const double2 *>(src + k * ng);
            const double2 x0 = __ldg(p2), x1 = __ldg(p2 + 1);
            raw[k][0] = x0.x; raw[k][1] = x0.y; raw[k][2] = x1.x; raw[k][3] = x1.y;
        }
        double *dst = vs + ((t2 * BR3 + t3) * 4 + x) * CHS + j * 4;
        // ORTHO: line of (block, component k, row j) at ((block * NCOMP + k) * 4 + j) * 16; plane x at + 2 x, + 8 + 2 x
        double *dsto = vs + ((size_t)(t2 * BR3 + t3) * NCOMP * 4 + j) * 16 + 2 * x;
        if constexpr (DERIV) {
            // w'_i = sum_c Hinv[i][c] w_c, so that w . grad_r f = w' . grad_u f
            double tr[4][4];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                tr[0][t] = raw[0][t];
#pragma unroll
                for (int i = 0; i < 3; i++)
                    tr[1 + i][t] = g.Hinv[i * 3 + 0] * raw[1][t] + g.Hinv[i * 3 + 1] * raw[2][t] +
                                   g.Hinv[i * 3 + 2] * raw[3][t];
            }
#pragma unroll
            for (int k = 0; k < 4; k++) {
                if constexpr (ORTHO) {
                    *reinterpret_cast<double2 *>(dsto + k * 64) = make_double2(tr[k][0], tr[k][1]);
                    *reinterpret_cast<double2 *>(dsto + k * 64 + 8) = make_double2(tr[k][2], tr[k][3]);
                } else {
                    *reinterpret_cast<double2 *>(dst + k * 16) = make_double2(tr[k][0], tr[k][1]);
                    *reinterpret_cast<double2 *>(dst + k * 16 + 2) = make_double2(tr[k][2], tr[k][3]);
                }
            }
        } else if constexpr (ORTHO) {
            *reinterpret_cast<double2 *>(dsto) = make_double2(raw[0][0], raw[0][1]);
            *reinterpret_cast<double2 *>(dsto + 8) = make_double2(raw[0][2], raw[0][3]);
        } else {
            *reinterpret_cast<double2 *>(dst) = make_double2(raw[0][0], raw[0][1]);
            *reinterpret_cast<double2 *>(dst + 2) = make_double2(raw[0][2], raw[0][3]);
        }
    }
    // Pair records (TaskK, 64 bytes) reach the group's shared-memory slot by cp.async, 16 bytes per lane, one chunk
    // ahead of their use (a record prefetched into registers was spilled to the stack at once, which made the
    // warp wait for the load: 6 % of the warp samples of profile r01g)
    double *mypair = s_pair + (warp * NGRP + grp) * 16;
    // ... together with the factor tables of the group's entry (ORTHO; the entry index does not depend on a load)
    double *mygt = s_gtab + (ORTHO ? (warp * NGRP + grp) * GT_STRIDE : 0);
    auto stage_pair = [&](const Chunk &ch, unsigned task, int slot) {
        cp_async16(smem_u32(mypair + slot * 8) + 16 * (lane & 3), reinterpret_cast<const char *>(tasks + task) + 16 * (lane & 3));
        if constexpr (ORTHO) {
            // a group without an entry of its own copies a valid entry's tables (never used: its mask is empty)
            const unsigned ei = ch.ok ? min(ch.base + grp, ch.hi - 1) : it_lo;
            const char *src = reinterpret_cast<const char *>(eg + (size_t)(ebase + ei) * EG) + 16 * (lane & 3);
            const unsigned dst = smem_u32(mygt + slot * EG) + 16 * (lane & 3);
#pragma unroll
            for (int t = 0; t < (EG / 2 + 3) / 4; t++)
                if (4 * t + (lane & 3) < EG / 2) cp_async16(dst + 64 * t, src + 64 * t);
        }
        cp_async_commit();
    };
    stage_pair(c0, e0.x, 0);
    __syncthreads();
    if (!c0.ok) { cp_async_wait<0>(); return; }

    BrickCtx c;
    c.vs = vs;
    c.gm = g.Gm;
    c.o1 = 4 * BR1 * k1; c.o2 = 4 * BR2 * k2; c.o3 = 4 * BR3 * k3;
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];
    c.x = lane & 3;
    c.gmask = 0xfu << (4 * grp);
    c.odd = grp & 1;

    int ps = 0;
    while (c0.ok) {
        const Chunk c2 = c1.ok ? take() : c1;
        const uint4 e2 = load_entry(c2);
        __syncwarp();                 // every lane has left the slot refilled next
        stage_pair(c1, e1.x, ps ^ 1); // e1 was requested one chunk ago
        cp_async_wait<1>();           // this chunk's record has landed
        __syncwarp();                 // ... for all four lanes of the group
        const double *prs = mypair + ps * 8;
        const double *gt = mygt + ps * EG;
        const bool valid = c0.base + grp < c0.hi;
        const BEntry enc = decode(e0);
        // the pair's moment vector: class base + pair index * vector length (degree L + LOFF)
        const int deg = c0.L + LOFF;
        double *dst = mom + P.coef_base[level][c0.L] + (long long)enc.task * (((deg + 1) * (deg + 2) * (deg + 3) / 6 + 1) & ~1);
        switch (c0.L) {
            case 0: if constexpr (LLO <= 0) integ_entry<0 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            case 1: if constexpr (LLO <= 1) integ_entry<1 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            case 2: if constexpr (LLO <= 2) integ_entry<2 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            case 3: if constexpr (LMAX >= 3 && LLO <= 3) integ_entry<3 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            case 4: if constexpr (LMAX >= 4 && LLO <= 4) integ_entry<4 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            case 5: if constexpr (LMAX >= 5) integ_entry<5 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
            default: if constexpr (LMAX >= 6) integ_entry<6 + LOFF, DERIV, ORTHO>(c, enc, prs, gt, valid, dst); break;
        }
        c0 = c1; e0 = e1;
        c1 = c2; e1 = e2;
        ps ^= 1;
    }
    cp_async_wait<0>();
}

template <int DERIV, int LMAX, bool ORTHO, int LOFF, int LLO = 0>
cudaError_t launch(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items, int nitem,
                   const double *eg, double *mom, cudaStream_t st) {
    constexpr int smem = brick_doubles(DERIV ? 4 : 1, ORTHO) * (int)sizeof(double);
    // the attribute is per device (and per instantiation)
    static bool configured_dev[64] = {false};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
    const bool known = dev >= 0 && dev < 64;
    if (!known || !configured_dev[dev]) {
        const cudaError_t e = cudaFuncSetAttribute(k_integrate<DERIV, LMAX, ORTHO, LOFF, LLO>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (known) configured_dev[dev] = true;
    }
    k_integrate<DERIV, LMAX, ORTHO, LOFF, LLO><<<nitem, NWARP * 32, smem, st>>>(P, tasks, entries, items, eg, mom);
    return cudaGetLastError();
}

template <int DERIV, bool ORTHO>
cudaError_t launch_l(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items, int nitem,
                     const double *eg, double *mom, int max_L, cudaStream_t st) {
    if (max_L <= 2) return launch<DERIV, 2, ORTHO, 0>(P, tasks, entries, items, nitem, eg, mom, st);
    if (max_L <= 4) return launch<DERIV, 4, ORTHO, 0>(P, tasks, entries, items, nitem, eg, mom, st);
    // two launches (see k_integrate): measured cfg3 k_integrate 2.32 -> 2.15 ms, cfg4 25.5 -> 23.9 ms
    const cudaError_t e = launch<DERIV, 4, ORTHO, 0>(P, tasks, entries, items, nitem, eg, mom, st);
    if (e != cudaSuccess) return e;
    return launch<DERIV, 6, ORTHO, 0, 5>(P, tasks, entries, items, nitem, eg, mom, st);
}
// moments of degree L + LOFF (nuclear gradient: LOFF = 1, value or value + gradient field; kinetic-energy
// potential: LOFF = 2, value only)
template <int DERIV, bool ORTHO, int LOFF>
cudaError_t launch_off(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items, int nitem,
                       const double *eg, double *mom, int max_L, cudaStream_t st) {
    if (max_L <= 4) return launch<DERIV, 4, ORTHO, LOFF>(P, tasks, entries, items, nitem, eg, mom, st);
    const cudaError_t e = launch<DERIV, 4, ORTHO, LOFF>(P, tasks, entries, items, nitem, eg, mom, st);   // two launches, as above
    if (e != cudaSuccess) return e;
    return launch<DERIV, 6, ORTHO, LOFF, 5>(P, tasks, entries, items, nitem, eg, mom, st);
}

}  // namespace

cudaError_t launch_integrate(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items,
                             int nitem, const double *eg, double *mom, int deriv, int off, int max_L, bool ortho, cudaStream_t st) {
    if (off == 2 && deriv == 0)
        return ortho ? launch_off<0, true, 2>(P, tasks, entries, items, nitem, eg, mom, max_L, st)
                     : launch_off<0, false, 2>(P, tasks, entries, items, nitem, eg, mom, max_L, st);
    if (off == 1 && deriv == 0)
        return ortho ? launch_off<0, true, 1>(P, tasks, entries, items, nitem, eg, mom, max_L, st)
                     : launch_off<0, false, 1>(P, tasks, entries, items, nitem, eg, mom, max_L, st);
    if (off == 1)
        return ortho ? launch_off<1, true, 1>(P, tasks, entries, items, nitem, eg, mom, max_L, st)
                     : launch_off<1, false, 1>(P, tasks, entries, items, nitem, eg, mom, max_L, st);
    if (off != 0) return cudaErrorInvalidValue;
    if (deriv) return ortho ? launch_l<1, true>(P, tasks, entries, items, nitem, eg, mom, max_L, st)
                            : launch_l<1, false>(P, tasks, entries, items, nitem, eg, mom, max_L, st);
    return ortho ? launch_l<0, true>(P, tasks, entries, items, nitem, eg, mom, max_L, st)
                 : launch_l<0, false>(P, tasks, entries, items, nitem, eg, mom, max_L, st);
}

// ---------------------------------------------------------------------------------------- plan-time kernel
// 1-D Gaussian factors of every brick entry (orthogonal cells), in the order of the entry list: one CTA per
// brick, one thread per table value, direct exp() (Eq. 24-25 give the same values by recursion):
//   [ gy(i) = exp(-a_p Gm22 (o2 + i + s2 N2 - nP2)^2), i < 4 BR2 | gz(i), i < 4 BR3 | gx(x), x < 4 ]
namespace {
__global__ void __launch_bounds__(128) k_entry_gauss(const __grid_constant__ GridParams P, const TaskK *__restrict__ tasks,
                                                     const BEntry *__restrict__ entries, double *__restrict__ eg) {
    int brick = blockIdx.x, level = 0;
    while (brick >= P.lev[level].nbrick) { brick -= P.lev[level].nbrick; level++; }
    const LevelGeom &g = P.lev[level];
    const long long lo = P.brick_base[level][brick], hi = P.brick_base[level][brick + 1];
    const int B2 = g.B[2], B1n = g.B[1];
    const int org[3] = {4 * BR1 * (brick / (B2 * B1n)), 4 * BR2 * ((brick / B2) % B1n), 4 * BR3 * (brick % B2)};
    for (long long i = threadIdx.x; i < (hi - lo) * EG; i += blockDim.x) {
        const long long e = lo + i / EG;
        const int v = (int)(i % EG);
        const int axis = v < GT2 ? 1 : (v < GT2 + GT3 ? 2 : 0);
        const int idx = axis == 1 ? v : (axis == 2 ? v - GT2 : v - GT2 - GT3);
        const BEntry en = entries[e];
        const TaskK &k = tasks[en.task];
        const double u = (double)(org[axis] + idx + en.s[axis] * g.N[axis]) - k.nP[axis];
        eg[e * EG + v] = exp(-(k.ap * g.Gm[axis] * u * u));
    }
}
}  // namespace

size_t entry_gauss_doubles(bool ortho) { return ortho ? (size_t)EG : 0; }

cudaError_t launch_entry_gauss(const GridParams &P, int nbrick_all, const TaskK *tasks, const BEntry *entries, double *eg,
                               cudaStream_t st) {
    if (nbrick_all <= 0) return cudaSuccess;
    k_entry_gauss<<<nbrick_all, 128, 0, st>>>(P, tasks, entries, eg);
    return cudaGetLastError();
}

}  // namespace gpw
