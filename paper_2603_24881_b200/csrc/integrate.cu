// Integration kernel (Eq. 4 with the quadrature of Eq. 29; the work of Alg. 2,
// PAPER.md:240-263, re-decomposed for B200).
//
// One CTA per work item = one brick of 3x3x3 grid blocks and a range of its entry list; an entry is a
// (pair, lattice image) with the mask of the brick's blocks it visits.  The CTA stages the brick of v in
// shared memory once (for DERIV with the vector field already mapped to grid-index components).  Each
// warp then takes entries: per visited block a half-warp works with a lane per column of 4 points,
// accumulating the pair's moment vector m[k] = sum_r w(r) G(r) u^k in private registers over ALL the
// entry's blocks; one shuffle reduce-scatter over the warp and one atomic add per moment finish the
// entry.  Alg. 2 instead adds nca*ncb values per (pair, block) to global memory;
// amortising over the brick cuts that traffic by the blocks per entry.
#include "gpw_kernels.cuh"

namespace gpw {
namespace {

constexpr int NWARP = 4;

// ---- full-warp reduce-scatter of an N-vector with per-step padding --------------------------------
// After the call lane holds `final_len(N)` sums in m[0..); element i of them is total[off + i] and is
// valid iff i < cnt.
GPW_CX int rs_final_len(int n) {
    for (int b = 0; b < 5; b++) n = n >= 2 ? (n + 1) / 2 : 1;
    return n;
}

template <int LEN, int BIT>
__device__ __forceinline__ void rs_step(double *m, int lane, int &off, int &cnt) {
    if constexpr (BIT >= 1) {
        const bool up = lane & BIT;
        if constexpr (LEN >= 2) {
            constexpr int HALF = (LEN + 1) / 2;
#pragma unroll
            for (int i = 0; i < HALF; i++) {
                const double lo = m[i];
                const double hi = (i + HALF < LEN) ? m[i + HALF] : 0.0;
                const double send = up ? lo : hi;
                const double keep = up ? hi : lo;
                m[i] = keep + __shfl_xor_sync(0xffffffffu, send, BIT);
            }
            off += up ? HALF : 0;
            cnt = up ? cnt - HALF : min(cnt, HALF);
            rs_step<HALF, BIT / 2>(m, lane, off, cnt);
        } else {
            m[0] += __shfl_xor_sync(0xffffffffu, m[0], BIT);
            if (up) cnt = 0;   // the partner with the bit clear owns the sum
            rs_step<1, BIT / 2>(m, lane, off, cnt);
        }
    }
}

struct BrickCtx {
    const TaskK *tasks;
    const BEntry *entries;   // already offset to the brick's list
    const double *vs;        // shared memory brick: [block][comp][64], in-block order h*32 + col*2 + e
    double gm[6];
    int o1, o2, o3;          // stored grid index of the brick origin
    int N0, N1, N2;
};

template <int L, int DERIV>
__device__ __forceinline__ void integ_entry(const BrickCtx &c, const BEntry en, const PairRec pr, int lane,
                                            double *__restrict__ mom) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    constexpr int NC = ncoef(L);
    const int half = lane >> 4, col = lane & 15;
    double q[6];
#pragma unroll
    for (int x = 0; x < 6; x++) q[x] = pr.ap * c.gm[x];
    // column position relative to P for block (0,0,0) of the brick
    const double u1b = (double)(c.o1 + (col >> 2) + en.s[0] * c.N0) - pr.nP0;
    const double u2b = (double)(c.o2 + (col & 3) + en.s[1] * c.N1) - pr.nP1;
    const double u3b = (double)(c.o3 + en.s[2] * c.N2) - pr.nP2;
    double m[NC];
#pragma unroll
    for (int i = 0; i < NC; i++) m[i] = 0.0;
    unsigned mask = en.mask;
    while (mask) {   // warp-uniform: two blocks per trip, one per half-warp
        const int bit0 = __ffs(mask) - 1;
        mask &= mask - 1;
        int bit1 = -1;
        if (mask) { bit1 = __ffs(mask) - 1; mask &= mask - 1; }
        const int my = half ? bit1 : bit0;
        if (my >= 0) {
            const int t1 = my / (BRICK * BRICK), t2 = (my / BRICK) % BRICK, t3 = my % BRICK;
            const double *vb = c.vs + (size_t)my * (NCOMP * 64) + col * 2;
            double vv[NCOMP][4];
#pragma unroll
            for (int k = 0; k < NCOMP; k++) {
                const double2 x0 = *reinterpret_cast<const double2 *>(vb + k * 64);
                const double2 x1 = *reinterpret_cast<const double2 *>(vb + k * 64 + 32);
                vv[k][0] = x0.x; vv[k][1] = x0.y; vv[k][2] = x1.x; vv[k][3] = x1.y;
            }
            integ_column<L, DERIV>(vv, q, pr.c33, u1b + 4 * t1, u2b + 4 * t2, u3b + 4 * t3, m);
        }
    }
    int off = 0, cnt = NC;
    rs_step<NC, 16>(m, lane, off, cnt);
    double *dst = mom + pr.coef_off + off;
#pragma unroll
    for (int i = 0; i < rs_final_len(NC); i++)
        if (i < cnt) atomicAdd(dst + i, m[i]);
}

template <int DERIV, int LMAX>
__global__ void __launch_bounds__(NWARP * 32) k_integrate(const __grid_constant__ GridParams P,
                                                           const TaskK *__restrict__ tasks,
                                                           const BEntry *__restrict__ entries,
                                                           const BItem *__restrict__ items,
                                                           double *__restrict__ mom) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    extern __shared__ __align__(16) double vs[];   // [BRICK_TILES][NCOMP][64]
    const BItem it = items[blockIdx.x];
    const LevelGeom &g = P.lev[it.level];
    const int B2 = g.B[2], B1 = g.B[1];
    const int k3 = it.brick % B2, k2 = (it.brick / B2) % B1, k1 = it.brick / (B2 * B1);
    const size_t ng = (size_t)g.N[0] * g.N[1] * g.N[2];
    const double *vin = P.grid[it.level];
    // ---- stage the brick: one column (4 points x NCOMP) per thread and trip ----
    for (int cidx_ = threadIdx.x; cidx_ < BRICK_TILES * 16; cidx_ += NWARP * 32) {
        const int lt = cidx_ >> 4, col = cidx_ & 15;
        const int t1 = lt / (BRICK * BRICK), t2 = (lt / BRICK) % BRICK, t3 = lt % BRICK;
        const int b1 = BRICK * k1 + t1, b2 = BRICK * k2 + t2, b3 = BRICK * k3 + t3;
        if (b1 >= g.T[0] || b2 >= g.T[1] || b3 >= g.T[2]) continue;   // ragged brick: never referenced
        const double *src = vin + ((size_t)(4 * b1 + (col >> 2)) * g.N[1] + 4 * b2 + (col & 3)) * g.N[2] + 4 * b3;
        double raw[NCOMP][4];
#pragma unroll
        for (int k = 0; k < NCOMP; k++) {
            const double2 *p2 = reinterpret_cast<const double2 *>(src + k * ng);
            const double2 x0 = __ldg(p2), x1 = __ldg(p2 + 1);
            raw[k][0] = x0.x; raw[k][1] = x0.y; raw[k][2] = x1.x; raw[k][3] = x1.y;
        }
        double *dst = vs + (size_t)lt * (NCOMP * 64) + col * 2;
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
                *reinterpret_cast<double2 *>(dst + k * 64) = make_double2(tr[k][0], tr[k][1]);
                *reinterpret_cast<double2 *>(dst + k * 64 + 32) = make_double2(tr[k][2], tr[k][3]);
            }
        } else {
            *reinterpret_cast<double2 *>(dst) = make_double2(raw[0][0], raw[0][1]);
            *reinterpret_cast<double2 *>(dst + 32) = make_double2(raw[0][2], raw[0][3]);
        }
    }
    __syncthreads();

    BrickCtx c;
    c.tasks = tasks;
    c.entries = entries + P.brick_base[it.level][it.brick];
    c.vs = vs;
#pragma unroll
    for (int x = 0; x < 6; x++) c.gm[x] = g.Gm[x];
    c.o1 = 4 * BRICK * k1; c.o2 = 4 * BRICK * k2; c.o3 = 4 * BRICK * k3;
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    unsigned e = it.lo + warp;
    if (e >= it.hi) return;
    BEntry en = c.entries[e];
    PairRec pr = load_pair(tasks, en.task);
    for (;;) {
        const unsigned e2 = e + NWARP;
        const bool more = e2 < it.hi;
        BEntry en2 = en;
        PairRec pr2 = pr;
        if (more) { en2 = c.entries[e2]; pr2 = load_pair(tasks, en2.task); }   // in flight during this entry
        switch (en.L) {
            case 0: integ_entry<0, DERIV>(c, en, pr, lane, mom); break;
            case 1: integ_entry<1, DERIV>(c, en, pr, lane, mom); break;
            case 2: integ_entry<2, DERIV>(c, en, pr, lane, mom); break;
            case 3: if constexpr (LMAX >= 3) integ_entry<3, DERIV>(c, en, pr, lane, mom); break;
            case 4: if constexpr (LMAX >= 4) integ_entry<4, DERIV>(c, en, pr, lane, mom); break;
            case 5: if constexpr (LMAX >= 5) integ_entry<5, DERIV>(c, en, pr, lane, mom); break;
            default: if constexpr (LMAX >= 6) integ_entry<6, DERIV>(c, en, pr, lane, mom); break;
        }
        if (!more) break;
        en = en2; pr = pr2; e = e2;
    }
}

template <int DERIV, int LMAX>
cudaError_t launch(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items, int nitem,
                   double *mom, cudaStream_t st) {
    constexpr int smem = BRICK_TILES * (DERIV ? 4 : 1) * 64 * (int)sizeof(double);
    static bool configured = false;   // per instantiation
    if (!configured) {
        const cudaError_t e = cudaFuncSetAttribute(k_integrate<DERIV, LMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k_integrate<DERIV, LMAX><<<nitem, NWARP * 32, smem, st>>>(P, tasks, entries, items, mom);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_integrate(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items,
                             int nitem, double *mom, int deriv, int max_L, cudaStream_t st) {
    if (deriv) {
        if (max_L <= 2) return launch<1, 2>(P, tasks, entries, items, nitem, mom, st);
        if (max_L <= 4) return launch<1, 4>(P, tasks, entries, items, nitem, mom, st);
        return launch<1, 6>(P, tasks, entries, items, nitem, mom, st);
    }
    if (max_L <= 2) return launch<0, 2>(P, tasks, entries, items, nitem, mom, st);
    if (max_L <= 4) return launch<0, 4>(P, tasks, entries, items, nitem, mom, st);
    return launch<0, 6>(P, tasks, entries, items, nitem, mom, st);
}

}  // namespace gpw
