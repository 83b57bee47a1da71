// Collocation kernel (Eq. 3; the work of Alg. 1, re-decomposed for B200).
//
// One warp per work item = one 4x4x4 grid block and a range of its visit list.  A half-warp evaluates
// one (pair, block) visit at a time, a lane owns a column of 4 grid points along n3 and keeps its rho
// values (and, for DERIV, the gradient in grid-index components) in registers for the whole list, so
// the block is written once (the theoretical minimum the paper aims at) and no
// cross-thread reduction per point is needed (the bottleneck of Alg. 1 l.11).  The next
// visit's pair record is fetched while the current one is evaluated.
#include "gpw_kernels.cuh"

namespace gpw {
namespace {

struct ColCtx {
    const TaskK *tasks;
    const Visit *visits;   // already offset to the block's list
    const double *work;    // pair polynomials
    double gm[6];
    int n1, n2, n3;        // stored index of the lane's column start
    int N0, N1, N2;
};

struct ColVisit {
    double u1, u2, u30, ap, cc;
    long long coef_off;
};

__device__ __forceinline__ ColVisit load_visit(const ColCtx &c, unsigned v) {
    const Visit vi = c.visits[v];
    const PairRec p = load_pair(c.tasks, vi.task);
    ColVisit r;
    r.u1 = (double)(c.n1 + vi.s[0] * c.N0) - p.nP0;
    r.u2 = (double)(c.n2 + vi.s[1] * c.N1) - p.nP1;
    r.u30 = (double)(c.n3 + vi.s[2] * c.N2) - p.nP2;
    r.ap = p.ap; r.cc = p.cc; r.coef_off = p.coef_off;
    return r;
}

template <int L, int DERIV>
__device__ __forceinline__ void colloc_segment(const ColCtx &c, unsigned lo, unsigned hi, int half,
                                               double (*acc)[4]) {
    unsigned v = lo + half;
    if (v >= hi) return;
    ColVisit cur = load_visit(c, v);
    for (;;) {
        const unsigned vn = v + 2;
        const bool more = vn < hi;
        ColVisit nxt = cur;
        if (more) nxt = load_visit(c, vn);   // in flight while this visit is evaluated
        double q[6];
#pragma unroll
        for (int x = 0; x < 6; x++) q[x] = cur.ap * c.gm[x];
        colloc_column<L, DERIV>(c.work + cur.coef_off, q, cur.cc, cur.u1, cur.u2, cur.u30, acc);
        if (!more) break;
        cur = nxt;
        v = vn;
    }
}

template <int DERIV, int LMAX>
__global__ void __launch_bounds__(128) k_collocate(const __grid_constant__ GridParams P,
                                                    const TaskK *__restrict__ tasks,
                                                    const Visit *__restrict__ visits,
                                                    const Item *__restrict__ items, int nitem,
                                                    const double *__restrict__ coef) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (w >= nitem) return;
    const Item it = items[w];
    const LevelGeom &g = P.lev[it.level];
    const int lane = threadIdx.x & 31, half = lane >> 4, col = lane & 15;
    const int T2 = g.T[2], T1 = g.T[1];
    const int b3 = it.tile % T2, b2 = (it.tile / T2) % T1, b1 = it.tile / (T2 * T1);
    ColCtx c;
    c.tasks = tasks;
    c.visits = visits + P.tile_base[it.level][it.tile];
    c.work = coef;
#pragma unroll
    for (int x = 0; x < 6; x++) c.gm[x] = g.Gm[x];
    c.n1 = 4 * b1 + (col >> 2); c.n2 = 4 * b2 + (col & 3); c.n3 = 4 * b3;
    c.N0 = g.N[0]; c.N1 = g.N[1]; c.N2 = g.N[2];
    const unsigned *seg = P.seg[it.level] + (size_t)it.tile * 8;

    double acc[NCOMP][4];
#pragma unroll
    for (int k = 0; k < NCOMP; k++)
#pragma unroll
        for (int t = 0; t < 4; t++) acc[k][t] = 0.0;

#pragma unroll 1
    for (int L = 0; L <= LMAX; L++) {
        const unsigned lo = max(it.lo, seg[L]), hi = min(it.hi, seg[L + 1]);
        if (lo >= hi) continue;
        switch (L) {
            case 0: colloc_segment<0, DERIV>(c, lo, hi, half, acc); break;
            case 1: colloc_segment<1, DERIV>(c, lo, hi, half, acc); break;
            case 2: colloc_segment<2, DERIV>(c, lo, hi, half, acc); break;
            case 3: if constexpr (LMAX >= 3) colloc_segment<3, DERIV>(c, lo, hi, half, acc); break;
            case 4: if constexpr (LMAX >= 4) colloc_segment<4, DERIV>(c, lo, hi, half, acc); break;
            case 5: if constexpr (LMAX >= 5) colloc_segment<5, DERIV>(c, lo, hi, half, acc); break;
            default: if constexpr (LMAX >= 6) colloc_segment<6, DERIV>(c, lo, hi, half, acc); break;
        }
    }
    // the two half-warps worked on alternate visits of the same block
#pragma unroll
    for (int k = 0; k < NCOMP; k++)
#pragma unroll
        for (int t = 0; t < 4; t++) acc[k][t] += __shfl_xor_sync(0xffffffffu, acc[k][t], 16);
    if (half) return;
    const size_t ng = (size_t)g.N[0] * g.N[1] * g.N[2];
    double *out = P.grid[it.level] + ((size_t)c.n1 * g.N[1] + c.n2) * g.N[2] + c.n3;
    double res[NCOMP][4];
#pragma unroll
    for (int t = 0; t < 4; t++) {
        res[0][t] = acc[0][t];
        if constexpr (DERIV) {
            // gradient: grid-index components -> Cartesian, d/dX_c = sum_i Hinv[i][c] d/du_i
#pragma unroll
            for (int x = 0; x < 3; x++)
                res[1 + x][t] = g.Hinv[0 * 3 + x] * acc[1][t] + g.Hinv[1 * 3 + x] * acc[2][t] +
                                g.Hinv[2 * 3 + x] * acc[3][t];
        }
    }
    if (it.single) {
#pragma unroll
        for (int k = 0; k < NCOMP; k++) {
            double2 *o = reinterpret_cast<double2 *>(out + k * ng);
            o[0] = make_double2(res[k][0], res[k][1]);
            o[1] = make_double2(res[k][2], res[k][3]);
        }
    } else {
#pragma unroll
        for (int k = 0; k < NCOMP; k++)
#pragma unroll
            for (int t = 0; t < 4; t++) atomicAdd(out + k * ng + t, res[k][t]);
    }
}

template <int DERIV, int LMAX>
cudaError_t launch(const GridParams &P, const TaskK *tasks, const Visit *visits, const Item *items, int nitem,
                   const double *coef, cudaStream_t st) {
    k_collocate<DERIV, LMAX><<<(nitem + 3) / 4, 128, 0, st>>>(P, tasks, visits, items, nitem, coef);
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
