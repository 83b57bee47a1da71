// Kernel of the register form (pairpass_reg.cuh), compiled once per direction in its own translation unit
// (pairpass_reg_pre.cu, pairpass_reg_post.cu).  One thread per pair; pairs are sorted by (level, L, la), so a warp's
// threads are in the same class except at class boundaries.  Every class body is a function of its own (noinline:
// ptxas then allocates registers per class instead of over one kernel holding all thirteen unrolled bodies, which
// took it ten minutes).  Pairs of the classes la + lb > REG_LMAX are left to the general kernel (pairpass.cu).
#pragma once
#include "gpw_kernels.cuh"
#include "pairpass_reg.cuh"

namespace gpw {
namespace {

constexpr int PR_THREADS = 128;

struct RegArgs {
    const double *S, *D, *m;
    double *out, *F;
    double scale;
    int nao;
};

template <int LA, int LB, bool POST>
__device__ __noinline__ void pair_reg_class(const TaskP &p, const RegArgs &a) {
    if (POST) ppr::post_mat<LA, LB, false>(p, a.m, a.S, a.scale, a.F, a.nao);
    else ppr::pre_dens<LA, LB, false>(p, a.D, a.nao, a.S, a.out);
}

template <bool POST>
__global__ void __launch_bounds__(PR_THREADS) k_pair_reg(const __grid_constant__ pp::PassArgs A) {
    const int t = blockIdx.x * PR_THREADS + threadIdx.x;
    if (t >= A.ntask) return;
    const TaskP p = A.tp[t];
    const int L = p.la + p.lb;
    if (L > REG_LMAX) return;
    const long long off = A.base[0][p.level][L] + (long long)t * ncoef_pad(L);
    RegArgs a;
    a.S = A.S_all + (size_t)p.level * S_TOTAL;
    a.D = A.D; a.F = A.F; a.nao = A.nao;
    a.out = A.rec[0] + off + 8 * (long long)t + 8;
    a.m = A.mom[0] + off;
    a.scale = p.pref * A.dV[p.level];
#define GPW_CASE(LA, LB)                                                    \
    case LA * 4 + LB:                                                       \
        if constexpr (LA + LB <= REG_LMAX) pair_reg_class<LA, LB, POST>(p, a); \
        break;
    switch (p.la * 4 + p.lb) {
        GPW_CASE(0, 0) GPW_CASE(0, 1) GPW_CASE(0, 2) GPW_CASE(0, 3)
        GPW_CASE(1, 0) GPW_CASE(1, 1) GPW_CASE(1, 2) GPW_CASE(1, 3)
        GPW_CASE(2, 0) GPW_CASE(2, 1) GPW_CASE(2, 2) GPW_CASE(2, 3)
        GPW_CASE(3, 0) GPW_CASE(3, 1) GPW_CASE(3, 2) GPW_CASE(3, 3)
        default: break;
    }
#undef GPW_CASE
}

template <bool POST>
cudaError_t launch_pair_reg_t(const pp::PassArgs &A, cudaStream_t st) {
    k_pair_reg<POST><<<(A.ntask + PR_THREADS - 1) / PR_THREADS, PR_THREADS, 0, st>>>(A);
    return cudaGetLastError();
}

}  // namespace
}  // namespace gpw
