// Kernels of the pre- and post-pass (pairpass.cuh): a group of eight lanes per primitive pair, the pair's
// polynomials in the group's shared memory.
#include "gpw_kernels.cuh"
#include "pairpass.cuh"

namespace gpw {

static cudaError_t launch_pair_reg(const pp::PassArgs &A, bool post, cudaStream_t st) {
    return post ? launch_pair_reg_post(A, st) : launch_pair_reg_pre(A, st);
}

namespace {

using namespace pp;

constexpr int PP_THREADS = 128;
constexpr int PP_GROUPS = PP_THREADS / PP_G;

// LS: the largest shell angular momentum the instantiation holds: q [ncart(LS)][ncoef(LS)], R of degree 2 LS + 2
template <int LS>
GPW_CX int group_doubles() { return ncart(LS) * ncoef(LS) + ncoef(2 * LS + NOFF - 1) + 1; }   // odd: groups start in different banks

template <int LS>
__global__ void __launch_bounds__(PP_THREADS) k_pair_pass(const __grid_constant__ PassArgs A) {
    extern __shared__ double sm[];
    const int grp = threadIdx.x / PP_G;
    const int t = blockIdx.x * PP_GROUPS + grp;
    if (t >= A.ntask) return;   // whole groups leave: the group's lanes synchronise among themselves only
    Grp g;
    g.gl = threadIdx.x % PP_G;
    g.G = PP_G;
    g.mask = 0xffu << (8 * ((threadIdx.x & 31) / PP_G));
    double *q = sm + (size_t)grp * group_doubles<LS>();
    pair_pass<ncoef(LS)>(A, t, q, q + ncart(LS) * ncoef(LS), g);
}

}  // namespace

cudaError_t launch_pair_pass(const pp::PassArgs &A0, int max_l, int max_L, cudaStream_t st) {
    if (A0.ntask <= 0) return cudaSuccess;
    // the hot path (degree offset 0) of the classes la + lb <= REG_LMAX in the register form, one thread per pair;
    // the larger classes and the derivative variants in the general form, eight lanes per pair
    pp::PassArgs A = A0;
    A.lmin_hot = 0;
    if (A.mode & PRE_DENS) {
        const cudaError_t e = launch_pair_reg(A, false, st);
        if (e != cudaSuccess) return e;
        A.lmin_hot = REG_LMAX + 1;
    }
    if (A.mode & POST_MAT) {
        const cudaError_t e = launch_pair_reg(A, true, st);
        if (e != cudaSuccess) return e;
        A.lmin_hot = REG_LMAX + 1;
    }
    if (max_L < A.lmin_hot) A.mode &= ~(PRE_DENS | POST_MAT);
    if (A.mode == 0) return cudaSuccess;
    const int nblk = (A.ntask + PP_GROUPS - 1) / PP_GROUPS;
    if (max_l <= 2) k_pair_pass<2><<<nblk, PP_THREADS, PP_GROUPS * group_doubles<2>() * sizeof(double), st>>>(A);
    else k_pair_pass<3><<<nblk, PP_THREADS, PP_GROUPS * group_doubles<3>() * sizeof(double), st>>>(A);
    return cudaGetLastError();
}

}  // namespace gpw
