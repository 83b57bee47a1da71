// Kernels of the pre- and post-pass (pairpass.cuh): a group of eight lanes per primitive pair, the pair's
// polynomials in the group's shared memory.
#include "gpw_kernels.cuh"
#include "pairpass.cuh"

namespace gpw {
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

cudaError_t launch_pair_pass(const pp::PassArgs &A, int max_l, cudaStream_t st) {
    if (A.ntask <= 0) return cudaSuccess;
    const int nblk = (A.ntask + PP_GROUPS - 1) / PP_GROUPS;
    if (max_l <= 2) k_pair_pass<2><<<nblk, PP_THREADS, PP_GROUPS * group_doubles<2>() * sizeof(double), st>>>(A);
    else k_pair_pass<3><<<nblk, PP_THREADS, PP_GROUPS * group_doubles<3>() * sizeof(double), st>>>(A);
    return cudaGetLastError();
}

}  // namespace gpw
