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

// LS: the largest shell angular momentum the instantiation holds: q [ncart(LS)][ncoef(LS)], R of degree 2 LS + off, off the
// largest degree offset of the launch's modes (0: density / Fock matrix, 1: nuclear gradient, 2: tau) -- sized per launch,
// because the shared memory is what limits the resident groups (LS = 3: 285 doubles per group on the hot path, 366 for tau)
template <int LS>
GPW_CX int group_doubles(int off) { return ncart(LS) * ncoef(LS) + ncoef(2 * LS + off) + 1; }

__device__ Tables d_tables;   // index tables (pairpass.cuh), written once per process and device by upload_tables

template <int LS>
__global__ void __launch_bounds__(PP_THREADS) k_pair_pass(const __grid_constant__ PassArgs A, int gdoubles) {
    extern __shared__ double sm[];
    __shared__ Tables s_tab;
    {
        static_assert(sizeof(Tables) % 2 == 0, "copied as 16-bit words");
        const unsigned short *src = reinterpret_cast<const unsigned short *>(&d_tables);
        unsigned short *dst = reinterpret_cast<unsigned short *>(&s_tab);
        for (int i = threadIdx.x; i < (int)(sizeof(Tables) / 2); i += PP_THREADS) dst[i] = src[i];
    }
    __syncthreads();
    const int grp = threadIdx.x / PP_G;
    const int j = blockIdx.x * PP_GROUPS + grp;
    if (j >= A.nsel) return;    // whole groups leave: the group's lanes synchronise among themselves only
    int r = 0;
    while (j >= A.sel_cum[r + 1]) r++;
    const int t = A.sel_lo[r] + (j - A.sel_cum[r]);
    Grp g;
    g.gl = threadIdx.x % PP_G;
    g.G = PP_G;
    g.mask = 0xffu << (8 * ((threadIdx.x & 31) / PP_G));
    g.tab = &s_tab;
    double *q = sm + (size_t)grp * gdoubles;
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
    {   // the index tables, once per device
        static bool ready[64] = {false};
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
        if (dev < 0 || dev >= 64 || !ready[dev]) {
            static Tables host_tab;
            fill_tables(host_tab);
            const cudaError_t e = cudaMemcpyToSymbolAsync(d_tables, &host_tab, sizeof(Tables), 0, cudaMemcpyHostToDevice, st);
            if (e != cudaSuccess) return e;
            if (dev >= 0 && dev < 64) ready[dev] = true;
        }
    }
    static_assert(REG_LMAX == 4, "big_lo / big_n list the classes la + lb >= 5");
    // the pairs of this launch: all of them for the derivative variants, else only the classes the register form left
    A.nsel = 0;
    if (A.mode & ~(PRE_DENS | POST_MAT)) {
        A.sel_lo[0] = 0;
        A.nsel = A.ntask;
        for (int a = 1; a <= GPW_MAX_LEVEL; a++) A.sel_cum[a] = A.ntask;
        A.sel_cum[0] = 0;
    } else {
        for (int a = 0; a < GPW_MAX_LEVEL; a++) {
            A.sel_cum[a] = A.nsel;
            A.sel_lo[a] = A.big_lo[a];
            A.nsel += A.big_n[a];
        }
        A.sel_cum[GPW_MAX_LEVEL] = A.nsel;
    }
    if (A.nsel == 0) return cudaSuccess;
    const int nblk = (A.nsel + PP_GROUPS - 1) / PP_GROUPS;
    const int off = (A.mode & (PRE_TAU | POST_TAU)) ? 2 : ((A.mode & POST_GRAD) ? 1 : 0);
    static_assert(NOFF == 3, "degree offsets 0, 1, 2");
    if (max_l <= 2) {
        const int gd = group_doubles<2>(off);
        k_pair_pass<2><<<nblk, PP_THREADS, PP_GROUPS * gd * sizeof(double), st>>>(A, gd);
    } else {
        const int gd = group_doubles<3>(off);
        k_pair_pass<3><<<nblk, PP_THREADS, PP_GROUPS * gd * sizeof(double), st>>>(A, gd);
    }
    return cudaGetLastError();
}

}  // namespace gpw
