// Declarations shared by the CUDA translation units (collocate.cu, integrate.cu, gpw_api.cu).
#pragma once
#include <cuda_runtime.h>

#include "gpw_math.cuh"

namespace gpw {

// Kernel parameters: geometry and per-level lists (lives in the constant bank).
struct GridParams {
    LevelGeom lev[GPW_MAX_LEVEL];
    const long long *tile_base[GPW_MAX_LEVEL];   // collocation: per block, start of its visit list
    const unsigned *seg[GPW_MAX_LEVEL];          // collocation: per block, start of each L segment
    const long long *brick_base[GPW_MAX_LEVEL];  // integration: per brick, start of its entry list
    double *grid[GPW_MAX_LEVEL];                 // rho (written) or v (read)
    int part_lo[GPW_MAX_LEVEL], part_hi[GPW_MAX_LEVEL];   // block rows [lo, hi) along n1 this process owns (gpw_plan_set_partition)
    long long coef_base[GPW_MAX_LEVEL][8];       // workspace offset of pair i of class (level, L) = base + i * ncoef_pad(L + off),
                                                 // off = the degree offset of the launch
};

// Pair record as the kernels use it.
struct PairRec {
    double nP0, nP1, nP2, ap, c22, c23, c33;
};

// cp.async helpers (records staged in shared memory ahead of their use)
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

// launchers (each picks the instantiation for the plan's largest L; ortho: every level's Gm is diagonal)
// rec: per-pair records of the collocation kernel, header (8 doubles: nP[3], a_p, c22, c23, c33, 0) followed
// by the pair polynomial; the record of pair i of class (level, L) starts at coef_base[level][L] + i * (8 + ncoef_pad(L))
// vg: Gaussian values of every visit (visit_gauss_doubles(ortho) per visit, order of `visits`), written once per
// plan by launch_visit_gauss
// off: degree offset of the launch (0, or 2 with deriv = 0: kinetic-energy density); rec and P.coef_base are those of `off`
// items_hi: the items over the visits of the classes L >= 5 alone (plans with f shells; the second launch of deriv = 1)
cudaError_t launch_collocate(const GridParams &P, const Visit *visits, const Item *items, int nitem,
                             const Item *items_hi, int nitem_hi,
                             const double *rec, const double *vg, int deriv, int off, int max_L, bool ortho, cudaStream_t st);
size_t visit_gauss_doubles(bool ortho);
cudaError_t launch_visit_gauss(const GridParams &P, int ntile_all, const TaskK *tasks, const Visit *visits, double *vg,
                               bool ortho, cudaStream_t st);
// eg: 1-D Gaussian factor tables of every brick entry (entry_gauss_doubles(ortho) per entry, order of `entries`;
// orthogonal cells only, else unused), written once per plan by launch_entry_gauss
// off: degree offset (0; 1 with deriv 0 / 1: nuclear gradient; 2 with deriv = 0: kinetic-energy potential); the moments of
// pair i of class (level, L) are added at mom + P.coef_base[level][L] + i * ncoef_pad(L + off)
cudaError_t launch_integrate(const GridParams &P, const TaskK *tasks, const BEntry *entries, const BItem *items,
                             int nitem, const double *eg, double *mom, int deriv, int off, int max_L, bool ortho, cudaStream_t st);
size_t entry_gauss_doubles(bool ortho);
cudaError_t launch_entry_gauss(const GridParams &P, int nbrick_all, const TaskK *tasks, const BEntry *entries, double *eg,
                               cudaStream_t st);

// pairpass.cu: pre- and post-pass (pairpass.cuh); max_l = the largest shell angular momentum of the plan
// and max_L the largest la + lb.  The classes la + lb <= REG_LMAX of the hot path (degree offset 0) go through the
// register form (pairpass_reg*.cu), one translation unit per direction.
namespace pp { struct PassArgs; }
constexpr int REG_LMAX = 4;
cudaError_t launch_pair_pass(const pp::PassArgs &A, int max_l, int max_L, cudaStream_t st);
cudaError_t launch_pair_reg_pre(const pp::PassArgs &A, cudaStream_t st);
cudaError_t launch_pair_reg_post(const pp::PassArgs &A, cudaStream_t st);

// interp.cu: Eq. (7)-(8) with cuFFT; the state (plans, scratch) is created on first use; return a gpw_status
struct InterpState;
int interp_up(const HostPlan *hp, InterpState **st, const double *const *rho, int ncomp, double *fine, cudaStream_t s);
int interp_down(const HostPlan *hp, InterpState **st, const double *fine, int ncomp, double *const *v, cudaStream_t s);
// kind 0: Hartree potential (in, out [N]); 1: gradient (in [N], out [3][N]); 2: divergence (in [3][N], out [N]); finest mesh
int gspace_apply(const HostPlan *hp, InterpState **st, int kind, const double *in, double *out, cudaStream_t s);
void interp_free(InterpState *st);
long interp_bytes(const InterpState *st);

}  // namespace gpw
