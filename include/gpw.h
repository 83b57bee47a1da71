/*
 * gpw.h -- C ABI of the B200-native multigrid Gaussian-Plane-Wave hot path.
 *
 * Operations (citations are lines of the paper's text, /root/reference/PAPER.md,
 * with the equation / algorithm they fall in; "DESIGN.md Tn / An" are the
 * readings of the paper listed in DESIGN.md):
 *
 *   gpw_build_pairs   shell cutoff radii (Eq. 20), pair screening
 *                     and lattice-image lists (Eq. 18-19; Alg. 4,
 *                     PAPER.md:435-479), level assignment by pair exponent
 *                     (PAPER.md:59), pair -> 4x4x4 grid-block lists (Alg. 5,
 *                     PAPER.md:485-561).
 *   gpw_eval_rho      density collocation, Eq. (3) PAPER.md:41 / Alg. 1
 *                     PAPER.md:204-234, on every level's grid; deriv=1 adds the
 *                     exact real-space gradient (Eq. 10 is its G-space form,
 *                     PAPER.md:76-82).
 *   gpw_eval_mat      potential integration, Eq. (4) PAPER.md:45 with the quadrature
 *                     weight of Eq. (29) PAPER.md:185 / Alg. 2 PAPER.md:240-263;
 *                     deriv=1 adds the Eq. (11) term sum_r w(r) . grad(phi_mu phi_nu)
 *                     (before the integration by parts of Eq. 13).
 *                     deriv=2 (meta-GGA) adds a fifth component to both: the kinetic-energy
 *                     density tau = 1/2 sum D grad phi_mu . grad phi_nu (Eq. 15)
 *                     and the term dV sum_r v_tau(r) 1/2 grad phi_mu . grad phi_nu of the Fock
 *                     matrix (Eq. 16, with the 1/2 of PAPER.md:265-268).
 *   gpw_eval_grad     nuclear gradient of the grid energy at fixed potential (Alg. 3,
 *                     PAPER.md:272-309).
 *   gpw_interp_up / gpw_restrict_down
 *                     inter-level Fourier combination, Eq. (7)-(8) PAPER.md:61-68
 *                     (cuFFT, off the optimisation target).
 *
 * Conventions
 *   - All functions return GPW_OK (0) or a negative gpw_status; they never throw,
 *     exit or print.  gpw_last_error() gives a thread-local message.
 *   - "host" / "device" on every pointer says where the memory lives.  The caller
 *     owns every buffer it passes; the library copies what it needs into the plan
 *     and keeps no caller pointer after a call returns.
 *   - Basis (Eq. 21-22): primitive k of a shell of angular
 *     momentum l centred at A is coef_k x^lx y^ly z^lz exp(-a_k |r-A|^2),
 *     lx+ly+lz = l; coef multiplies the bare primitive as is (normalisation is the
 *     caller's business, A1).  AO order: shells in input order, within a
 *     shell the Cartesian components with decreasing lx, then decreasing ly
 *     (s; x y z; xx xy xz yy yz zz; xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz; A2).
 *   - Grids (PAPER.md:483 with u0 = 0): level alpha has mesh (N1,N2,N3), points
 *     r_n = (n1/N1) a1 + (n2/N2) a2 + (n3/N3) a3; arrays are [ncomp][N1][N2][N3]
 *     doubles, C order (n3 fastest), ncomp = 1 (deriv=0), 4 (deriv=1: value,
 *     d/dx, d/dy, d/dz; component-major) or 5 (deriv=2: those four, then tau / v_tau).
 *   - Truncation (T1-T7): a primitive pair is evaluated on all 64 points
 *     of every aligned 4x4x4 grid block that has at least one point within the pair
 *     radius R_t of the Gaussian-product centre; out-of-cell blocks are folded back
 *     (Eq. 18-19).
 *   - eval calls are asynchronous on the given CUDA stream, allocate nothing
 *     visible to the caller and do not synchronise.  Results may differ from run to
 *     run at the 1e-15 level (floating-point atomics).
 *   - Concurrency: the eval / interp calls write workspaces owned by the plan (pair
 *     polynomials, pair moments, FFT scratch).  Calls on ONE plan are therefore
 *     serialised on the device: each call makes its stream wait for the previous
 *     call on the same plan, whichever stream that ran on, so issuing them on
 *     different streams is safe but gives no overlap; use one plan per concurrent
 *     pipeline.  A plan must not be used from two host threads at the same time.
 *     The current CUDA device of an eval call must be the device the plan was built
 *     on (GPW_EINVAL otherwise).
 *   - Alignment: every level pointer (rho_dev[a], v_dev[a]) must be 16-byte aligned
 *     (the kernels use 16-byte loads and stores); D_dev / F_dev 8-byte.
 *   - Size cap: the plan holds geometry-only tables of about 112 bytes per
 *     (pair, block) visit (gpw_info.device_bytes: 4 GB for 256 waters, 24 GB for 512
 *     waters with f shells); gpw_build_pairs returns GPW_ENOMEM when they do not fit.
 */
#ifndef GPW_H
#define GPW_H

#ifdef __cplusplus
extern "C" {
#endif

#define GPW_MAX_LEVEL 8
#define GPW_MAX_L 3

typedef struct gpw_plan gpw_plan; /* opaque; owned by the library; freed by gpw_free_plan */

typedef enum {
    GPW_OK = 0,
    GPW_EINVAL = -1,       /* null pointer, l > 3, exponent/tau <= 0, singular cell (|det| < 1e-12),
                              mesh entry not a positive multiple of 4, a level finer than level 0 on some axis,
                              deriv out of range, nlevel > 8, misaligned level pointer, wrong current device */
    GPW_ENOMEM = -2,
    GPW_ECUDA = -3,        /* a CUDA / cuFFT call failed, or the plan has no device copy */
    GPW_EUNSUPPORTED = -4  /* l >= 4, more lattice wraps than the visit encoding holds, a pair so sharp
                              that its Gaussian underflows inside its own grid blocks (a_p (R_t + block
                              diagonal)^2 > 600: the mesh is far too coarse for the basis) */
} gpw_status;

/* Plan summary (host struct filled by gpw_plan_info). */
typedef struct {
    int nao, nshl, nlevel, hermi, on_device;
    long ntask;                               /* primitive pairs (a, b, T) kept (unordered if hermi) */
    long ntask_level[GPW_MAX_LEVEL];
    long nvisit_level[GPW_MAX_LEVEL];         /* (pair, 4x4x4 block) visits */
    long nvisit_class[GPW_MAX_LEVEL][GPW_MAX_L + 1][GPW_MAX_L + 1]; /* per (la, lb); points = 64 * visits */
    long nitem;                               /* work items (block, visit range) of the kernels */
    long ncoef_total;                         /* doubles in the per-pair polynomial workspace */
    double build_seconds;                     /* host time spent in gpw_build_pairs */
    long device_bytes;                        /* device memory held by the plan */
} gpw_info;

/* One kept primitive pair (host struct filled by gpw_plan_export_tasks). */
typedef struct {
    int shl_a, prim_a, shl_b, prim_b;  /* shell index, global primitive index */
    int T[3];                          /* lattice translation applied to b */
    int level;
    double R;                          /* pair radius R_t (T4) */
} gpw_task;

/* One (pair, lattice image, 4x4x4 block) visit of the plan's lists (host struct filled by gpw_plan_export_visits). */
typedef struct {
    int task;       /* index of the pair in the order of gpw_plan_export_tasks */
    int block[3];   /* UNWRAPPED block coordinates beta_i = floor(n_i / 4) on the pair's level (T6);
                       the stored block is beta mod (N / 4) */
} gpw_visit;

/*
 * Screening, radii, level assignment, lattice images and block lists.
 * All pointer arguments are HOST memory.
 *   cell        [9]  row-major, rows = lattice vectors a1, a2, a3 (Bohr)
 *   xyz         [natm][3] Bohr, used as given (need not lie inside the cell)
 *   shl_atom    [nshl] centre index;  shl_l [nshl] 0..3;  shl_nprim [nshl] >= 1;
 *   shl_prim_off[nshl] offset of the shell's first primitive in prim_exp / prim_coef
 *   prim_exp    [nprim] Bohr^-2, > 0;  prim_coef [nprim]
 *   mesh        [nlevel][3], finest level first (no level may exceed level 0 on any axis), every entry a
 *               positive multiple of 4
 *   tau         threshold of Eq. (20);  rel_cutoff  level-assignment constant (T5):
 *               a pair goes to the coarsest level with E_alpha >= rel_cutoff * a_p
 *   hermi       1: D and F symmetric, unordered pairs processed once;  0: ordered pairs
 * On success *plan_out holds a plan with a device copy on the current CUDA device.
 * If no CUDA device is usable the plan is host-only (info.on_device = 0): it serves
 * gpw_plan_info / gpw_plan_export_tasks, and every eval call on it fails with
 * GPW_ECUDA (there is no CPU fallback).  May synchronise the device.
 */
int gpw_build_pairs(const double *cell, int natm, const double *xyz, int nshl, const int *shl_atom,
                    const int *shl_l, const int *shl_nprim, const int *shl_prim_off,
                    const double *prim_exp, const double *prim_coef, int nlevel, const int *mesh,
                    double tau, double rel_cutoff, int hermi, gpw_plan **plan_out);

/*
 * Collocation.  D_dev: DEVICE [nao][nao] row-major (read only).  deriv: 0, 1 or 2 (the first call with
 * deriv = 2 allocates the plan's degree-(L+2) workspace).
 * rho_dev: HOST array of nlevel DEVICE pointers, each [ncomp][N1][N2][N3]; every level
 * is OVERWRITTEN (levels without pairs are zero-filled).  cuda_stream: a cudaStream_t
 * (NULL = default stream).  With hermi = 1 the pair (a,b) uses D_ab + D_ba, so the
 * result equals the ordered double sum of Eq. (3) for any D.
 */
int gpw_eval_rho(const gpw_plan *plan, const double *D_dev, int deriv, double *const *rho_dev,
                 void *cuda_stream);

/*
 * Integration.  v_dev: HOST array of nlevel DEVICE pointers, each [ncomp][N1][N2][N3]
 * (component 0 = v, components 1..3 = the vector field w contracted with
 * grad(phi_mu phi_nu)).  F_dev: DEVICE [nao][nao] row-major, OVERWRITTEN, includes
 * dV = Omega / (N1 N2 N3) of each level and the sum over levels.  With hermi = 1 both
 * triangles are written.  deriv = 2: component 4 = v_tau, contracted with 1/2 grad phi_mu . grad phi_nu.
 */
int gpw_eval_mat(const gpw_plan *plan, const double *const *v_dev, int deriv, double *F_dev,
                 void *cuda_stream);

/*
 * Integration without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops,
 * harnesses that forbid it): gpw_eval_mat with the same arguments and the same result, whose scratch -- the moment
 * workspace the integration kernel accumulates into and the post-pass reads, m[pair][k] = sum_n w(n) G(n) u^k,
 * PAPER.md:238-282 (Alg. 2) -- is a static device array inside the library instead of plan-owned memory.  The call makes
 * no cudaMalloc / cudaFree and uses no allocating library routine.
 *   Limit: the plan's moment workspace, gpw_info.ncoef_total doubles (deriv = 2: that, rounded up to a multiple of 32,
 *   plus the degree-(L+2) moments, about 2.4 times as much in all), must fit GPW_STATIC_MOM_DOUBLES doubles (16 MiB,
 *   held by every GPU that loads the library until the process exits); a larger plan is rejected with GPW_EUNSUPPORTED
 *   before anything is launched -- use gpw_eval_mat for it.
 *   The array is one per device and shared by EVERY call and every plan; it keeps the previous call's contents, so each
 *   call clears the part it uses on cuda_stream first.  Calls on one plan are ordered by the plan as for gpw_eval_mat;
 *   calls on DIFFERENT plans that overlap on the GPU (different streams) race on the array -- the caller orders them.
 */
#define GPW_STATIC_MOM_DOUBLES (1L << 21)
int gpw_eval_mat_static(const gpw_plan *plan, const double *const *v_dev, int deriv, double *F_dev,
                        void *cuda_stream);

/*
 * Host-buffer variants: the same two operations with every array in HOST memory (D_host [nao][nao]; rho_host /
 * v_host: HOST arrays of nlevel HOST pointers [ncomp][N1][N2][N3]; F_host [nao][nao]).  The library uploads the
 * inputs into staging buffers it owns, runs the kernels and downloads the results, on three streams of its own
 * (upload, kernels, download) so that the copies of one call overlap the kernels and the opposite copies of its
 * neighbours: an upload never waits for a download.  Pinned host memory (cudaHostAlloc / cudaHostRegister) is
 * needed for that overlap; pageable memory works but serialises.
 * Ordering: a call starts after the work already queued on cuda_stream; its OUTPUTS ARE COMPLETE only after
 * gpw_plan_wait(plan, s) has been passed on a stream s (or the device has been synchronised) -- the caller's stream
 * is not made to wait at the end of the call, so that successive calls pipeline.  Input buffers may be reused
 * after the same point.  First use allocates the staging buffers (gpw_info.device_bytes).
 */
int gpw_eval_rho_host(gpw_plan *plan, const double *D_host, int deriv, double *const *rho_host, void *cuda_stream);
int gpw_eval_mat_host(gpw_plan *plan, const double *const *v_host, int deriv, double *F_host, void *cuda_stream);
/* Makes cuda_stream wait for every host-buffer call issued so far on the plan (their downloads included). */
int gpw_plan_wait(gpw_plan *plan, void *cuda_stream);

/*
 * Sharding over processes, one GPU each: after gpw_plan_set_partition(plan, rank, nranks)
 * the eval calls of this plan work on the slab of grid-block rows along n1 that `rank` owns on every level -- rows
 * [T1 rank / nranks, T1 (rank + 1) / nranks) of the T1 = N1 / 4 rows, i.e. grid indices n1 in [n1_lo, n1_hi) as
 * gpw_plan_partition_bounds returns them (HOST pointers).  Every process builds the same plan (pairs and lists are
 * replicated) and passes full-size arrays:
 *   gpw_eval_rho   writes the owned slab of every level and zero-fills the rest: no exchange is needed for rho, the
 *                  slabs of the ranks are disjoint;
 *   gpw_eval_mat / gpw_eval_grad   read v only inside the owned slab and return this rank's PARTIAL F / gradient:
 *                  the caller sums them over the ranks (one all-reduce, e.g. NCCL through torch.distributed).
 * rank = 0, nranks = 1 (the default) restores the whole.
 */
int gpw_plan_set_partition(gpw_plan *plan, int rank, int nranks);
int gpw_plan_partition_bounds(const gpw_plan *plan, int level, int rank, int nranks, int *n1_lo, int *n1_hi);

/*
 * Nuclear gradient (Alg. 3) of the grid energy
 *     E = sum_alpha dV_alpha sum_r [ v0(r) rho_alpha(r) + w(r) . grad rho_alpha(r) ]
 * at FIXED v0, w and fixed visit set, rho_alpha being the collocated density of gpw_eval_rho:
 *     grad[A][c] = dE / dR_{A,c},   d/dR_A phi(r - R_A) = -grad_r phi   (a lattice image moves with its atom).
 * v_dev as in gpw_eval_mat with deriv = 0 (v0 only) or 1 (v0 and w); D_dev: DEVICE [nao][nao];
 * grad_dev: DEVICE [natm][3], OVERWRITTEN.  The first call allocates the plan's degree-(L+1) workspace.
 */
int gpw_eval_grad(gpw_plan *plan, const double *const *v_dev, int deriv, const double *D_dev, double *grad_dev,
                  void *cuda_stream);

/*
 * Off-target helpers (cuFFT), Eq. (7)-(8):
 *   up:   rho_fine = IFFT( sum_alpha [FFT(rho_alpha)]_{|G| < G_alpha} ) on the finest mesh
 *   down: v_alpha  = IFFT( [FFT(v_fine)]_{|G| < G_alpha} )   (the exact adjoint of up)
 * G_alpha = min_i pi N_alpha,i |b_i| (inscribed sphere; excludes Nyquist planes; A17).
 * rho_dev / v_dev: HOST arrays of nlevel DEVICE pointers [ncomp][N1][N2][N3];
 * rho_fine_dev / v_fine_dev: DEVICE [ncomp] arrays on the finest (level 0) mesh.
 * These allocate cuFFT plans and scratch inside the plan on first use.
 */
int gpw_interp_up(gpw_plan *plan, const double *const *rho_dev, int ncomp, double *rho_fine_dev,
                  void *cuda_stream);
int gpw_restrict_down(gpw_plan *plan, const double *v_fine_dev, int ncomp, double *const *v_dev,
                      void *cuda_stream);

/*
 * G-space operators of the Fock build on the FINEST mesh (cuFFT + one pointwise kernel each; off target):
 *   gpw_hartree            v_H(r) = sum_{G != 0} 4 pi / |G|^2 F(rho)(G) exp(i G . r)      Eq. (5)-(6)
 *   gpw_gspace_gradient    grad rho (r) = sum_G i G F(rho)(G) exp(i G . r)                Eq. (10)
 *   gpw_gspace_divergence  div w (r) = sum_G i G . F(w)(G) exp(i G . r)                   Eq. (14)
 * G_m = 2 pi sum_i m_i b_i, b_i = i-th column of inverse(cell); plane waves on a Nyquist plane |m_i| = N_i / 2 are
 * dropped (A26).  All pointers DEVICE, 16-byte aligned, on the level-0 mesh: rho / v_H / div [N1][N2][N3],
 * grad / w [3][N1][N2][N3]; outputs OVERWRITTEN; in and out must not overlap.
 */
int gpw_hartree(gpw_plan *plan, const double *rho_fine_dev, double *vh_fine_dev, void *cuda_stream);
int gpw_gspace_gradient(gpw_plan *plan, const double *rho_fine_dev, double *grad_fine_dev, void *cuda_stream);
int gpw_gspace_divergence(gpw_plan *plan, const double *w_fine_dev, double *div_fine_dev, void *cuda_stream);

/* Introspection (host). */
int gpw_plan_info(const gpw_plan *plan, gpw_info *out);
/* Copies up to cap tasks into host_buf (may be NULL with cap = 0); *ntask = total. */
int gpw_plan_export_tasks(const gpw_plan *plan, gpw_task *host_buf, long cap, long *ntask);

/* Copies up to cap visits of the collocation lists into host_buf (may be NULL with cap = 0); *nvisit = total.
 * Order: level, stored block, then list order.  Reads the lists back from the device (synchronises). */
int gpw_plan_export_visits(const gpw_plan *plan, gpw_visit *host_buf, long cap, long *nvisit);

/*
 * Measurement aid: with timing enabled the eval calls bracket each of their kernels with CUDA events on
 * the call's stream (no synchronisation is added).  gpw_plan_get_timing waits for the last call of the
 * given kind (which = 0: gpw_eval_rho, 1: gpw_eval_mat) and writes two durations in milliseconds to the
 * HOST array ms_out[2]:  which = 0: {pre-pass D -> pair polynomials, collocation kernel};
 * which = 1: {integration kernel, post-pass pair moments -> F}.
 */
int gpw_plan_set_timing(gpw_plan *plan, int enable);
int gpw_plan_get_timing(gpw_plan *plan, int which, float *ms_out);

/*
 * Measurement aid: FP64 FMA throughput of the current device (register-only DFMA loop on every SM, 8
 * independent chains per thread, best launch over at least min_seconds), in TFLOP/s.  The denominator
 * of the "alu" roofline that bench.py reports.  Host pointers; synchronises the device.
 */
int gpw_dfma_peak(double min_seconds, double *tflops_out, int *sm_count_out);

/*
 * Measurement aid: the same for the FP64 tensor-core path (mma.sync.m8n8k4.f64, eight independent accumulator tiles
 * per warp): TFLOP/s of DMMA alone and of DMMA with DFMA chains issued in the same loop (flops counted per
 * instruction issued).  The evidence behind "FP64 CUDA cores, not DMMA".  Host pointers.
 */
int gpw_dmma_peak(double min_seconds, double *tflops_dmma_out, double *tflops_mixed_out);

void gpw_free_plan(gpw_plan *plan);
const char *gpw_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GPW_H */
