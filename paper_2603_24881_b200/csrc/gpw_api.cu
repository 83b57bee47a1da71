// The C ABI of include/gpw.h, the pre/post-pass kernels and the FP64 peak probe (sm_100a).
//
// Kernels:
//   k_pair_pass         pairpass.cu: pre-pass (D block -> pair polynomial about P in grid-index coordinates) and
//                       post-pass (pair moments -> F block x dV, or atom gradients), eight lanes per pair
//   k_collocate         collocate.cu
//   k_integrate         integrate.cu
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "gpw_kernels.cuh"
#include "pairpass.cuh"
#include "plan_device.h"

namespace gpw {
const char *last_error_cstr();

// header of every pair's record in a collocation workspace (plan time / first use): the polynomial of degree
// L + off follows it, rewritten by every call
__global__ void __launch_bounds__(128) k_rec_headers(const TaskK *__restrict__ tk, const TaskP *__restrict__ tp, int ntask,
                                                     pp::PassArgs A, int off, double *__restrict__ rec) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntask) return;
    const TaskK k = tk[t];
    const int L = tp[t].la + tp[t].lb, level = tp[t].level;
    double *h = rec + A.base[off][level][L] + (long long)t * (ncoef_pad(L + off) + 8);
    h[0] = k.nP[0]; h[1] = k.nP[1]; h[2] = k.nP[2]; h[3] = k.ap; h[4] = k.c22; h[5] = k.c23; h[6] = k.c33; h[7] = 0.0;
}

// ------------------------------------------------------------------------------------------ FP64 peak probe
// Register-only DFMA loop, 8 independent chains per thread: the denominator of the "alu" roofline.
__global__ void __launch_bounds__(256) k_dfma_peak(double *out, int iters, double seed) {
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-9;
#pragma unroll 1
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < 16; k++) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

// FP64 tensor-core probe: mma.sync.m8n8k4.f64 (DMMA), eight independent accumulator tiles per warp; with_dfma adds
// the DFMA chains of k_dfma_peak to the same loop.  Flops are counted per instruction issued (512 per warp-level DMMA).
__global__ void __launch_bounds__(256) k_dmma_peak(double *out, int iters, double seed, int with_dfma) {
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; k++) { c[k][0] = seed + k; c[k][1] = seed - k; }
    double f0 = seed + threadIdx.x, f1 = f0 + 1, f2 = f0 + 2, f3 = f0 + 3;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 0.999999, m = 0.999999, e = 1e-9;
#pragma unroll 1
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int r = 0; r < 8; r++) {
#pragma unroll
            for (int k = 0; k < 8; k++)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
            if (with_dfma) { f0 = fma(f0, m, e); f1 = fma(f1, m, e); f2 = fma(f2, m, e); f3 = fma(f3, m, e); }
        }
    }
    double s = (f0 + f1) + (f2 + f3);
#pragma unroll
    for (int k = 0; k < 8; k++) s += c[k][0] + c[k][1];
    if (s == 12345.678) out[0] = s;
}

}  // namespace gpw

// =============================================================================================== C ABI
using namespace gpw;

// State of gpw_eval_rho_host / gpw_eval_mat_host: device staging buffers owned by the plan, one stream per copy
// direction and one for the kernels, so that a call's uploads, its kernels and the previous call's downloads overlap.
struct HostIO {
    cudaStream_t s_in = nullptr, s_out = nullptr, s_cmp = nullptr;
    cudaEvent_t call = nullptr;                                             // the caller's stream at the start of a call
    cudaEvent_t D_in = nullptr, rho_done = nullptr, rho_out = nullptr;      // upload of D, collocation, download of rho
    cudaEvent_t v_in = nullptr, mat_done = nullptr, F_out = nullptr;        // upload of v, integration, download of F
    double *D = nullptr, *F = nullptr;
    double *rho[GPW_MAX_LEVEL] = {nullptr}, *v[GPW_MAX_LEVEL] = {nullptr};
    int ncomp = 0;                                                          // components the level buffers hold
    long bytes = 0;
};

struct gpw_plan {
    HostPlan *hp = nullptr;
    bool on_device = false;
    int device = -1;
    long device_bytes = 0;
    // device copies
    TaskK *d_taskK = nullptr;
    TaskP *d_taskP = nullptr;
    gpw_task *d_export = nullptr;   // the pairs as gpw_plan_export_tasks returns them (screened on the device)
    DeviceLists lists;          // visit / brick lists and work items, built on the device (plan_device.cu)
    double *d_S = nullptr;
    // per degree offset (0: Eq. 3-4; 1: nuclear gradient; 2: kinetic-energy density); offsets 1, 2 allocated on first use
    double *d_coef[NOFF] = {nullptr, nullptr, nullptr};   // per-pair records of gpw_eval_rho: header (static) + polynomial (written per call)
    double *d_mom[NOFF] = {nullptr, nullptr, nullptr};    // moment workspaces of gpw_eval_mat / gpw_eval_grad
    double *d_vg = nullptr;     // Gaussian values of every (pair, block) visit (geometry only; written at build time)
    double *d_eg = nullptr;     // 1-D Gaussian factor tables of every brick entry (orthogonal cells; geometry only)
    // optional kernel timing (gpw_plan_set_timing): events around each kernel of the last eval calls
    bool timing = false;
    cudaEvent_t ev[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
    bool ev_valid[2] = {false, false};
    InterpState *interp = nullptr;   // cuFFT plans and scratch of gpw_interp_up / gpw_restrict_down (first use)
    // The eval / interp calls write plan-owned workspaces (d_coef, d_mom, the interp scratch): calls on one plan are
    // serialised on the device -- every call first makes its stream wait for `busy`, recorded at the end of the
    // previous call on this plan, whatever stream that one ran on.
    cudaEvent_t busy = nullptr;
    HostIO *hio = nullptr;      // staging buffers, streams and events of the host-buffer variants (first use)
    int part_rank = 0, part_n = 1;   // gpw_plan_set_partition: this process evaluates the n1 slab `part_rank` of `part_n`
};

namespace {

bool cuda_ok(cudaError_t e, const char *what) {
    if (e == cudaSuccess) return true;
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return false;
}

template <class T>
bool upload(T **dst, const T *src, size_t n, long &bytes, const char *what) {
    *dst = nullptr;
    const size_t nb = sizeof(T) * (n ? n : 1);
    if (!cuda_ok(cudaMalloc((void **)dst, nb), what)) return false;
    bytes += (long)nb;
    if (n && !cuda_ok(cudaMemcpy(*dst, src, sizeof(T) * n, cudaMemcpyHostToDevice), what)) return false;
    return true;
}

void free_hostio(HostIO *h) {
    if (!h) return;
    for (cudaStream_t s : {h->s_in, h->s_out, h->s_cmp}) if (s) { cudaStreamSynchronize(s); cudaStreamDestroy(s); }
    for (cudaEvent_t e : {h->call, h->D_in, h->rho_done, h->rho_out, h->v_in, h->mat_done, h->F_out}) if (e) cudaEventDestroy(e);
    cudaFree(h->D); cudaFree(h->F);
    for (int a = 0; a < GPW_MAX_LEVEL; a++) { cudaFree(h->rho[a]); cudaFree(h->v[a]); }
    delete h;
}

void free_device(gpw_plan *p) {
    free_hostio(p->hio);
    p->hio = nullptr;
    if (p->busy) cudaEventDestroy(p->busy);
    p->busy = nullptr;
    interp_free(p->interp);
    p->interp = nullptr;
    for (int w = 0; w < 2; w++)
        for (int k = 0; k < 3; k++)
            if (p->ev[w][k]) cudaEventDestroy(p->ev[w][k]);
    cudaFree(p->d_taskK); cudaFree(p->d_taskP); cudaFree(p->d_export); cudaFree(p->d_S);
    for (int off = 0; off < NOFF; off++) { cudaFree(p->d_coef[off]); cudaFree(p->d_mom[off]); }
    cudaFree(p->d_vg); cudaFree(p->d_eg);
    free_device_lists(&p->lists);
}

// block rows [lo, hi) along n1 of slab `rank` of `n`: equal shares of the T1 rows, the remainder spread from the front
void partition_rows(int T1, int rank, int n, int *lo, int *hi) {
    *lo = (int)((long long)T1 * rank / n);
    *hi = (int)((long long)T1 * (rank + 1) / n);
}

void fill_params(const gpw_plan *p, GridParams &P, double *const *grids, int off = 0, size_t comp = 0) {
    std::memset(&P, 0, sizeof(P));
    const HostPlan *hp = p->hp;
    long long tile0 = 0, brick0 = 0;
    for (int a = 0; a < hp->nlevel; a++) {
        P.lev[a] = hp->lev[a];
        // one array over all levels: the entry after a level's last block is the next level's first
        P.tile_base[a] = p->lists.tile_base + tile0;
        P.seg[a] = p->lists.seg + tile0 * 8;
        P.brick_base[a] = p->lists.brick_base + brick0;
        tile0 += hp->lev[a].ntile; brick0 += hp->lev[a].nbrick;
        // comp: the launch works on component `comp` of every level's array (the fifth component of deriv = 2)
        P.grid[a] = grids[a] ? grids[a] + comp * (size_t)hp->lev[a].N[0] * hp->lev[a].N[1] * hp->lev[a].N[2] : nullptr;
        for (int L = 0; L < 8; L++) P.coef_base[a][L] = hp->coef_base[off][a][L];
        partition_rows(hp->lev[a].T[0], p->part_rank, p->part_n, &P.part_lo[a], &P.part_hi[a]);
    }
}

// Start of a call that uses the plan's device state: the current device must be the plan's, and the call's stream
// waits for the previous call on this plan (see gpw_plan::busy).
int begin_call(const gpw_plan *p, cudaStream_t st, const char *who) {
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), who)) return GPW_ECUDA;
    if (dev != p->device) {
        set_error(std::string(who) + ": the current CUDA device (" + std::to_string(dev) + ") is not the device the plan was built on (" +
                  std::to_string(p->device) + ")");
        return GPW_EINVAL;
    }
    if (!cuda_ok(cudaStreamWaitEvent(st, p->busy, 0), who)) return GPW_ECUDA;
    return GPW_OK;
}
int end_call(const gpw_plan *p, cudaStream_t st, const char *who) {
    return cuda_ok(cudaEventRecord(p->busy, st), who) ? GPW_OK : GPW_ECUDA;
}
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

void fill_pass(const gpw_plan *p, pp::PassArgs &A, int mode) {
    std::memset(&A, 0, sizeof(A));
    const HostPlan *hp = p->hp;
    A.tp = p->d_taskP; A.ntask = (int)hp->ntask; A.nao = hp->nao; A.hdiag = hp->hdiag ? 1 : 0; A.mode = mode;
    A.S_all = p->d_S;
    for (int off = 0; off < NOFF; off++) {
        for (int a = 0; a < GPW_MAX_LEVEL; a++)
            for (int L = 0; L < 8; L++) A.base[off][a][L] = hp->coef_base[off][a][L];
        A.rec[off] = p->d_coef[off]; A.mom[off] = p->d_mom[off];
    }
    for (int a = 0; a < GPW_MAX_LEVEL; a++) A.dV[a] = a < hp->nlevel ? hp->lev[a].dV : 0.0;
    for (int a = 0; a < GPW_MAX_LEVEL; a++) {
        A.big_lo[a] = a < hp->nlevel ? (int)hp->big_lo[a] : 0;
        A.big_n[a] = a < hp->nlevel ? (int)(hp->big_hi[a] - hp->big_lo[a]) : 0;
    }
}

// Workspaces of the derivative variants (degree offsets 1, 2), allocated when first needed: collocation records
// (with their static headers) and / or the moment vector.
int need_workspace(gpw_plan *p, int off, bool coef, bool mom, cudaStream_t st, const char *who) {
    const HostPlan *hp = p->hp;
    const size_t nt = (size_t)hp->ntask;
    const size_t nw = (size_t)(hp->ncoef_total[off] ? hp->ncoef_total[off] : 1);
    if (coef && !p->d_coef[off]) {
        const size_t nrec = nw + 8 * nt;
        if (!cuda_ok(cudaMalloc((void **)&p->d_coef[off], sizeof(double) * nrec), who)) return GPW_ENOMEM;
        p->device_bytes += (long)(sizeof(double) * nrec);
        if (!cuda_ok(cudaMemsetAsync(p->d_coef[off], 0, sizeof(double) * nrec, st), who)) return GPW_ECUDA;
        if (nt) {
            pp::PassArgs A;
            fill_pass(p, A, 0);
            k_rec_headers<<<((int)nt + 127) / 128, 128, 0, st>>>(p->d_taskK, p->d_taskP, (int)nt, A, off, p->d_coef[off]);
            if (!cuda_ok(cudaGetLastError(), who)) return GPW_ECUDA;
        }
    }
    if (mom && !p->d_mom[off]) {
        if (!cuda_ok(cudaMalloc((void **)&p->d_mom[off], sizeof(double) * nw), who)) return GPW_ENOMEM;
        p->device_bytes += (long)(sizeof(double) * nw);
    }
    return GPW_OK;
}

}  // namespace

extern "C" {

const char *gpw_last_error(void) { return gpw::last_error_cstr(); }

int gpw_build_pairs(const double *cell, int natm, const double *xyz, int nshl, const int *shl_atom,
                    const int *shl_l, const int *shl_nprim, const int *shl_prim_off,
                    const double *prim_exp, const double *prim_coef, int nlevel, const int *mesh,
                    double tau, double rel_cutoff, int hermi, gpw_plan **plan_out) {
    if (!plan_out) { set_error("gpw_build_pairs: plan_out is null"); return GPW_EINVAL; }
    *plan_out = nullptr;
    HostPlan *hp = nullptr;
    int ndev = 0;
    const bool have_dev = cudaGetDeviceCount(&ndev) == cudaSuccess && ndev >= 1;
    if (!have_dev) cudaGetLastError();
    // with a device the host only checks the arguments and computes the level geometry and the primitive radii; pairs
    // and lists are built on the device.  Without one the host builds everything (introspection only: eval calls fail
    // with GPW_ECUDA)
    const int rc = build_host_plan(cell, natm, xyz, nshl, shl_atom, shl_l, shl_nprim, shl_prim_off, prim_exp,
                                   prim_coef, nlevel, mesh, tau, rel_cutoff, hermi, !have_dev, &hp);
    if (rc != GPW_OK) return rc;
    gpw_plan *p = new (std::nothrow) gpw_plan();
    if (!p) { delete hp; set_error("out of host memory"); return GPW_ENOMEM; }
    p->hp = hp;
    if (!have_dev) {   // host-only plan
        *plan_out = p;
        return GPW_OK;
    }
    cudaGetDevice(&p->device);
    bool ok = true;
    long &nb = p->device_bytes;
    {
        DevicePairs dp;
        const int prc = build_device_pairs(hp, &dp);
        if (prc != GPW_OK) { delete hp; delete p; return prc; }
        p->d_taskK = dp.taskK; p->d_taskP = dp.taskP; p->d_export = dp.exported;
        nb += dp.bytes - (long)(sizeof(DevTask) * (size_t)dp.ntask);
        const int lrc = build_device_lists(hp, dp.devtask, (int)dp.ntask, &p->lists);
        cudaFree(dp.devtask);
        if (lrc != GPW_OK) {
            free_device(p);
            delete hp;
            delete p;
            return lrc;
        }
        nb += p->lists.bytes;
        hp->nitem = p->lists.nitem; hp->nbitem = p->lists.nbitem; hp->nvisit_total = p->lists.nvisit;
        hp->build_seconds += p->lists.seconds;
        for (int a = 0; a < GPW_MAX_LEVEL; a++) {
            hp->nvisit_level[a] = 0;
            for (int i = 0; i <= MAXL; i++)
                for (int j = 0; j <= MAXL; j++) {
                    hp->nvisit_class[a][i][j] = (long)p->lists.cls[a][i][j];
                    hp->nvisit_level[a] += (long)p->lists.cls[a][i][j];
                }
        }
    }
    if (ok) {
        std::vector<double> S_all((size_t)hp->nlevel * S_TOTAL);
        for (int a = 0; a < hp->nlevel; a++) std::memcpy(S_all.data() + (size_t)a * S_TOTAL, hp->S[a].data(), sizeof(double) * S_TOTAL);
        ok = upload(&p->d_S, S_all.data(), S_all.size(), nb, "upload monomial maps");
    }
    ok = ok && cuda_ok(cudaEventCreateWithFlags(&p->busy, cudaEventDisableTiming), "create event");
    // collocation records [nP0 nP1 nP2 a_p c22 c23 c33 0 | polynomial] per pair (headers written once) and the
    // moment workspace, for the degree offset 0; the derivative variants allocate theirs on first use
    if (ok) {
        const int wrc = need_workspace(p, 0, true, true, 0, "allocate pair workspaces");
        if (wrc != GPW_OK) { free_device(p); delete hp; delete p; return wrc; }
    }
    if (ok) {
        const size_t nvg = (size_t)hp->nvisit_total * visit_gauss_doubles(hp->ortho);
        ok = cuda_ok(cudaMalloc((void **)&p->d_vg, sizeof(double) * (nvg ? nvg : 1)), "allocate visit Gaussians");
        if (ok) {
            nb += (long)(sizeof(double) * nvg);
            GridParams P;
            double *none[GPW_MAX_LEVEL] = {nullptr};
            fill_params(p, P, none);
            int ntile_all = 0;
            for (int a = 0; a < hp->nlevel; a++) ntile_all += hp->lev[a].ntile;
            ok = hp->nvisit_total == 0 ||
                 (cuda_ok(launch_visit_gauss(P, ntile_all, p->d_taskK, p->lists.visit, p->d_vg, hp->ortho, 0), "visit Gaussians") &&
                  cuda_ok(cudaDeviceSynchronize(), "visit Gaussians"));
        }
    }
    if (ok && hp->ortho && p->lists.nentry > 0) {
        const size_t neg = (size_t)p->lists.nentry * entry_gauss_doubles(true);
        ok = cuda_ok(cudaMalloc((void **)&p->d_eg, sizeof(double) * neg), "allocate entry Gaussians");
        if (ok) {
            nb += (long)(sizeof(double) * neg);
            GridParams P;
            double *none[GPW_MAX_LEVEL] = {nullptr};
            fill_params(p, P, none);
            int nbrick_all = 0;
            for (int a = 0; a < hp->nlevel; a++) nbrick_all += hp->lev[a].nbrick;
            ok = cuda_ok(launch_entry_gauss(P, nbrick_all, p->d_taskK, p->lists.bentry, p->d_eg, 0), "entry Gaussians") &&
                 cuda_ok(cudaDeviceSynchronize(), "entry Gaussians");
        }
    }
    if (!ok) {
        free_device(p);
        delete hp;
        delete p;
        return GPW_ECUDA;
    }
    p->on_device = true;
    *plan_out = p;
    return GPW_OK;
}

void gpw_free_plan(gpw_plan *p) {
    if (!p) return;
    if (p->on_device) free_device(p);
    delete p->hp;
    delete p;
}

int gpw_plan_info(const gpw_plan *p, gpw_info *out) {
    if (!p || !out) { set_error("gpw_plan_info: null argument"); return GPW_EINVAL; }
    const HostPlan *hp = p->hp;
    std::memset(out, 0, sizeof(*out));
    out->nao = hp->nao; out->nshl = hp->nshl; out->nlevel = hp->nlevel; out->hermi = hp->hermi;
    out->on_device = p->on_device ? 1 : 0;
    out->ntask = hp->ntask;
    for (int a = 0; a < GPW_MAX_LEVEL; a++) {
        out->ntask_level[a] = hp->ntask_level[a];
        out->nvisit_level[a] = hp->nvisit_level[a];
        for (int i = 0; i <= MAXL; i++)
            for (int j = 0; j <= MAXL; j++) out->nvisit_class[a][i][j] = hp->nvisit_class[a][i][j];
    }
    out->nitem = hp->nitem;
    out->ncoef_total = (long)hp->ncoef_total[0];
    out->build_seconds = hp->build_seconds;
    out->device_bytes = p->device_bytes + interp_bytes(p->interp) + (p->hio ? p->hio->bytes : 0);
    return GPW_OK;
}

int gpw_plan_export_tasks(const gpw_plan *p, gpw_task *buf, long cap, long *ntask) {
    if (!p || !ntask) { set_error("gpw_plan_export_tasks: null argument"); return GPW_EINVAL; }
    const HostPlan *hp = p->hp;
    *ntask = hp->ntask;
    if (!buf) return GPW_OK;
    const long n = std::min(cap, *ntask);
    if (p->on_device) {   // screened on the device: copy the records back
        if (n > 0 && !cuda_ok(cudaMemcpy(buf, p->d_export, sizeof(gpw_task) * (size_t)n, cudaMemcpyDeviceToHost), "gpw_plan_export_tasks")) return GPW_ECUDA;
        return GPW_OK;
    }
    for (long i = 0; i < n; i++) {
        const HostTask &t = hp->task[i];
        gpw_task &o = buf[i];
        o.shl_a = t.shl_a; o.prim_a = t.prim_a; o.shl_b = t.shl_b; o.prim_b = t.prim_b;
        o.T[0] = t.T[0]; o.T[1] = t.T[1]; o.T[2] = t.T[2];
        o.level = t.level; o.R = t.R;
    }
    return GPW_OK;
}

int gpw_plan_export_visits(const gpw_plan *p, gpw_visit *buf, long cap, long *nvisit) {
    if (!p || !nvisit) { set_error("gpw_plan_export_visits: null argument"); return GPW_EINVAL; }
    const HostPlan *hp = p->hp;
    *nvisit = (long)hp->nvisit_total;
    if (!buf || cap <= 0) return GPW_OK;
    long long ntile_all = 0;
    for (int a = 0; a < hp->nlevel; a++) ntile_all += hp->lev[a].ntile;
    std::vector<Visit> vis;
    std::vector<long long> base;
    const Visit *V = nullptr;
    if (p->on_device) {   // the lists live on the device only
        try { vis.resize((size_t)hp->nvisit_total); base.resize((size_t)ntile_all + 1); }
        catch (const std::bad_alloc &) { set_error("gpw_plan_export_visits: out of host memory"); return GPW_ENOMEM; }
        if (!cuda_ok(cudaMemcpy(vis.data(), p->lists.visit, sizeof(Visit) * vis.size(), cudaMemcpyDeviceToHost), "gpw_plan_export_visits") ||
            !cuda_ok(cudaMemcpy(base.data(), p->lists.tile_base, sizeof(long long) * base.size(), cudaMemcpyDeviceToHost), "gpw_plan_export_visits"))
            return GPW_ECUDA;
        V = vis.data();
    } else {
        for (int a = 0; a < hp->nlevel; a++) base.insert(base.end(), hp->tile_base[a].begin(), hp->tile_base[a].begin() + hp->lev[a].ntile);
        base.push_back(hp->nvisit_total);
        V = hp->visit.data();
    }
    long long tile0 = 0;
    long n = 0;
    for (int a = 0; a < hp->nlevel && n < cap; a++) {
        const LevelGeom &g = hp->lev[a];
        for (int tl = 0; tl < g.ntile && n < cap; tl++) {
            const int w3 = tl % g.T[2], w2 = (tl / g.T[2]) % g.T[1], w1 = tl / (g.T[2] * g.T[1]);
            for (long long i = base[tile0 + tl]; i < base[tile0 + tl + 1] && n < cap; i++, n++) {
                buf[n].task = V[i].task;
                buf[n].block[0] = w1 + V[i].s[0] * g.T[0];
                buf[n].block[1] = w2 + V[i].s[1] * g.T[1];
                buf[n].block[2] = w3 + V[i].s[2] * g.T[2];
            }
        }
        tile0 += g.ntile;
    }
    return GPW_OK;
}

int gpw_eval_rho(const gpw_plan *p, const double *D_dev, int deriv, double *const *rho_dev, void *cuda_stream) {
    if (!p || !D_dev || !rho_dev) { set_error("gpw_eval_rho: null argument"); return GPW_EINVAL; }
    if (deriv < 0 || deriv > 2) { set_error("gpw_eval_rho: deriv must be 0, 1 or 2"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_rho: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++) {
        if (!rho_dev[a]) { set_error("gpw_eval_rho: null level pointer"); return GPW_EINVAL; }
        if (!aligned16(rho_dev[a])) { set_error("gpw_eval_rho: level pointers must be 16-byte aligned"); return GPW_EINVAL; }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, "gpw_eval_rho")) return rc;
    gpw_plan *pm = const_cast<gpw_plan *>(p);
    const int ncomp = deriv == 0 ? 1 : (deriv == 1 ? 4 : 5);
    for (int a = 0; a < hp->nlevel; a++) {
        const LevelGeom &g = hp->lev[a];
        const size_t nb = sizeof(double) * (size_t)g.N[0] * g.N[1] * g.N[2] * ncomp;
        if (!cuda_ok(cudaMemsetAsync(rho_dev[a], 0, nb, st), "gpw_eval_rho: memset")) return GPW_ECUDA;
    }
    const int ntask = (int)hp->ntask, nitem = (int)hp->nitem;
    if (ntask == 0 || nitem == 0) return end_call(p, st, "gpw_eval_rho");
    if (deriv == 2)
        if (const int rc = need_workspace(pm, 2, true, false, st, "gpw_eval_rho: kinetic-energy workspace")) return rc;
    if (p->timing) { cudaEventRecord(p->ev[0][0], st); pm->ev_valid[0] = true; }
    pp::PassArgs A;
    fill_pass(p, A, pp::PRE_DENS | (deriv == 2 ? pp::PRE_TAU : 0));
    A.D = D_dev;
    if (!cuda_ok(launch_pair_pass(A, hp->max_l, hp->max_L, st), "gpw_eval_rho: pre-pass launch")) return GPW_ECUDA;
    if (p->timing) cudaEventRecord(p->ev[0][1], st);
    GridParams P;
    fill_params(p, P, rho_dev);
    if (!cuda_ok(launch_collocate(P, p->lists.visit, p->lists.item, nitem, p->lists.item_hi, (int)p->lists.nitem_hi, p->d_coef[0], p->d_vg,
                                  deriv ? 1 : 0, 0, hp->max_L, hp->ortho, st),
                 "gpw_eval_rho: collocation launch")) return GPW_ECUDA;
    if (deriv == 2) {   // fifth component: tau, polynomials of degree L + 2, value only (Eq. 15)
        fill_params(p, P, rho_dev, 2, 4);
        if (!cuda_ok(launch_collocate(P, p->lists.visit, p->lists.item, nitem, nullptr, 0, p->d_coef[2], p->d_vg, 0, 2, hp->max_L, hp->ortho, st),
                     "gpw_eval_rho: kinetic-energy collocation launch")) return GPW_ECUDA;
    }
    if (p->timing) cudaEventRecord(p->ev[0][2], st);
    if (!cuda_ok(cudaGetLastError(), "gpw_eval_rho: kernel launch")) return GPW_ECUDA;
    return end_call(p, st, "gpw_eval_rho");
}

int gpw_eval_mat(const gpw_plan *p, const double *const *v_dev, int deriv, double *F_dev, void *cuda_stream) {
    if (!p || !v_dev || !F_dev) { set_error("gpw_eval_mat: null argument"); return GPW_EINVAL; }
    if (deriv < 0 || deriv > 2) { set_error("gpw_eval_mat: deriv must be 0, 1 or 2"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_mat: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++) {
        if (!v_dev[a]) { set_error("gpw_eval_mat: null level pointer"); return GPW_EINVAL; }
        if (!aligned16(v_dev[a])) { set_error("gpw_eval_mat: level pointers must be 16-byte aligned"); return GPW_EINVAL; }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, "gpw_eval_mat")) return rc;
    gpw_plan *pm = const_cast<gpw_plan *>(p);
    if (!cuda_ok(cudaMemsetAsync(F_dev, 0, sizeof(double) * (size_t)hp->nao * hp->nao, st), "gpw_eval_mat: memset")) return GPW_ECUDA;
    const int ntask = (int)hp->ntask, nitem = (int)hp->nitem;
    if (ntask == 0 || nitem == 0) return end_call(p, st, "gpw_eval_mat");
    if (deriv == 2)
        if (const int rc = need_workspace(pm, 2, false, true, st, "gpw_eval_mat: kinetic-energy workspace")) return rc;
    if (!cuda_ok(cudaMemsetAsync(p->d_mom[0], 0, sizeof(double) * (size_t)hp->ncoef_total[0], st), "gpw_eval_mat: memset")) return GPW_ECUDA;
    if (deriv == 2 && !cuda_ok(cudaMemsetAsync(p->d_mom[2], 0, sizeof(double) * (size_t)hp->ncoef_total[2], st), "gpw_eval_mat: memset")) return GPW_ECUDA;
    GridParams P;
    fill_params(p, P, const_cast<double *const *>(v_dev));
    if (p->timing) { cudaEventRecord(p->ev[1][0], st); pm->ev_valid[1] = true; }
    if (!cuda_ok(launch_integrate(P, p->d_taskK, p->lists.bentry, p->lists.bitem, (int)hp->nbitem, p->d_eg, p->d_mom[0], deriv ? 1 : 0, 0,
                                  hp->max_L, hp->ortho, st), "gpw_eval_mat: integration launch")) return GPW_ECUDA;
    if (deriv == 2) {   // fifth component: the kinetic-energy potential against 1/2 grad phi . grad phi (Eq. 16): moments to degree L + 2
        fill_params(p, P, const_cast<double *const *>(v_dev), 2, 4);
        if (!cuda_ok(launch_integrate(P, p->d_taskK, p->lists.bentry, p->lists.bitem, (int)hp->nbitem, p->d_eg, p->d_mom[2], 0, 2,
                                      hp->max_L, hp->ortho, st), "gpw_eval_mat: kinetic-energy integration launch")) return GPW_ECUDA;
    }
    if (p->timing) cudaEventRecord(p->ev[1][1], st);
    pp::PassArgs A;
    fill_pass(p, A, pp::POST_MAT | (deriv == 2 ? pp::POST_TAU : 0));
    A.F = F_dev;
    if (!cuda_ok(launch_pair_pass(A, hp->max_l, hp->max_L, st), "gpw_eval_mat: post-pass launch")) return GPW_ECUDA;
    if (p->timing) cudaEventRecord(p->ev[1][2], st);
    if (!cuda_ok(cudaGetLastError(), "gpw_eval_mat: kernel launch")) return GPW_ECUDA;
    return end_call(p, st, "gpw_eval_mat");
}

int gpw_eval_grad(gpw_plan *p, const double *const *v_dev, int deriv, const double *D_dev, double *grad_dev, void *cuda_stream) {
    if (!p || !v_dev || !D_dev || !grad_dev) { set_error("gpw_eval_grad: null argument"); return GPW_EINVAL; }
    if (deriv != 0 && deriv != 1) { set_error("gpw_eval_grad: deriv must be 0 or 1"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_grad: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++) {
        if (!v_dev[a]) { set_error("gpw_eval_grad: null level pointer"); return GPW_EINVAL; }
        if (!aligned16(v_dev[a])) { set_error("gpw_eval_grad: level pointers must be 16-byte aligned"); return GPW_EINVAL; }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, "gpw_eval_grad")) return rc;
    if (!cuda_ok(cudaMemsetAsync(grad_dev, 0, sizeof(double) * 3 * (size_t)hp->natm, st), "gpw_eval_grad: memset")) return GPW_ECUDA;
    const int ntask = (int)hp->ntask, nitem = (int)hp->nitem;
    if (ntask == 0 || nitem == 0) return end_call(p, st, "gpw_eval_grad");
    if (const int rc = need_workspace(p, 1, false, true, st, "gpw_eval_grad: workspace")) return rc;
    if (!cuda_ok(cudaMemsetAsync(p->d_mom[1], 0, sizeof(double) * (size_t)hp->ncoef_total[1], st), "gpw_eval_grad: memset")) return GPW_ECUDA;
    GridParams P;
    fill_params(p, P, const_cast<double *const *>(v_dev), 1);
    if (!cuda_ok(launch_integrate(P, p->d_taskK, p->lists.bentry, p->lists.bitem, (int)hp->nbitem, p->d_eg, p->d_mom[1], deriv, 1,
                                  hp->max_L, hp->ortho, st), "gpw_eval_grad: integration launch")) return GPW_ECUDA;
    pp::PassArgs A;
    fill_pass(p, A, pp::POST_GRAD);
    A.D = D_dev; A.grad = grad_dev;
    if (!cuda_ok(launch_pair_pass(A, hp->max_l, hp->max_L, st), "gpw_eval_grad: post-pass launch")) return GPW_ECUDA;
    return end_call(p, st, "gpw_eval_grad");
}

// ---- integration without any allocation: the moment workspace in a static device array ----
// gpw_eval_mat's scratch is the moment vector (one block of ncoef(L + off) doubles per pair, added to atomically by
// k_integrate, read by the post-pass).  Here it lives in the library's image: every GPU that loads the library holds
// GPW_STATIC_MOM_DOUBLES * 8 bytes until exit.  The name below is a device symbol; host code may only use the
// address cudaGetSymbolAddress returns for the current device.
static __device__ __align__(256) double g_static_mom[GPW_STATIC_MOM_DOUBLES];

// device address of g_static_mom on the current device, looked up once per device (with that device current)
static int static_mom_address(double **out, const char *who) {
    constexpr int MAXDEV = 64;
    static double *addr[MAXDEV] = {nullptr};
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), who)) return GPW_ECUDA;
    if (dev < 0 || dev >= MAXDEV) { set_error(std::string(who) + ": device ordinal out of range"); return GPW_EUNSUPPORTED; }
    if (!addr[dev]) {
        double *ptr = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress((void **)&ptr, g_static_mom), who)) return GPW_ECUDA;
        if (!ptr) { set_error(std::string(who) + ": cudaGetSymbolAddress returned a null address"); return GPW_ECUDA; }
        addr[dev] = ptr;
    }
    *out = addr[dev];
    return GPW_OK;
}

int gpw_eval_mat_static(const gpw_plan *p, const double *const *v_dev, int deriv, double *F_dev, void *cuda_stream) {
    const char *who = "gpw_eval_mat_static";
    if (!p || !v_dev || !F_dev) { set_error("gpw_eval_mat_static: null argument"); return GPW_EINVAL; }
    if (deriv < 0 || deriv > 2) { set_error("gpw_eval_mat_static: deriv must be 0, 1 or 2"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_mat_static: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++) {
        if (!v_dev[a]) { set_error("gpw_eval_mat_static: null level pointer"); return GPW_EINVAL; }
        if (!aligned16(v_dev[a])) { set_error("gpw_eval_mat_static: level pointers must be 16-byte aligned"); return GPW_EINVAL; }
    }
    // the moments of degree offset 0, then (deriv = 2) those of offset 2 from the next 256-byte boundary
    const size_t n0 = (size_t)hp->ncoef_total[0];
    const size_t off2 = (n0 + 31) / 32 * 32;
    const size_t need = deriv == 2 ? off2 + (size_t)hp->ncoef_total[2] : n0;
    if (need > (size_t)GPW_STATIC_MOM_DOUBLES) {
        set_error("gpw_eval_mat_static: the plan's moment workspace (" + std::to_string(need) + " doubles) exceeds GPW_STATIC_MOM_DOUBLES (" +
                  std::to_string((long long)GPW_STATIC_MOM_DOUBLES) + "); use gpw_eval_mat");
        return GPW_EUNSUPPORTED;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, who)) return rc;
    double *mom = nullptr;
    if (const int rc = static_mom_address(&mom, who)) return rc;
    if (!cuda_ok(cudaMemsetAsync(F_dev, 0, sizeof(double) * (size_t)hp->nao * hp->nao, st), "gpw_eval_mat_static: memset")) return GPW_ECUDA;
    const int ntask = (int)hp->ntask, nitem = (int)hp->nitem;
    if (ntask == 0 || nitem == 0) return end_call(p, st, who);
    // the array keeps the previous call's moments: clear the part this call accumulates into
    if (!cuda_ok(cudaMemsetAsync(mom, 0, sizeof(double) * need, st), "gpw_eval_mat_static: memset")) return GPW_ECUDA;
    GridParams P;
    fill_params(p, P, const_cast<double *const *>(v_dev));
    if (!cuda_ok(launch_integrate(P, p->d_taskK, p->lists.bentry, p->lists.bitem, (int)hp->nbitem, p->d_eg, mom, deriv ? 1 : 0, 0,
                                  hp->max_L, hp->ortho, st), "gpw_eval_mat_static: integration launch")) return GPW_ECUDA;
    if (deriv == 2) {
        fill_params(p, P, const_cast<double *const *>(v_dev), 2, 4);
        if (!cuda_ok(launch_integrate(P, p->d_taskK, p->lists.bentry, p->lists.bitem, (int)hp->nbitem, p->d_eg, mom + off2, 0, 2,
                                      hp->max_L, hp->ortho, st), "gpw_eval_mat_static: kinetic-energy integration launch")) return GPW_ECUDA;
    }
    pp::PassArgs A;
    fill_pass(p, A, pp::POST_MAT | (deriv == 2 ? pp::POST_TAU : 0));
    A.mom[0] = mom;
    A.mom[2] = deriv == 2 ? mom + off2 : nullptr;
    A.F = F_dev;
    if (!cuda_ok(launch_pair_pass(A, hp->max_l, hp->max_L, st), "gpw_eval_mat_static: post-pass launch")) return GPW_ECUDA;
    if (!cuda_ok(cudaGetLastError(), "gpw_eval_mat_static: kernel launch")) return GPW_ECUDA;
    return end_call(p, st, who);
}

// ---- host-buffer variants ----
static int ensure_hostio(gpw_plan *p, int ncomp, const char *who) {
    const HostPlan *hp = p->hp;
    if (!p->hio) {
        HostIO *h = new (std::nothrow) HostIO();
        if (!h) { set_error("out of host memory"); return GPW_ENOMEM; }
        p->hio = h;
        bool ok = true;
        for (cudaStream_t *s : {&h->s_in, &h->s_out, &h->s_cmp}) ok = ok && cuda_ok(cudaStreamCreateWithFlags(s, cudaStreamNonBlocking), who);
        for (cudaEvent_t *e : {&h->call, &h->D_in, &h->rho_done, &h->rho_out, &h->v_in, &h->mat_done, &h->F_out})
            ok = ok && cuda_ok(cudaEventCreateWithFlags(e, cudaEventDisableTiming), who);
        const size_t nb = sizeof(double) * (size_t)hp->nao * hp->nao;
        ok = ok && cuda_ok(cudaMalloc((void **)&h->D, nb ? nb : 8), who) && cuda_ok(cudaMalloc((void **)&h->F, nb ? nb : 8), who);
        if (!ok) return GPW_ECUDA;
        h->bytes += (long)(2 * nb);
    }
    HostIO *h = p->hio;
    if (ncomp > h->ncomp) {   // (re)allocate the level buffers; earlier calls may still use the old ones
        if (!cuda_ok(cudaDeviceSynchronize(), who)) return GPW_ECUDA;
        for (int a = 0; a < hp->nlevel; a++) {
            const size_t nb = sizeof(double) * (size_t)hp->lev[a].N[0] * hp->lev[a].N[1] * hp->lev[a].N[2];
            cudaFree(h->rho[a]); cudaFree(h->v[a]);
            h->rho[a] = h->v[a] = nullptr;
            h->bytes -= (long)(2 * nb * h->ncomp);
            if (!cuda_ok(cudaMalloc((void **)&h->rho[a], nb * ncomp), who) || !cuda_ok(cudaMalloc((void **)&h->v[a], nb * ncomp), who)) {
                h->ncomp = 0;
                return GPW_ENOMEM;
            }
            h->bytes += (long)(2 * nb * ncomp);
        }
        h->ncomp = ncomp;
    }
    return GPW_OK;
}

int gpw_eval_rho_host(gpw_plan *p, const double *D_host, int deriv, double *const *rho_host, void *cuda_stream) {
    if (!p || !D_host || !rho_host) { set_error("gpw_eval_rho_host: null argument"); return GPW_EINVAL; }
    if (deriv < 0 || deriv > 2) { set_error("gpw_eval_rho_host: deriv must be 0, 1 or 2"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_rho_host: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++)
        if (!rho_host[a]) { set_error("gpw_eval_rho_host: null level pointer"); return GPW_EINVAL; }
    const int ncomp = deriv == 0 ? 1 : (deriv == 1 ? 4 : 5);
    if (const int rc = ensure_hostio(p, ncomp, "gpw_eval_rho_host")) return rc;
    HostIO *h = p->hio;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const char *who = "gpw_eval_rho_host";
    bool ok = cuda_ok(cudaEventRecord(h->call, st), who);
    // upload of D: after the caller's earlier work, and after the previous collocation has read the staging copy
    ok = ok && cuda_ok(cudaStreamWaitEvent(h->s_in, h->call, 0), who) && cuda_ok(cudaStreamWaitEvent(h->s_in, h->rho_done, 0), who) &&
         cuda_ok(cudaMemcpyAsync(h->D, D_host, sizeof(double) * (size_t)hp->nao * hp->nao, cudaMemcpyHostToDevice, h->s_in), who) &&
         cuda_ok(cudaEventRecord(h->D_in, h->s_in), who);
    // collocation: after the upload, and after the previous download has left the staging grids
    ok = ok && cuda_ok(cudaStreamWaitEvent(h->s_cmp, h->D_in, 0), who) && cuda_ok(cudaStreamWaitEvent(h->s_cmp, h->rho_out, 0), who);
    if (!ok) return GPW_ECUDA;
    if (const int rc = gpw_eval_rho(p, h->D, deriv, h->rho, h->s_cmp)) return rc;
    ok = cuda_ok(cudaEventRecord(h->rho_done, h->s_cmp), who) && cuda_ok(cudaStreamWaitEvent(h->s_out, h->rho_done, 0), who);
    for (int a = 0; ok && a < hp->nlevel; a++) {
        const size_t nb = sizeof(double) * (size_t)hp->lev[a].N[0] * hp->lev[a].N[1] * hp->lev[a].N[2] * ncomp;
        ok = cuda_ok(cudaMemcpyAsync(rho_host[a], h->rho[a], nb, cudaMemcpyDeviceToHost, h->s_out), who);
    }
    ok = ok && cuda_ok(cudaEventRecord(h->rho_out, h->s_out), who);
    return ok ? GPW_OK : GPW_ECUDA;
}

int gpw_eval_mat_host(gpw_plan *p, const double *const *v_host, int deriv, double *F_host, void *cuda_stream) {
    if (!p || !v_host || !F_host) { set_error("gpw_eval_mat_host: null argument"); return GPW_EINVAL; }
    if (deriv < 0 || deriv > 2) { set_error("gpw_eval_mat_host: deriv must be 0, 1 or 2"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_eval_mat_host: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    const HostPlan *hp = p->hp;
    for (int a = 0; a < hp->nlevel; a++)
        if (!v_host[a]) { set_error("gpw_eval_mat_host: null level pointer"); return GPW_EINVAL; }
    const int ncomp = deriv == 0 ? 1 : (deriv == 1 ? 4 : 5);
    if (const int rc = ensure_hostio(p, ncomp, "gpw_eval_mat_host")) return rc;
    HostIO *h = p->hio;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const char *who = "gpw_eval_mat_host";
    bool ok = cuda_ok(cudaEventRecord(h->call, st), who);
    ok = ok && cuda_ok(cudaStreamWaitEvent(h->s_in, h->call, 0), who) && cuda_ok(cudaStreamWaitEvent(h->s_in, h->mat_done, 0), who);
    for (int a = 0; ok && a < hp->nlevel; a++) {
        const size_t nb = sizeof(double) * (size_t)hp->lev[a].N[0] * hp->lev[a].N[1] * hp->lev[a].N[2] * ncomp;
        ok = cuda_ok(cudaMemcpyAsync(h->v[a], v_host[a], nb, cudaMemcpyHostToDevice, h->s_in), who);
    }
    ok = ok && cuda_ok(cudaEventRecord(h->v_in, h->s_in), who);
    ok = ok && cuda_ok(cudaStreamWaitEvent(h->s_cmp, h->v_in, 0), who) && cuda_ok(cudaStreamWaitEvent(h->s_cmp, h->F_out, 0), who);
    if (!ok) return GPW_ECUDA;
    if (const int rc = gpw_eval_mat(p, h->v, deriv, h->F, h->s_cmp)) return rc;
    ok = cuda_ok(cudaEventRecord(h->mat_done, h->s_cmp), who) && cuda_ok(cudaStreamWaitEvent(h->s_out, h->mat_done, 0), who) &&
         cuda_ok(cudaMemcpyAsync(F_host, h->F, sizeof(double) * (size_t)hp->nao * hp->nao, cudaMemcpyDeviceToHost, h->s_out), who) &&
         cuda_ok(cudaEventRecord(h->F_out, h->s_out), who);
    return ok ? GPW_OK : GPW_ECUDA;
}

int gpw_plan_wait(gpw_plan *p, void *cuda_stream) {
    if (!p) { set_error("gpw_plan_wait: null plan"); return GPW_EINVAL; }
    if (!p->hio) return GPW_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return cuda_ok(cudaStreamWaitEvent(st, p->hio->rho_out, 0), "gpw_plan_wait") && cuda_ok(cudaStreamWaitEvent(st, p->hio->F_out, 0), "gpw_plan_wait")
               ? GPW_OK : GPW_ECUDA;
}

int gpw_plan_set_partition(gpw_plan *p, int rank, int nranks) {
    if (!p) { set_error("gpw_plan_set_partition: null plan"); return GPW_EINVAL; }
    if (nranks < 1 || rank < 0 || rank >= nranks) { set_error("gpw_plan_set_partition: need 0 <= rank < nranks"); return GPW_EINVAL; }
    p->part_rank = rank; p->part_n = nranks;
    return GPW_OK;
}

int gpw_plan_partition_bounds(const gpw_plan *p, int level, int rank, int nranks, int *n1_lo, int *n1_hi) {
    if (!p || !n1_lo || !n1_hi) { set_error("gpw_plan_partition_bounds: null argument"); return GPW_EINVAL; }
    if (level < 0 || level >= p->hp->nlevel || nranks < 1 || rank < 0 || rank >= nranks) {
        set_error("gpw_plan_partition_bounds: level or rank out of range");
        return GPW_EINVAL;
    }
    int lo, hi;
    partition_rows(p->hp->lev[level].T[0], rank, nranks, &lo, &hi);
    *n1_lo = TILE * lo; *n1_hi = TILE * hi;
    return GPW_OK;
}

int gpw_plan_set_timing(gpw_plan *p, int enable) {
    if (!p) { set_error("gpw_plan_set_timing: null plan"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_plan_set_timing: the plan has no device copy"); return GPW_ECUDA; }
    if (enable && !p->ev[0][0])
        for (int w = 0; w < 2; w++)
            for (int k = 0; k < 3; k++)
                if (!cuda_ok(cudaEventCreate(&p->ev[w][k]), "gpw_plan_set_timing")) return GPW_ECUDA;
    p->timing = enable != 0;
    p->ev_valid[0] = p->ev_valid[1] = false;
    return GPW_OK;
}

int gpw_plan_get_timing(gpw_plan *p, int which, float *ms_out) {
    if (!p || !ms_out || which < 0 || which > 1) { set_error("gpw_plan_get_timing: bad argument"); return GPW_EINVAL; }
    if (!p->timing || !p->ev_valid[which]) { set_error("gpw_plan_get_timing: no timed call of that kind yet"); return GPW_EINVAL; }
    if (!cuda_ok(cudaEventSynchronize(p->ev[which][2]), "gpw_plan_get_timing")) return GPW_ECUDA;
    cudaEventElapsedTime(&ms_out[0], p->ev[which][0], p->ev[which][1]);
    cudaEventElapsedTime(&ms_out[1], p->ev[which][1], p->ev[which][2]);
    return GPW_OK;
}

int gpw_dfma_peak(double min_seconds, double *tflops_out, int *sm_count_out) {
    if (!tflops_out) { set_error("gpw_dfma_peak: null argument"); return GPW_EINVAL; }
    int dev = 0, nsm = 0;
    if (!cuda_ok(cudaGetDevice(&dev), "gpw_dfma_peak") ||
        !cuda_ok(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), "gpw_dfma_peak")) return GPW_ECUDA;
    if (sm_count_out) *sm_count_out = nsm;
    double *d = nullptr;
    if (!cuda_ok(cudaMalloc((void **)&d, 8), "gpw_dfma_peak")) return GPW_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = nsm * 8, threads = 256;
    int iters = 2048;
    double best = 0.0, spent = 0.0;
    k_dfma_peak<<<blocks, threads>>>(d, 64, 1.0);   // warm-up
    while (spent < min_seconds || best == 0.0) {
        cudaEventRecord(e0);
        k_dfma_peak<<<blocks, threads>>>(d, iters, 1.0);
        cudaEventRecord(e1);
        if (!cuda_ok(cudaEventSynchronize(e1), "gpw_dfma_peak")) { cudaFree(d); return GPW_ECUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 8 * 16 * (double)iters * blocks * threads;
        best = std::max(best, flops / (ms * 1e-3) / 1e12);
        spent += ms * 1e-3;
        if (ms < 20.0f) iters *= 2;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    *tflops_out = best;
    return GPW_OK;
}

int gpw_dmma_peak(double min_seconds, double *tflops_dmma_out, double *tflops_mixed_out) {
    if (!tflops_dmma_out || !tflops_mixed_out) { set_error("gpw_dmma_peak: null argument"); return GPW_EINVAL; }
    int dev = 0, nsm = 0;
    if (!cuda_ok(cudaGetDevice(&dev), "gpw_dmma_peak") ||
        !cuda_ok(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), "gpw_dmma_peak")) return GPW_ECUDA;
    double *d = nullptr;
    if (!cuda_ok(cudaMalloc((void **)&d, 8), "gpw_dmma_peak")) return GPW_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = nsm * 8, threads = 256;
    for (int mixed = 0; mixed < 2; mixed++) {
        int iters = 512;
        double best = 0.0, spent = 0.0;
        k_dmma_peak<<<blocks, threads>>>(d, 16, 1.0, mixed);   // warm-up
        while (spent < min_seconds || best == 0.0) {
            cudaEventRecord(e0);
            k_dmma_peak<<<blocks, threads>>>(d, iters, 1.0, mixed);
            cudaEventRecord(e1);
            if (!cuda_ok(cudaEventSynchronize(e1), "gpw_dmma_peak")) { cudaFree(d); return GPW_ECUDA; }
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            // per loop trip and warp: 64 DMMA of 512 flops; mixed: + 32 DFMA per thread = 32 * 2 * 32 flops per warp
            const double per_warp = 64.0 * 512.0 + (mixed ? 32.0 * 2.0 * 32.0 : 0.0);
            const double flops = per_warp * (double)iters * blocks * (threads / 32);
            best = std::max(best, flops / (ms * 1e-3) / 1e12);
            spent += ms * 1e-3;
            if (ms < 20.0f) iters *= 2;
        }
        *(mixed ? tflops_mixed_out : tflops_dmma_out) = best;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    return GPW_OK;
}

int gpw_interp_up(gpw_plan *p, const double *const *rho_dev, int ncomp, double *rho_fine_dev, void *cuda_stream) {
    if (!p || !rho_dev || !rho_fine_dev) { set_error("gpw_interp_up: null argument"); return GPW_EINVAL; }
    if (ncomp < 1) { set_error("gpw_interp_up: ncomp must be >= 1"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_interp_up: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    for (int a = 0; a < p->hp->nlevel; a++)
        if (!rho_dev[a]) { set_error("gpw_interp_up: null level pointer"); return GPW_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, "gpw_interp_up")) return rc;
    if (const int rc = interp_up(p->hp, &p->interp, rho_dev, ncomp, rho_fine_dev, st)) return rc;
    return end_call(p, st, "gpw_interp_up");
}

static int gspace_call(gpw_plan *p, int kind, const double *in, double *out, void *cuda_stream, const char *who) {
    if (!p || !in || !out) { set_error(std::string(who) + ": null argument"); return GPW_EINVAL; }
    if (!p->on_device) { set_error(std::string(who) + ": the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    if (!aligned16(in) || !aligned16(out)) { set_error(std::string(who) + ": pointers must be 16-byte aligned"); return GPW_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, who)) return rc;
    if (const int rc = gspace_apply(p->hp, &p->interp, kind, in, out, st)) return rc;
    return end_call(p, st, who);
}
int gpw_hartree(gpw_plan *p, const double *rho_fine_dev, double *vh_fine_dev, void *cuda_stream) {
    return gspace_call(p, 0, rho_fine_dev, vh_fine_dev, cuda_stream, "gpw_hartree");
}
int gpw_gspace_gradient(gpw_plan *p, const double *rho_fine_dev, double *grad_fine_dev, void *cuda_stream) {
    return gspace_call(p, 1, rho_fine_dev, grad_fine_dev, cuda_stream, "gpw_gspace_gradient");
}
int gpw_gspace_divergence(gpw_plan *p, const double *w_fine_dev, double *div_fine_dev, void *cuda_stream) {
    return gspace_call(p, 2, w_fine_dev, div_fine_dev, cuda_stream, "gpw_gspace_divergence");
}

int gpw_restrict_down(gpw_plan *p, const double *v_fine_dev, int ncomp, double *const *v_dev, void *cuda_stream) {
    if (!p || !v_fine_dev || !v_dev) { set_error("gpw_restrict_down: null argument"); return GPW_EINVAL; }
    if (ncomp < 1) { set_error("gpw_restrict_down: ncomp must be >= 1"); return GPW_EINVAL; }
    if (!p->on_device) { set_error("gpw_restrict_down: the plan has no device copy (no CUDA device at build time); there is no CPU path"); return GPW_ECUDA; }
    for (int a = 0; a < p->hp->nlevel; a++)
        if (!v_dev[a]) { set_error("gpw_restrict_down: null level pointer"); return GPW_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (const int rc = begin_call(p, st, "gpw_restrict_down")) return rc;
    if (const int rc = interp_down(p->hp, &p->interp, v_fine_dev, ncomp, v_dev, st)) return rc;
    return end_call(p, st, "gpw_restrict_down");
}

}  // extern "C"
