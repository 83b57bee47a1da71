// Device side of gpw_build_pairs, first half: pair screening (Alg. 4, re-decomposed: no atomics
// into pooled lists, a count / scan / fill pass instead, so that the pair order is deterministic).  Written from the
// readings T2-T5 of DESIGN.md:
//   T2  keep (a, b, T) iff |A - B - T| < r_a + r_b, over every lattice vector T that can satisfy it: in fractional
//       coordinates |f_i - t_i| <= (r_a + r_b) |b_i|, f = (A - B) . b;   hermi: prim a >= prim b, and for a == b only
//       T = 0 or T lexicographically positive
//   T3  a_p = a_a + a_b,  P = (a_a A + a_b (B + T)) / a_p,  kappa = |c_a c_b| exp(-(a_a a_b / a_p) |A - B - T|^2)
//   T4  R_t = largest root of r^2 kappa (r + dA)^la (r + dB)^lb exp(-a_p r^2) = tau, 40 fixed-point steps from
//       sqrt(max(C, 1) / a_p) + dA + dB + 5,  C = ln kappa - ln tau
//   T5  the coarsest level with E_alpha >= rel_cutoff a_p, else level 0
// The primitive radii r_a (T1) come from the host (one per primitive).  One thread per ordered primitive pair walks
// its few lattice vectors; the kept pairs are written in (prim a, prim b, T) order, then sorted (stable radix sort)
// by class (level, L, la), and the records the kernels read (TaskK, TaskP), the list builder's DevTask and the
// export record are written in that order.
//
// Compiled with -fmad=false like plan_device.cu, so that the expressions round as on the host.
#include <cub/cub.cuh>
#include <cuda_runtime.h>

#include <chrono>
#include <cstring>

#include "gpw_kernels.cuh"
#include "plan_device.h"

namespace gpw {
namespace {

struct PairGeom {
    double cell[9], binv[9], bnorm[3];
    double ecut[GPW_MAX_LEVEL], circ[GPW_MAX_LEVEL];
    double Nlev[GPW_MAX_LEVEL][3];
    double tau, rel_cutoff;
    int nlevel, hermi, nprim, pad;
};

struct Kept {          // what the screen knows about a kept pair
    double P[3], Bt[3];
    double ap, pref, R;
    int level;
};

// T3-T5 for one candidate (a, b, T); false if the pair is dropped.  sharp: set when the pair's Gaussian underflows
// inside its own blocks (the kernels anchor the recursion of Eq. 24-25 at a block corner).
__device__ bool screen_pair(const PairGeom &G, const DevPrim &a, const DevPrim &b, int t0, int t1, int t2, Kept &k, int *sharp) {
    const double rsum = a.rad + b.rad;
    double dd = 0.0;
    for (int x = 0; x < 3; x++) {
        const double Tv = t0 * G.cell[0 * 3 + x] + t1 * G.cell[1 * 3 + x] + t2 * G.cell[2 * 3 + x];
        k.Bt[x] = b.A[x] + Tv;
        dd += (a.A[x] - k.Bt[x]) * (a.A[x] - k.Bt[x]);
    }
    if (!(sqrt(dd) < rsum)) return false;
    k.ap = a.exp + b.exp;
    double dA = 0.0, dB = 0.0;
    for (int x = 0; x < 3; x++) {
        k.P[x] = (a.exp * a.A[x] + b.exp * k.Bt[x]) / k.ap;
        dA += (k.P[x] - a.A[x]) * (k.P[x] - a.A[x]);
        dB += (k.P[x] - k.Bt[x]) * (k.P[x] - k.Bt[x]);
    }
    dA = sqrt(dA); dB = sqrt(dB);
    const double ex = exp(-(a.exp * b.exp / k.ap) * dd);
    k.pref = a.coef * b.coef * ex;
    const double kappa = fabs(a.coef * b.coef) * ex;
    // T4
    const double C = log(kappa) - log(G.tau);
    double r = sqrt(fmax(C, 1.0) / k.ap) + dA + dB + 5.0;
    for (int it = 0; it < 40; it++) {
        const double arg = (C + 2.0 * log(r) + a.l * log(r + dA) + b.l * log(r + dB)) / k.ap;
        if (arg <= 0.0) return false;
        r = sqrt(arg);
    }
    k.R = r;
    // T5
    k.level = 0;
    for (int lev = G.nlevel - 1; lev >= 0; lev--)
        if (G.ecut[lev] >= G.rel_cutoff * k.ap) { k.level = lev; break; }
    const double reach = k.R + 2.0 * G.circ[k.level];
    if (k.ap * reach * reach > 600.0) { *sharp = 1; return false; }
    return true;
}

// One thread per ordered primitive pair (pa, pb): the lattice vectors of T2, in lexicographic order.
template <bool FILL>
__global__ void __launch_bounds__(128) k_pair_enum(const __grid_constant__ PairGeom G, const DevPrim *__restrict__ prims,
                                                   unsigned *__restrict__ cnt, const long long *__restrict__ off,
                                                   RawPair *__restrict__ raw, unsigned *__restrict__ key, int *__restrict__ sharp) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= (long long)G.nprim * G.nprim) return;
    const int pa = (int)(e / G.nprim), pb = (int)(e % G.nprim);
    unsigned n = 0;
    if (!(G.hermi && pa < pb)) {
        const DevPrim a = prims[pa], b = prims[pb];
        if (a.rad > 0.0 && b.rad > 0.0) {
            const double rsum = a.rad + b.rad;
            const double d[3] = {a.A[0] - b.A[0], a.A[1] - b.A[1], a.A[2] - b.A[2]};
            int lo[3], hi[3];
            for (int i = 0; i < 3; i++) {
                const double f = d[0] * G.binv[0 * 3 + i] + d[1] * G.binv[1 * 3 + i] + d[2] * G.binv[2 * 3 + i];
                const double w = rsum * G.bnorm[i];
                lo[i] = (int)ceil(f - w);
                hi[i] = (int)floor(f + w);
            }
            long long o = FILL ? off[e] : 0;
            for (int t0 = lo[0]; t0 <= hi[0]; t0++)
                for (int t1 = lo[1]; t1 <= hi[1]; t1++)
                    for (int t2 = lo[2]; t2 <= hi[2]; t2++) {
                        if (G.hermi && pa == pb && (t0 < 0 || (t0 == 0 && (t1 < 0 || (t1 == 0 && t2 < 0))))) continue;
                        Kept k;
                        if (!screen_pair(G, a, b, t0, t1, t2, k, sharp)) continue;
                        if (FILL) {
                            RawPair &r = raw[o];
                            r.pa = pa; r.pb = pb; r.T[0] = t0; r.T[1] = t1; r.T[2] = t2; r.level = k.level;
                            r.R = k.R; r.ap = k.ap; r.pref = k.pref;
                            for (int x = 0; x < 3; x++) { r.P[x] = k.P[x]; r.Bt[x] = k.Bt[x]; }
                            r.sym = (G.hermi && !(pa == pb && t0 == 0 && t1 == 0 && t2 == 0)) ? 1 : 0;
                            key[o] = (unsigned)((k.level * 8 + a.l + b.l) * 4 + a.l);
                            o++;
                        }
                        n++;
                    }
        }
    }
    if (!FILL) cnt[e] = n;
}

__global__ void __launch_bounds__(256) k_widen_counts(const unsigned *__restrict__ in, long long n, long long *__restrict__ out) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i];
}

__global__ void __launch_bounds__(256) k_iota(unsigned *p, long long n) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) p[i] = (unsigned)i;
}

struct ClassBase { long long v[GPW_MAX_LEVEL][8]; };

// Records of the sorted pairs: what the grid kernels (TaskK), the pre/post-pass (TaskP), the list builder (DevTask) and
// gpw_plan_export_tasks (gpw_task) read.
__global__ void __launch_bounds__(128) k_pair_records(const __grid_constant__ PairGeom G, const __grid_constant__ ClassBase base,
                                                      const DevPrim *__restrict__ prims, const RawPair *__restrict__ raw,
                                                      const unsigned *__restrict__ perm, int ntask, const double *__restrict__ gm,
                                                      TaskK *__restrict__ tk, TaskP *__restrict__ tp, DevTask *__restrict__ dt,
                                                      gpw_task *__restrict__ ex) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ntask) return;
    const RawPair r = raw[perm[i]];
    const DevPrim a = prims[r.pa], b = prims[r.pb];
    const int L = a.l + b.l;
    TaskK k;
    for (int x = 0; x < 3; x++)
        k.nP[x] = (r.P[0] * G.binv[0 * 3 + x] + r.P[1] * G.binv[1 * 3 + x] + r.P[2] * G.binv[2 * 3 + x]) * G.Nlev[r.level][x];
    k.ap = r.ap;
    const double *g = gm + 6 * r.level;    // the level's metric, packed 11 22 33 12 13 23
    k.c22 = exp(-2.0 * r.ap * g[1]);
    k.c23 = exp(-2.0 * r.ap * g[5]);
    k.c33 = exp(-2.0 * r.ap * g[2]);
    k.coef_off = base.v[r.level][L] + (long long)i * ncoef_pad(L);
    tk[i] = k;
    TaskP p;
    for (int x = 0; x < 3; x++) { p.PA[x] = r.P[x] - a.A[x]; p.PB[x] = r.P[x] - r.Bt[x]; }
    p.pref = r.pref; p.aa = a.exp; p.ab = b.exp;
    p.ao_a = a.ao; p.ao_b = b.ao; p.atom_a = a.atom; p.atom_b = b.atom;
    p.la = (short)a.l; p.lb = (short)b.l; p.level = (short)r.level; p.sym = (short)r.sym;
    tp[i] = p;
    DevTask d;
    d.P[0] = r.P[0]; d.P[1] = r.P[1]; d.P[2] = r.P[2]; d.R = r.R;
    d.level = r.level; d.L = L; d.la = a.l; d.lb = b.l;
    dt[i] = d;
    gpw_task t;
    t.shl_a = a.shl; t.prim_a = r.pa; t.shl_b = b.shl; t.prim_b = r.pb;
    t.T[0] = r.T[0]; t.T[1] = r.T[1]; t.T[2] = r.T[2]; t.level = r.level; t.R = r.R;
    ex[i] = t;
}

struct Scr {
    std::vector<void *> ptrs;
    ~Scr() { for (void *p : ptrs) cudaFree(p); }
    template <class T> bool alloc(T **p, size_t n) {
        *p = nullptr;
        if (cudaMalloc((void **)p, sizeof(T) * (n ? n : 1)) != cudaSuccess) return false;
        ptrs.push_back(*p);
        return true;
    }
    void release(void *p) { for (auto &q : ptrs) if (q == p) { q = ptrs.back(); ptrs.pop_back(); return; } }
};

int pfail(const char *what, cudaError_t e) {
    set_error(std::string("gpw_build_pairs (device pairs): ") + what + ": " + cudaGetErrorString(e));
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? GPW_ENOMEM : GPW_ECUDA;
}
#define PTRY(call, what) do { const cudaError_t e_ = (call); if (e_ != cudaSuccess) return pfail(what, e_); } while (0)
#define PALLOC(ptr, n, what) do { if (!S.alloc(ptr, n)) return pfail(what, cudaErrorMemoryAllocation); } while (0)

}  // namespace

void free_device_pairs(DevicePairs *d) {
    if (!d) return;
    cudaFree(d->taskK); cudaFree(d->taskP); cudaFree(d->devtask); cudaFree(d->exported);
    d->taskK = nullptr; d->taskP = nullptr; d->devtask = nullptr; d->exported = nullptr;
}

static int build_device_pairs_body(HostPlan *hp, DevicePairs *out, Scr &S) {
    const auto t_start = std::chrono::steady_clock::now();
    cudaStream_t st = 0;
    const int nprim = (int)hp->prims.size();
    PairGeom G;
    std::memset(&G, 0, sizeof(G));
    std::memcpy(G.cell, hp->cell, sizeof(G.cell));
    std::memcpy(G.binv, hp->binv, sizeof(G.binv));
    std::memcpy(G.bnorm, hp->bnorm, sizeof(G.bnorm));
    std::vector<double> gm(6 * (size_t)hp->nlevel);
    for (int a = 0; a < hp->nlevel; a++) {
        G.ecut[a] = hp->lev[a].ecut; G.circ[a] = hp->circ[a];
        for (int i = 0; i < 3; i++) G.Nlev[a][i] = hp->lev[a].N[i];
        for (int k = 0; k < 6; k++) gm[6 * a + k] = hp->lev[a].Gm[k];
    }
    G.tau = hp->tau; G.rel_cutoff = hp->rel_cutoff; G.nlevel = hp->nlevel; G.hermi = hp->hermi; G.nprim = nprim;

    DevPrim *d_prim = nullptr;
    double *d_gm = nullptr;
    unsigned *cnt = nullptr;
    long long *off = nullptr;
    int *d_sharp = nullptr;
    const long long npp = (long long)nprim * nprim;
    PALLOC(&d_prim, (size_t)nprim, "primitives"); PALLOC(&d_gm, gm.size(), "metric");
    PALLOC(&cnt, (size_t)npp, "counts"); PALLOC(&off, (size_t)npp, "counts"); PALLOC(&d_sharp, 1, "flag");
    PTRY(cudaMemcpyAsync(d_prim, hp->prims.data(), sizeof(DevPrim) * (size_t)nprim, cudaMemcpyHostToDevice, st), "primitives");
    PTRY(cudaMemcpyAsync(d_gm, gm.data(), sizeof(double) * gm.size(), cudaMemcpyHostToDevice, st), "metric");
    PTRY(cudaMemsetAsync(d_sharp, 0, sizeof(int), st), "flag");
    const unsigned grid = (unsigned)((npp + 127) / 128);
    k_pair_enum<false><<<grid, 128, 0, st>>>(G, d_prim, cnt, nullptr, nullptr, nullptr, d_sharp);
    PTRY(cudaGetLastError(), "count kernel");
    // exclusive scan of the counts (64-bit offsets)
    long long ntask = 0;
    {
        size_t tb = 0;
        k_widen_counts<<<(unsigned)((npp + 255) / 256), 256, 0, st>>>(cnt, npp, off);
        PTRY(cudaGetLastError(), "scan");
        PTRY(cub::DeviceScan::ExclusiveSum(nullptr, tb, off, off, npp, st), "scan");
        void *tmp = nullptr;
        PALLOC((char **)&tmp, tb, "scan scratch");
        PTRY(cub::DeviceScan::ExclusiveSum(tmp, tb, off, off, npp, st), "scan");
        long long last_off = 0;
        unsigned last_cnt = 0;
        int sharp = 0;
        PTRY(cudaMemcpyAsync(&last_off, off + npp - 1, sizeof(long long), cudaMemcpyDeviceToHost, st), "scan");
        PTRY(cudaMemcpyAsync(&last_cnt, cnt + npp - 1, sizeof(unsigned), cudaMemcpyDeviceToHost, st), "scan");
        PTRY(cudaMemcpyAsync(&sharp, d_sharp, sizeof(int), cudaMemcpyDeviceToHost, st), "scan");
        PTRY(cudaStreamSynchronize(st), "scan");
        ntask = last_off + last_cnt;
        if (sharp) {
            set_error("gpw_build_pairs: a primitive pair is far too sharp for the finest mesh (a_p (R_t + block diagonal)^2 > 600: "
                      "the Gaussian underflows at the corner of its own grid blocks); use a finer level 0");
            return GPW_EUNSUPPORTED;
        }
    }
    if (ntask > 2000000000LL) { set_error("gpw_build_pairs: more than 2^31 pairs"); return GPW_EUNSUPPORTED; }
    hp->ntask = (long)ntask;
    out->ntask = (long)ntask;
    if (ntask == 0) {
        hp->build_seconds += std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        return GPW_OK;
    }
    RawPair *raw = nullptr;
    unsigned *key = nullptr, *key2 = nullptr, *idx = nullptr, *perm = nullptr;
    PALLOC(&raw, (size_t)ntask, "pairs"); PALLOC(&key, (size_t)ntask, "keys"); PALLOC(&key2, (size_t)ntask, "keys");
    PALLOC(&idx, (size_t)ntask, "keys"); PALLOC(&perm, (size_t)ntask, "keys");
    k_pair_enum<true><<<grid, 128, 0, st>>>(G, d_prim, nullptr, off, raw, key, d_sharp);
    PTRY(cudaGetLastError(), "fill kernel");
    k_iota<<<(unsigned)((ntask + 255) / 256), 256, 0, st>>>(idx, ntask);
    {
        size_t tb = 0;
        PTRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, key, key2, idx, perm, (int)ntask, 0, 8, st), "sort");
        void *tmp = nullptr;
        PALLOC((char **)&tmp, tb, "sort scratch");
        PTRY(cub::DeviceRadixSort::SortPairs(tmp, tb, key, key2, idx, perm, (int)ntask, 0, 8, st), "sort");
    }
    // class sizes from the sorted keys (host: 256 classes)
    std::vector<unsigned> hkey((size_t)ntask);
    PTRY(cudaMemcpyAsync(hkey.data(), key2, sizeof(unsigned) * (size_t)ntask, cudaMemcpyDeviceToHost, st), "keys");
    PTRY(cudaStreamSynchronize(st), "keys");
    constexpr int NCLS = GPW_MAX_LEVEL * 8 * 4;
    long cls_first[NCLS + 1];
    {
        long pos = 0;
        for (int c = 0; c <= NCLS; c++) {
            while (pos < ntask && (int)hkey[(size_t)pos] < c) pos++;
            cls_first[c] = pos;
        }
    }
    long long coff[NOFF] = {0};
    ClassBase base;
    std::memset(&base, 0, sizeof(base));
    for (int c = 0; c < NCLS; c += 4) {
        const long n = cls_first[c + 4] - cls_first[c];
        const int level = c / 32, L = (c / 4) % 8;
        if (n == 0 || L > MAXLP) continue;
        for (int o = 0; o < NOFF; o++) {
            hp->coef_base[o][level][L] = coff[o] - (long long)cls_first[c] * ncoef_pad(L + o);
            coff[o] += (long long)n * ncoef_pad(L + o);
        }
        base.v[level][L] = hp->coef_base[0][level][L];
        hp->ntask_level[level] += n;
        hp->max_L = std::max(hp->max_L, L);
    }
    for (int o = 0; o < NOFF; o++) hp->ncoef_total[o] = coff[o];
    for (int a = 0; a < hp->nlevel; a++) { hp->big_lo[a] = cls_first[(a * 8 + 5) * 4]; hp->big_hi[a] = cls_first[(a * 8 + 7) * 4]; }
    PALLOC(&out->taskK, (size_t)ntask, "pair records"); PALLOC(&out->taskP, (size_t)ntask, "pair records");
    PALLOC(&out->devtask, (size_t)ntask, "pair records"); PALLOC(&out->exported, (size_t)ntask, "pair records");
    k_pair_records<<<(unsigned)((ntask + 127) / 128), 128, 0, st>>>(G, base, d_prim, raw, perm, (int)ntask, d_gm, out->taskK, out->taskP,
                                                                   out->devtask, out->exported);
    PTRY(cudaGetLastError(), "record kernel");
    PTRY(cudaStreamSynchronize(st), "record kernel");
    S.release(out->taskK); S.release(out->taskP); S.release(out->devtask); S.release(out->exported);
    out->bytes = (long)((sizeof(TaskK) + sizeof(TaskP) + sizeof(DevTask) + sizeof(gpw_task)) * (size_t)ntask);
    hp->build_seconds += std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    return GPW_OK;
}

int build_device_pairs(HostPlan *hp, DevicePairs *out) {
    Scr S;   // frees whatever has not been released to `out`
    const int rc = build_device_pairs_body(hp, out, S);
    if (rc != GPW_OK) { out->taskK = nullptr; out->taskP = nullptr; out->devtask = nullptr; out->exported = nullptr; }
    return rc;
}

}  // namespace gpw
