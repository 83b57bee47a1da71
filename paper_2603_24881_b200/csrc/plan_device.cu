// Device side of gpw_build_pairs: the block set of every pair (T6, T7; Alg. 4 l.10-13
// and Alg. 5 at :488-561 build the same kind of lists on the GPU) and from it the collocation visit lists, the
// integration brick lists and the work items of both grid kernels.  The pairs themselves (screening, level) come
// from pairs_device.cu.
//
// This file is compiled with -fmad=false: the geometric block test then performs exactly the IEEE operations of
// the host builder, so a block is visited on the device iff it is on the host, bit for bit.
//
// Pipeline (all on one stream):
//   k_task_lists<false>   one warp per pair: count its visits and brick entries
//   exclusive scans       offsets of every pair's visits / entries
//   k_task_lists<true>    write (key, record) of every visit and entry, in pair order
//   stable radix sorts    visits by (block, L); entries by (brick, L, blocks visited descending)
//   k_bounds_*            start of every block's / brick's list and of its L segments (binary search)
//   k_items_* / k_bitems_*  cut the lists into work items; sort the items by decreasing work
#include <cub/cub.cuh>
#include <cuda_runtime.h>

#include <chrono>
#include <cstring>

#include "gpw_kernels.cuh"
#include "plan_device.h"

namespace gpw {
namespace {

constexpr unsigned ITEM_MAX = 384;    // visits per collocation work item
// entries per integration work item: an item stages its brick of v once, so longer items stage less (cfg2
// k_integrate 3.58 -> 3.51 -> 3.46 ms, cfg4 26.8 -> 26.1 -> 25.3 ms with 768 -> 1536 -> 3072), but only while enough
// items are left to balance the SMs (cfg3: +3 % with 1536; cfg4: +3 % with one item per brick); the longest form that
// still leaves BITEM_PER_SM items per SM is used
constexpr unsigned BITEM_MAX = 768, BITEM_BIG = 1536, BITEM_HUGE = 3072;
constexpr long long BITEM_PER_SM = 40;

__device__ __forceinline__ int floordiv_d(int n, int d) { return n >= 0 ? n / d : -((-n + d - 1) / d); }
__device__ __forceinline__ int posmod_d(int n, int d) { const int m = n % d; return m < 0 ? m + d : m; }

// T6: is at least one of the 64 points of block (b1,b2,b3) (unbounded indices) within R of P?
__device__ bool block_hit(const ListGeom &G, const LevelList &g, const DevTask &t, double rc, int b1, int b2, int b3) {
    const int *N = g.N;
    double dc = 0.0;
    {
        const double u1 = (4 * b1 + 1.5) / N[0], u2 = (4 * b2 + 1.5) / N[1], u3 = (4 * b3 + 1.5) / N[2];
        for (int x = 0; x < 3; x++) {
            const double cp = u1 * G.cell[0 * 3 + x] + u2 * G.cell[1 * 3 + x] + u3 * G.cell[2 * 3 + x];
            dc += (cp - t.P[x]) * (cp - t.P[x]);
        }
        dc = sqrt(dc);
    }
    if (dc - rc > t.R * (1.0 + 1e-9) + 1e-9) return false;
    if (dc + rc < t.R * (1.0 - 1e-9) - 1e-9) return true;
    const double R2 = t.R * t.R;
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++)
            for (int k = 0; k < 4; k++) {
                // r_n = (n1/N1) a1 + (n2/N2) a2 + (n3/N3) a3   (u0 = 0)
                const double u1 = (double)(4 * b1 + i) / N[0], u2 = (double)(4 * b2 + j) / N[1],
                             u3 = (double)(4 * b3 + k) / N[2];
                double r[3];
                for (int x = 0; x < 3; x++) r[x] = u1 * G.cell[0 * 3 + x] + u2 * G.cell[1 * 3 + x] + u3 * G.cell[2 * 3 + x];
                const double d2 = (r[0] - t.P[0]) * (r[0] - t.P[0]) + (r[1] - t.P[1]) * (r[1] - t.P[1]) +
                                  (r[2] - t.P[2]) * (r[2] - t.P[2]);
                if (d2 <= R2) return true;
            }
    return false;
}

// One warp per pair.  The candidate box is walked in runs that stay inside one brick and one lattice image
// along n2 and n3 (at most BR2 x BR3 = 25 blocks, one per lane), so the ballot of the hits IS the entry's mask.
template <bool FILL>
__global__ void __launch_bounds__(128) k_task_lists(const __grid_constant__ ListGeom G, const DevTask *__restrict__ tasks,
                                                    int ntask, unsigned *__restrict__ nvis, unsigned *__restrict__ nent,
                                                    const long long *__restrict__ voff, const long long *__restrict__ eoff,
                                                    unsigned *__restrict__ vkey, unsigned long long *__restrict__ vval,
                                                    unsigned *__restrict__ ekey, uint4 *__restrict__ eval,
                                                    unsigned long long *__restrict__ cls, int *__restrict__ overflow) {
    const int ti = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    if (ti >= ntask) return;
    const int lane = threadIdx.x & 31;
    const DevTask t = tasks[ti];
    const LevelList &g = G.lev[t.level];
    const double rc = G.circ[t.level];
    int blo[3], bhi[3];
    for (int i = 0; i < 3; i++) {
        const double u = t.P[0] * G.binv[0 * 3 + i] + t.P[1] * G.binv[1 * 3 + i] + t.P[2] * G.binv[2 * 3 + i];
        const double w = t.R * G.bnorm[i] * g.N[i];
        blo[i] = floordiv_d((int)ceil(u * g.N[i] - w), TILE);
        bhi[i] = floordiv_d((int)floor(u * g.N[i] + w), TILE);
    }
    const int j2 = lane / BR3, j3 = lane - j2 * BR3;
    long long vpos = FILL ? voff[ti] : 0, epos = FILL ? eoff[ti] : 0;
    unsigned cv = 0, ce = 0;
    for (int b1 = blo[0]; b1 <= bhi[0]; b1++) {
        const int w1 = posmod_d(b1, g.T[0]), s1 = (b1 - w1) / g.T[0];
        for (int r2 = blo[1]; r2 <= bhi[1];) {
            const int w2 = posmod_d(r2, g.T[1]), o2 = w2 % BR2;
            const int start2 = r2 - o2, len2 = min(BR2, g.T[1] - (w2 - o2));   // the brick's run along n2 (ragged last brick)
            const int s2 = (r2 - w2) / g.T[1];
            for (int r3 = blo[2]; r3 <= bhi[2];) {
                const int w3 = posmod_d(r3, g.T[2]), o3 = w3 % BR3;
                const int start3 = r3 - o3, len3 = min(BR3, g.T[2] - (w3 - o3));
                const int s3 = (r3 - w3) / g.T[2];
                const int b2 = start2 + j2, b3 = start3 + j3;
                bool hit = false;
                if (lane < BRICK_TILES && j2 < len2 && j3 < len3 && b2 >= blo[1] && b2 <= bhi[1] && b3 >= blo[2] && b3 <= bhi[2])
                    hit = block_hit(G, g, t, rc, b1, b2, b3);
                const unsigned mask = __ballot_sync(0xffffffffu, hit);
                if (mask) {
                    if (s1 < -127 || s1 > 127 || s2 < -127 || s2 > 127 || s3 < -127 || s3 > 127) {
                        if (lane == 0) *overflow = 1;
                    } else {
                        if (FILL) {
                            const unsigned sb = (unsigned)(unsigned char)(signed char)s1 | ((unsigned)(unsigned char)(signed char)s2 << 8) |
                                                ((unsigned)(unsigned char)(signed char)s3 << 16);
                            if (hit) {
                                const long long p = vpos + __popc(mask & ((1u << lane) - 1u));
                                const int ws2 = w2 - o2 + j2, ws3 = w3 - o3 + j3;
                                const unsigned blk = (unsigned)(g.tile0 + ((long long)w1 * g.T[1] + ws2) * g.T[2] + ws3);
                                vkey[p] = (blk << 3) | (unsigned)t.L;
                                vval[p] = (unsigned long long)(unsigned)ti | ((unsigned long long)sb << 32);
                            }
                            if (lane == 0) {
                                const unsigned brick = (unsigned)(g.brick0 + ((long long)(w1 / BR1) * g.B[1] + (w2 / BR2)) * g.B[2] + (w3 / BR3));
                                ekey[epos] = (brick << 8) | ((unsigned)t.L << 5) | (unsigned)(BRICK_TILES - __popc(mask));
                                eval[epos] = make_uint4((unsigned)ti, sb | ((unsigned)t.L << 24), mask, 0u);
                            }
                        }
                        vpos += __popc(mask);
                        epos += 1;
                        cv += (unsigned)__popc(mask);
                        ce += 1u;
                    }
                }
                r3 = start3 + len3;
            }
            r2 = start2 + len2;
        }
    }
    if (!FILL && lane == 0) {
        nvis[ti] = cv;
        nent[ti] = ce;
        if (cv) atomicAdd(cls + ((size_t)t.level * (MAXL + 1) + t.la) * (MAXL + 1) + t.lb, (unsigned long long)cv);
    }
}

// ---------------------------------------------------------------------------------------- list bounds
__device__ __forceinline__ long long lower_bound_u32(const unsigned *__restrict__ a, long long n, unsigned key) {
    long long lo = 0, hi = n;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// start of every (block, L) segment in the sorted visit keys; base[b] = start of block b, base[nblock] = n
__global__ void k_bounds_visits(const unsigned *__restrict__ keys, long long n, long long nblock,
                                long long *__restrict__ base, unsigned *__restrict__ seg) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;   // (block, L)
    if (i > nblock * 8) return;
    if (i == nblock * 8) { base[nblock] = n; return; }
    const long long b = i >> 3;
    const long long first = lower_bound_u32(keys, n, (unsigned)(b << 3));
    const long long mine = (i & 7) ? lower_bound_u32(keys, n, (unsigned)i) : first;
    if ((i & 7) == 0) base[b] = first;
    seg[i] = (unsigned)(mine - first);
}

// start of every brick's entry list in the sorted entry keys
__global__ void k_bounds_bricks(const unsigned *__restrict__ keys, long long n, long long nbrick, long long *__restrict__ base) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b > nbrick) return;
    base[b] = b == nbrick ? n : lower_bound_u32(keys, n, (unsigned)(b << 8));
}

__device__ __forceinline__ int level_of(const ListGeom &G, long long id, bool brick, long long *local) {
    int a = 0;
    for (; a + 1 < G.nlevel; a++) {
        const long long next = brick ? G.lev[a + 1].brick0 : G.lev[a + 1].tile0;
        if (id < next) break;
    }
    *local = id - (brick ? G.lev[a].brick0 : G.lev[a].tile0);
    return a;
}

// ---------------------------------------------------------------------------------------- work items
// seg != nullptr: only the tail of every block's list that starts at its segment llo (classes L >= llo)
__global__ void k_items_count(const long long *__restrict__ base, long long nblock, unsigned *__restrict__ nparts, unsigned maxlen,
                              const unsigned *__restrict__ seg = nullptr, int llo = 0) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= nblock) return;
    unsigned n = (unsigned)(base[b + 1] - base[b]);
    if (seg) n -= seg[b * 8 + llo];
    nparts[b] = (n + maxlen - 1) / maxlen;
}

__global__ void k_items_fill(const __grid_constant__ ListGeom G, const long long *__restrict__ base, long long nblock,
                             const unsigned *__restrict__ nparts, const long long *__restrict__ off,
                             unsigned *__restrict__ key, Item *__restrict__ items,
                             const unsigned *__restrict__ seg = nullptr, int llo = 0) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= nblock) return;
    const unsigned np = nparts[b];
    if (!np) return;
    const unsigned first = seg ? seg[b * 8 + llo] : 0u;   // the items cover [first, end of the block's list)
    const unsigned n = (unsigned)(base[b + 1] - base[b]) - first;
    long long local;
    const int level = level_of(G, b, false, &local);
    for (unsigned p = 0; p < np; p++) {
        Item it;
        it.level = level; it.tile = (int)local;
        it.lo = first + (unsigned)((unsigned long long)n * p / np);
        it.hi = first + (unsigned)((unsigned long long)n * (p + 1) / np);
        it.single = np == 1; it.pad = 0;
        it.vstart = base[b] + it.lo;
        items[off[b] + p] = it;
        key[off[b] + p] = ITEM_MAX - (it.hi - it.lo);   // ascending key = decreasing length
    }
}

__global__ void k_bitems_fill(const __grid_constant__ ListGeom G, const long long *__restrict__ base, long long nbrick,
                              const unsigned *__restrict__ nparts, const long long *__restrict__ off,
                              const unsigned *__restrict__ ekeys, long long nentry, const uint4 *__restrict__ entries,
                              unsigned *__restrict__ key, BItem *__restrict__ items) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= nbrick) return;
    const unsigned np = nparts[b];
    if (!np) return;
    const long long first = base[b];
    const unsigned n = (unsigned)(base[b + 1] - first);
    long long local;
    const int level = level_of(G, b, true, &local);
    BItem proto;
    proto.level = level; proto.brick = (int)local; proto.base = first; proto.lo = 0; proto.hi = 0;
    proto.pad[0] = proto.pad[1] = 0;
    for (int L = 0; L < 8; L++)
        proto.seg[L] = (unsigned)(lower_bound_u32(ekeys + first, n, (unsigned)((b << 8) | ((unsigned)L << 5))));
    for (unsigned p = 0; p < np; p++) {
        BItem it = proto;
        it.lo = (unsigned)((unsigned long long)n * p / np);
        it.hi = (unsigned)((unsigned long long)n * (p + 1) / np);
        unsigned work = 0;
        for (unsigned e = it.lo; e < it.hi; e++) {
            const uint4 en = entries[first + e];
            work += (unsigned)__popc(en.z) * (4u + (en.y >> 24));
        }
        items[off[b] + p] = it;
        key[off[b] + p] = 0x7fffffffu - work;   // ascending key = decreasing work
    }
}

}  // namespace

// =========================================================================================== host driver
namespace {

struct Scratch {   // frees what is still held when it goes out of scope
    std::vector<void *> ptrs;
    ~Scratch() { for (void *p : ptrs) cudaFree(p); }
    template <class T> bool alloc(T **p, size_t n, long *bytes = nullptr) {
        *p = nullptr;
        const size_t nb = sizeof(T) * (n ? n : 1);
        if (cudaMalloc((void **)p, nb) != cudaSuccess) return false;
        ptrs.push_back(*p);
        if (bytes) *bytes += (long)nb;
        return true;
    }
    void release(void *p) {   // ownership moves to the caller
        for (auto &q : ptrs) if (q == p) { q = ptrs.back(); ptrs.pop_back(); return; }
    }
    void free_now(void *p) { release(p); cudaFree(p); }
};

int fail(const char *what, cudaError_t e) {
    set_error(std::string("gpw_build_pairs (device lists): ") + what + ": " + cudaGetErrorString(e));
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? GPW_ENOMEM : GPW_ECUDA;
}

#define GPW_TRY(call, what) do { const cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(what, e_); } while (0)
#define GPW_ALLOC(ptr, n, what) do { if (!S.alloc(ptr, n)) return fail(what, cudaErrorMemoryAllocation); } while (0)

__global__ void k_widen(const unsigned *__restrict__ in, long long n, long long *__restrict__ out) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i];
}

// exclusive sum of unsigned counts into long long offsets; total returned on the host
int scan_counts(Scratch &S, const unsigned *cnt, long long n, long long *off, long long *total, cudaStream_t st) {
    if (n == 0) { *total = 0; return GPW_OK; }
    k_widen<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cnt, n, off);
    GPW_TRY(cudaGetLastError(), "scan");
    size_t tb = 0;
    GPW_TRY(cub::DeviceScan::ExclusiveSum(nullptr, tb, off, off, n, st), "scan");
    void *tmp = nullptr;
    GPW_ALLOC((char **)&tmp, tb, "scan scratch");
    GPW_TRY(cub::DeviceScan::ExclusiveSum(tmp, tb, off, off, n, st), "scan");
    long long last_off = 0;
    unsigned last_cnt = 0;
    GPW_TRY(cudaMemcpyAsync(&last_off, off + n - 1, sizeof(long long), cudaMemcpyDeviceToHost, st), "scan");
    GPW_TRY(cudaMemcpyAsync(&last_cnt, cnt + n - 1, sizeof(unsigned), cudaMemcpyDeviceToHost, st), "scan");
    GPW_TRY(cudaStreamSynchronize(st), "scan");
    S.free_now(tmp);
    *total = last_off + last_cnt;
    return GPW_OK;
}

template <class V>
int sort_pairs(Scratch &S, const unsigned *kin, unsigned *kout, const V *vin, V *vout, long long n, int bits, cudaStream_t st) {
    if (n == 0) return GPW_OK;
    if (n > 0x7fffffffLL) { set_error("gpw_build_pairs: more than 2^31 list elements"); return GPW_EUNSUPPORTED; }
    size_t tb = 0;
    GPW_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, kin, kout, vin, vout, (int)n, 0, bits, st), "sort");
    void *tmp = nullptr;
    GPW_ALLOC((char **)&tmp, tb, "sort scratch");
    GPW_TRY(cub::DeviceRadixSort::SortPairs(tmp, tb, kin, kout, vin, vout, (int)n, 0, bits, st), "sort");
    GPW_TRY(cudaStreamSynchronize(st), "sort");
    S.free_now(tmp);
    return GPW_OK;
}

int bits_for(unsigned long long maxval) {
    int b = 1;
    while (b < 32 && (maxval >> b)) b++;
    return b;
}

}  // namespace

void free_device_lists(DeviceLists *l) {
    if (!l) return;
    cudaFree(l->visit); cudaFree(l->tile_base); cudaFree(l->seg); cudaFree(l->item); cudaFree(l->item_hi);
    l->item_hi = nullptr; l->nitem_hi = 0;
    cudaFree(l->bentry); cudaFree(l->brick_base); cudaFree(l->bitem);
    l->visit = nullptr; l->tile_base = nullptr; l->seg = nullptr; l->item = nullptr;
    l->bentry = nullptr; l->brick_base = nullptr; l->bitem = nullptr;
}

int build_device_lists(const HostPlan *hp, const DevTask *d_task, int ntask, DeviceLists *out) {
    cudaStream_t st = 0;
    const auto t_start = std::chrono::steady_clock::now();
    Scratch S;
    // ---- geometry and the pairs ----
    ListGeom G;
    std::memset(&G, 0, sizeof(G));
    std::memcpy(G.cell, hp->cell, sizeof(G.cell));
    std::memcpy(G.binv, hp->binv, sizeof(G.binv));
    std::memcpy(G.bnorm, hp->bnorm, sizeof(G.bnorm));
    G.nlevel = hp->nlevel;
    long long ntile_all = 0, nbrick_all = 0;
    for (int a = 0; a < hp->nlevel; a++) {
        const LevelGeom &g = hp->lev[a];
        LevelList &l = G.lev[a];
        for (int i = 0; i < 3; i++) { l.N[i] = g.N[i]; l.T[i] = g.T[i]; l.B[i] = g.B[i]; }
        l.ntile = g.ntile; l.nbrick = g.nbrick; l.tile0 = ntile_all; l.brick0 = nbrick_all;
        G.circ[a] = hp->circ[a];
        ntile_all += g.ntile; nbrick_all += g.nbrick;
    }
    if (ntile_all >= (1LL << 29) || nbrick_all >= (1LL << 24)) {
        set_error("gpw_build_pairs: meshes too large for the 32-bit list keys");
        return GPW_EUNSUPPORTED;
    }
    long &nb = out->bytes;
    // list offsets exist even for an empty plan
    {
        long long *tb = nullptr, *bb = nullptr;
        unsigned *sg = nullptr;
        if (!S.alloc(&tb, (size_t)ntile_all + 1, &nb) || !S.alloc(&sg, (size_t)ntile_all * 8, &nb) ||
            !S.alloc(&bb, (size_t)nbrick_all + 1, &nb))
            return fail("list offsets", cudaErrorMemoryAllocation);
        out->tile_base = tb; out->seg = sg; out->brick_base = bb;
    }
    auto give_up = [&](int rc) { out->tile_base = nullptr; out->seg = nullptr; out->brick_base = nullptr; out->visit = nullptr;
                                 out->item = nullptr; out->item_hi = nullptr; out->nitem_hi = 0;
                                 out->bentry = nullptr; out->bitem = nullptr; return rc; };
    if (ntask == 0) {
        cudaMemsetAsync(out->tile_base, 0, sizeof(long long) * ((size_t)ntile_all + 1), st);
        cudaMemsetAsync(out->seg, 0, sizeof(unsigned) * (size_t)ntile_all * 8, st);
        cudaMemsetAsync(out->brick_base, 0, sizeof(long long) * ((size_t)nbrick_all + 1), st);
        if (cudaStreamSynchronize(st) != cudaSuccess) return give_up(fail("clear", cudaGetLastError()));
        S.release(out->tile_base); S.release(out->seg); S.release(out->brick_base);
        return GPW_OK;
    }
    int rc = GPW_OK;
    auto body = [&]() -> int {
        // ---- count ----
        unsigned *nvis = nullptr, *nent = nullptr;
        long long *voff = nullptr, *eoff = nullptr;
        unsigned long long *d_cls = nullptr;
        int *d_ovf = nullptr;
        constexpr size_t NCLS = (size_t)GPW_MAX_LEVEL * (MAXL + 1) * (MAXL + 1);
        GPW_ALLOC(&nvis, (size_t)ntask, "counts"); GPW_ALLOC(&nent, (size_t)ntask, "counts");
        GPW_ALLOC(&voff, (size_t)ntask, "counts"); GPW_ALLOC(&eoff, (size_t)ntask, "counts");
        GPW_ALLOC(&d_cls, NCLS, "counts"); GPW_ALLOC(&d_ovf, 1, "counts");
        GPW_TRY(cudaMemsetAsync(d_cls, 0, sizeof(unsigned long long) * NCLS, st), "counts");
        GPW_TRY(cudaMemsetAsync(d_ovf, 0, sizeof(int), st), "counts");
        const unsigned tgrid = (unsigned)(((long long)ntask * 32 + 127) / 128);
        k_task_lists<false><<<tgrid, 128, 0, st>>>(G, d_task, ntask, nvis, nent, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, d_cls, d_ovf);
        GPW_TRY(cudaGetLastError(), "count kernel");
        long long nvisit = 0, nentry = 0;
        if ((rc = scan_counts(S, nvis, ntask, voff, &nvisit, st)) != GPW_OK) return rc;
        if ((rc = scan_counts(S, nent, ntask, eoff, &nentry, st)) != GPW_OK) return rc;
        int ovf = 0;
        GPW_TRY(cudaMemcpy(&ovf, d_ovf, sizeof(int), cudaMemcpyDeviceToHost), "counts");
        GPW_TRY(cudaMemcpy(out->cls, d_cls, sizeof(unsigned long long) * NCLS, cudaMemcpyDeviceToHost), "counts");
        if (ovf) { set_error("gpw_build_pairs: a pair wraps the cell more than 127 times"); return GPW_EUNSUPPORTED; }
        out->nvisit = nvisit; out->nentry = nentry;
        // ---- fill ----
        unsigned *vkey = nullptr, *vkey2 = nullptr, *ekey = nullptr, *ekey2 = nullptr;
        unsigned long long *vval = nullptr, *vval2 = nullptr;
        uint4 *eval = nullptr, *eval2 = nullptr;
        GPW_ALLOC(&vkey, (size_t)nvisit, "visit keys"); GPW_ALLOC(&vval, (size_t)nvisit, "visit records");
        GPW_ALLOC(&ekey, (size_t)nentry, "entry keys"); GPW_ALLOC(&eval, (size_t)nentry, "entry records");
        k_task_lists<true><<<tgrid, 128, 0, st>>>(G, d_task, ntask, nvis, nent, voff, eoff, vkey, vval, ekey, eval, d_cls, d_ovf);
        GPW_TRY(cudaGetLastError(), "fill kernel");
        GPW_TRY(cudaStreamSynchronize(st), "fill kernel");
        S.free_now(nvis); S.free_now(nent); S.free_now(voff); S.free_now(eoff);
        // ---- visits: stable sort by (block, L); pair order is kept inside ----
        GPW_ALLOC(&vkey2, (size_t)nvisit, "visit keys");
        if (!S.alloc(&vval2, (size_t)nvisit, &nb)) return fail("visit lists", cudaErrorMemoryAllocation);
        if ((rc = sort_pairs(S, vkey, vkey2, vval, vval2, nvisit, bits_for((unsigned long long)ntile_all << 3), st)) != GPW_OK) return rc;
        S.free_now(vkey); S.free_now(vval);
        {
            const long long n = ntile_all * 8 + 1;
            k_bounds_visits<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(vkey2, nvisit, ntile_all, out->tile_base, out->seg);
            GPW_TRY(cudaGetLastError(), "visit bounds");
        }
        // ---- collocation work items ----
        {
            unsigned *np = nullptr, *ikey = nullptr, *ikey2 = nullptr;
            long long *ioff = nullptr;
            Item *it = nullptr, *it2 = nullptr;
            GPW_ALLOC(&np, (size_t)ntile_all, "items"); GPW_ALLOC(&ioff, (size_t)ntile_all, "items");
            k_items_count<<<(unsigned)((ntile_all + 255) / 256), 256, 0, st>>>(out->tile_base, ntile_all, np, ITEM_MAX);
            GPW_TRY(cudaGetLastError(), "items");
            long long nitem = 0;
            if ((rc = scan_counts(S, np, ntile_all, ioff, &nitem, st)) != GPW_OK) return rc;
            GPW_ALLOC(&ikey, (size_t)nitem, "items"); GPW_ALLOC(&ikey2, (size_t)nitem, "items");
            GPW_ALLOC(&it, (size_t)nitem, "items");
            if (!S.alloc(&it2, (size_t)nitem, &nb)) return fail("items", cudaErrorMemoryAllocation);
            k_items_fill<<<(unsigned)((ntile_all + 255) / 256), 256, 0, st>>>(G, out->tile_base, ntile_all, np, ioff, ikey, it);
            GPW_TRY(cudaGetLastError(), "items");
            if ((rc = sort_pairs(S, ikey, ikey2, it, it2, nitem, bits_for(ITEM_MAX), st)) != GPW_OK) return rc;
            S.free_now(np); S.free_now(ioff); S.free_now(ikey); S.free_now(ikey2); S.free_now(it);
            out->item = it2; out->nitem = (long)nitem;
        }
        // ---- ... and, on plans with f shells, the items of the second collocation launch: the visits of the classes
        //      L >= 5 (the tail of every block's list), so that the launch holds no item without work ----
        if (hp->max_L >= 5) {
            unsigned *np = nullptr, *ikey = nullptr, *ikey2 = nullptr;
            long long *ioff = nullptr;
            Item *it = nullptr, *it2 = nullptr;
            GPW_ALLOC(&np, (size_t)ntile_all, "items"); GPW_ALLOC(&ioff, (size_t)ntile_all, "items");
            k_items_count<<<(unsigned)((ntile_all + 255) / 256), 256, 0, st>>>(out->tile_base, ntile_all, np, ITEM_MAX, out->seg, 5);
            GPW_TRY(cudaGetLastError(), "items");
            long long nitem = 0;
            if ((rc = scan_counts(S, np, ntile_all, ioff, &nitem, st)) != GPW_OK) return rc;
            if (nitem > 0) {
                GPW_ALLOC(&ikey, (size_t)nitem, "items"); GPW_ALLOC(&ikey2, (size_t)nitem, "items");
                GPW_ALLOC(&it, (size_t)nitem, "items");
                if (!S.alloc(&it2, (size_t)nitem, &nb)) return fail("items", cudaErrorMemoryAllocation);
                k_items_fill<<<(unsigned)((ntile_all + 255) / 256), 256, 0, st>>>(G, out->tile_base, ntile_all, np, ioff, ikey, it, out->seg, 5);
                GPW_TRY(cudaGetLastError(), "items");
                if ((rc = sort_pairs(S, ikey, ikey2, it, it2, nitem, bits_for(ITEM_MAX), st)) != GPW_OK) return rc;
                S.free_now(ikey); S.free_now(ikey2); S.free_now(it);
                out->item_hi = it2; out->nitem_hi = (long)nitem;
            }
            S.free_now(np); S.free_now(ioff);
        }
        S.free_now(vkey2);
        out->visit = reinterpret_cast<Visit *>(vval2);
        // ---- brick entries: stable sort by (brick, L, blocks visited descending) ----
        GPW_ALLOC(&ekey2, (size_t)nentry, "entry keys");
        if (!S.alloc(&eval2, (size_t)nentry, &nb)) return fail("brick lists", cudaErrorMemoryAllocation);
        if ((rc = sort_pairs(S, ekey, ekey2, eval, eval2, nentry, bits_for((unsigned long long)nbrick_all << 8), st)) != GPW_OK) return rc;
        S.free_now(ekey); S.free_now(eval);
        k_bounds_bricks<<<(unsigned)((nbrick_all + 1 + 255) / 256), 256, 0, st>>>(ekey2, nentry, nbrick_all, out->brick_base);
        GPW_TRY(cudaGetLastError(), "brick bounds");
        {
            unsigned *np = nullptr, *ikey = nullptr, *ikey2 = nullptr;
            long long *ioff = nullptr;
            BItem *it = nullptr, *it2 = nullptr;
            GPW_ALLOC(&np, (size_t)nbrick_all, "brick items"); GPW_ALLOC(&ioff, (size_t)nbrick_all, "brick items");
            int dev = 0, nsm = 0;
            GPW_TRY(cudaGetDevice(&dev), "brick items");
            GPW_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), "brick items");
            long long nbitem = 0;
            for (unsigned maxlen : {BITEM_HUGE, BITEM_BIG, BITEM_MAX}) {
                k_items_count<<<(unsigned)((nbrick_all + 255) / 256), 256, 0, st>>>(out->brick_base, nbrick_all, np, maxlen);
                GPW_TRY(cudaGetLastError(), "brick items");
                if ((rc = scan_counts(S, np, nbrick_all, ioff, &nbitem, st)) != GPW_OK) return rc;
                if (nbitem >= BITEM_PER_SM * nsm) break;
            }
            GPW_ALLOC(&ikey, (size_t)nbitem, "brick items"); GPW_ALLOC(&ikey2, (size_t)nbitem, "brick items");
            GPW_ALLOC(&it, (size_t)nbitem, "brick items");
            if (!S.alloc(&it2, (size_t)nbitem, &nb)) return fail("brick items", cudaErrorMemoryAllocation);
            k_bitems_fill<<<(unsigned)((nbrick_all + 255) / 256), 256, 0, st>>>(G, out->brick_base, nbrick_all, np, ioff, ekey2, nentry, eval2, ikey, it);
            GPW_TRY(cudaGetLastError(), "brick items");
            if ((rc = sort_pairs(S, ikey, ikey2, it, it2, nbitem, 31, st)) != GPW_OK) return rc;
            S.free_now(np); S.free_now(ioff); S.free_now(ikey); S.free_now(ikey2); S.free_now(it);
            out->bitem = it2; out->nbitem = (long)nbitem;
        }
        S.free_now(ekey2);
        out->bentry = reinterpret_cast<BEntry *>(eval2);
        GPW_TRY(cudaStreamSynchronize(st), "device lists");
        return GPW_OK;
    };
    rc = body();
    if (rc != GPW_OK) return give_up(rc);   // Scratch frees everything, including what `out` pointed at
    S.release(out->tile_base); S.release(out->seg); S.release(out->brick_base);
    S.release(out->visit); S.release(out->item); S.release(out->bentry); S.release(out->bitem);
    if (out->item_hi) S.release(out->item_hi);
    out->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    return GPW_OK;
}

}  // namespace gpw
