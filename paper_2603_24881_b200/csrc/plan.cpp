// Host side of gpw_build_pairs: argument checks, level geometry and the primitive cutoff radii (T1) always; pair
// screening, lattice images, level assignment and per-block visit lists only when there is no CUDA device (a
// host-only plan for introspection -- with a device these run there: pairs_device.cu, plan_device.cu).  Follows DESIGN.md T1..T6 (readings of PAPER.md:59, :123-138, :162-164, :200,
// Alg. 4-5 at :435-561).  Plain C++17 + std::thread; no code shared with oracle/.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstring>
#include <thread>

#include "gpw_internal.h"

namespace gpw {

static thread_local std::string g_err;
void set_error(const std::string &msg) { g_err = msg; }
const char *last_error_cstr() { return g_err.c_str(); }

namespace {

// A grid block index (unbounded) folded into the cell: stored index and the number of lattice wraps (T7).
struct Folded { int stored, wraps; };
inline Folded fold(int b, int nblk) {
    const int stored = ((b % nblk) + nblk) % nblk;
    return Folded{stored, (b - stored) / nblk};
}
// block that holds grid index n (floor division by the block edge)
inline int block_of(int n) { return n >= 0 ? n / TILE : -((TILE - 1 - n) / TILE); }

// Readings T1 and T4 share one scheme: the largest root of
//     K prod_k (r + shift_k)^power_k exp(-a r^2) = tau
// by 40 steps of  r <- sqrt((ln K - ln tau + sum_k power_k ln(r + shift_k)) / a)  from a start value beyond the root;
// a non-positive argument means that the envelope never reaches tau (radius 0: dropped).
struct EnvelopeTerm { double power, shift; };
double envelope_root(double lnK_over_tau, double a, double start, const EnvelopeTerm *term, int nterm) {
    double r = start;
    for (int step = 0; step < 40; step++) {
        double num = lnK_over_tau;
        for (int k = 0; k < nterm; k++) num += term[k].power * std::log(r + term[k].shift);
        const double arg = num / a;
        if (arg <= 0.0) return 0.0;
        r = std::sqrt(arg);
    }
    return r;
}
// T1 (Eq. 20): r^2 |coef| r^l exp(-a r^2) = tau
double prim_radius(int l, double a, double coef, double tau) {
    const double C = std::log(std::fabs(coef)) - std::log(tau);
    const EnvelopeTerm t[1] = {{(double)(l + 2), 0.0}};
    return envelope_root(C, a, std::sqrt(std::max(C, 1.0) / a) + 5.0, t, 1);
}
// T4: r^2 kappa (r + dA)^la (r + dB)^lb exp(-a_p r^2) = tau
double pair_radius(int la, int lb, double ap, double kappa, double dA, double dB, double tau) {
    const double C = std::log(kappa) - std::log(tau);
    const EnvelopeTerm t[3] = {{2.0, 0.0}, {(double)la, dA}, {(double)lb, dB}};
    return envelope_root(C, ap, std::sqrt(std::max(C, 1.0) / ap) + dA + dB + 5.0, t, 3);
}

// Reciprocal vectors b_i = (a_j x a_k) / det (i, j, k cyclic), stored as the columns of inverse(cell):
// binv[c*3+i] = component c of b_i.  False for a singular cell.
bool reciprocal_vectors(const double *cell, double *binv, double *det_out) {
    auto cross = [](const double *u, const double *v, double *w) {
        w[0] = u[1] * v[2] - u[2] * v[1]; w[1] = u[2] * v[0] - u[0] * v[2]; w[2] = u[0] * v[1] - u[1] * v[0];
    };
    const double *a0 = cell, *a1 = cell + 3, *a2 = cell + 6;
    double n0[3], n1[3], n2[3];
    cross(a1, a2, n0); cross(a2, a0, n1); cross(a0, a1, n2);
    const double det = a0[0] * n0[0] + a0[1] * n0[1] + a0[2] * n0[2];
    *det_out = det;
    if (std::fabs(det) < 1e-12) return false;
    for (int c = 0; c < 3; c++) { binv[c * 3 + 0] = n0[c] / det; binv[c * 3 + 1] = n1[c] / det; binv[c * 3 + 2] = n2[c] / det; }
    return true;
}

// index of monomial (a,b,c), a+b+c = d, inside its degree block: decreasing a, then decreasing b
inline int graded_idx(int a, int b, int d) {
    const int r = d - a;  // number of rows before: sum_{a'>a} (d-a'+1)
    return r * (r + 1) / 2 + (r - b);
}

// S_d[row (p,q,r)][col (a,b,c)] = coefficient of u1^p u2^q u3^r in (H0.u)^a (H1.u)^b (H2.u)^c
void build_S(const double *H, std::vector<double> &S) {
    S.assign(S_TOTAL, 0.0);
    constexpr int ND = MAXDEG + 1;
    for (int d = 0; d <= MAXDEG; d++) {
        const int nd = (d + 1) * (d + 2) / 2;
        double *blk = S.data() + s_block_off(d);
        for (int a = d; a >= 0; a--)
            for (int b = d - a; b >= 0; b--) {
                const int c = d - a - b;
                const int col = graded_idx(a, b, d);
                double poly[ND][ND][ND];
                std::memset(poly, 0, sizeof(poly));
                poly[0][0][0] = 1.0;
                int deg = 0;
                const int reps[3] = {a, b, c};
                for (int x = 0; x < 3; x++)
                    for (int rep = 0; rep < reps[x]; rep++) {
                        double nxt[ND][ND][ND];
                        std::memset(nxt, 0, sizeof(nxt));
                        for (int p = 0; p <= deg; p++)
                            for (int q = 0; q <= deg - p; q++) {
                                const int r = deg - p - q;
                                const double v = poly[p][q][r];
                                if (v == 0.0) continue;
                                nxt[p + 1][q][r] += v * H[x * 3 + 0];
                                nxt[p][q + 1][r] += v * H[x * 3 + 1];
                                nxt[p][q][r + 1] += v * H[x * 3 + 2];
                            }
                        std::memcpy(poly, nxt, sizeof(poly));
                        deg++;
                    }
                for (int p = d; p >= 0; p--)
                    for (int q = d - p; q >= 0; q--)
                        blk[graded_idx(p, q, d) * nd + col] = poly[p][q][d - p - q];
            }
    }
}

// T6: does block (b1, b2, b3) (unbounded block indices on a mesh N) hold a grid point within R of P?  The centre of the
// block decides when the answer is clear of the block's circumradius rc by a margin; otherwise its 64 points are tried,
// r_n = (n1/N1) a1 + (n2/N2) a2 + (n3/N3) a3 (PAPER.md:483 with u0 = 0).  The expressions are those of plan_device.cu's
// block_hit, term by term (that file is compiled without FMA contraction), so that both builders decide alike.
bool sphere_meets_block(const double *cell, const int *N, const double *P, double R, double R2, double rc, int b1, int b2, int b3) {
    auto point = [&](double u1, double u2, double u3, double *r) {
        for (int x = 0; x < 3; x++) r[x] = u1 * cell[0 * 3 + x] + u2 * cell[1 * 3 + x] + u3 * cell[2 * 3 + x];
    };
    double c[3];
    point((4 * b1 + 1.5) / N[0], (4 * b2 + 1.5) / N[1], (4 * b3 + 1.5) / N[2], c);
    double dc = 0;
    for (int x = 0; x < 3; x++) dc += (c[x] - P[x]) * (c[x] - P[x]);
    dc = std::sqrt(dc);
    if (dc - rc > R * (1.0 + 1e-9) + 1e-9) return false;
    if (dc + rc < R * (1.0 - 1e-9) - 1e-9) return true;
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++)
            for (int k = 0; k < 4; k++) {
                double r[3];
                point((double)(4 * b1 + i) / N[0], (double)(4 * b2 + j) / N[1], (double)(4 * b3 + k) / N[2], r);
                const double d2 = (r[0] - P[0]) * (r[0] - P[0]) + (r[1] - P[1]) * (r[1] - P[1]) + (r[2] - P[2]) * (r[2] - P[2]);
                if (d2 <= R2) return true;
            }
    return false;
}

struct RawEntry {
    long long key;  // global brick id (level-major)
    int task;
    signed char s[3];
    unsigned char L;
    unsigned mask;
};

struct RawVisit {
    long long key;  // global block id (level-major)
    int task;
    signed char s[3];
    unsigned char L;
};

template <class F>
void parallel_chunks(long n, long chunk, int nthread, F &&fn) {
    std::atomic<long> next(0);
    auto worker = [&](int tid) {
        for (;;) {
            const long c = next.fetch_add(1);
            const long lo = c * chunk;
            if (lo >= n) break;
            fn(c, lo, std::min(n, lo + chunk), tid);
        }
    };
    std::vector<std::thread> th;
    for (int t = 1; t < nthread; t++) th.emplace_back(worker, t);
    worker(0);
    for (auto &t : th) t.join();
}

}  // namespace

int build_host_plan(const double *cell, int natm, const double *xyz, int nshl, const int *shl_atom,
                    const int *shl_l, const int *shl_nprim, const int *shl_prim_off,
                    const double *prim_exp, const double *prim_coef, int nlevel, const int *mesh,
                    double tau, double rel_cutoff, int hermi, bool on_host, HostPlan **out) {
    const auto t_start = std::chrono::steady_clock::now();
    if (!cell || !xyz || !shl_atom || !shl_l || !shl_nprim || !shl_prim_off || !prim_exp || !prim_coef ||
        !mesh || !out) { set_error("gpw_build_pairs: null pointer argument"); return GPW_EINVAL; }
    if (natm < 1 || nshl < 1) { set_error("gpw_build_pairs: natm and nshl must be >= 1"); return GPW_EINVAL; }
    if (nlevel < 1 || nlevel > GPW_MAX_LEVEL) { set_error("gpw_build_pairs: nlevel must be in 1..8"); return GPW_EINVAL; }
    if (!(tau > 0.0) || !(rel_cutoff > 0.0)) { set_error("gpw_build_pairs: tau and rel_cutoff must be > 0"); return GPW_EINVAL; }
    if (hermi != 0 && hermi != 1) { set_error("gpw_build_pairs: hermi must be 0 or 1"); return GPW_EINVAL; }
    for (int i = 0; i < 3 * nlevel; i++)
        if (mesh[i] < 4 || mesh[i] % 4) { set_error("gpw_build_pairs: every mesh entry must be a positive multiple of 4"); return GPW_EINVAL; }
    for (int i = 3; i < 3 * nlevel; i++)
        if (mesh[i] > mesh[i % 3]) { set_error("gpw_build_pairs: level 0 must be the finest mesh on every axis (gpw_interp_up / gpw_restrict_down embed every level's spectrum in level 0's)"); return GPW_EINVAL; }
    int nprim = 0;
    for (int s = 0; s < nshl; s++) {
        if (shl_l[s] < 0) { set_error("gpw_build_pairs: negative angular momentum"); return GPW_EINVAL; }
        if (shl_l[s] > MAXL) { set_error("gpw_build_pairs: shells beyond f (l >= 4) are not supported"); return GPW_EUNSUPPORTED; }
        if (shl_atom[s] < 0 || shl_atom[s] >= natm) { set_error("gpw_build_pairs: shl_atom out of range"); return GPW_EINVAL; }
        if (shl_nprim[s] < 1 || shl_prim_off[s] < 0) { set_error("gpw_build_pairs: shl_nprim must be >= 1 and offsets >= 0"); return GPW_EINVAL; }
        nprim = std::max(nprim, shl_prim_off[s] + shl_nprim[s]);
    }
    for (int s = 0; s < nshl; s++)
        for (int k = 0; k < shl_nprim[s]; k++)
            if (!(prim_exp[shl_prim_off[s] + k] > 0.0)) { set_error("gpw_build_pairs: primitive exponents must be > 0"); return GPW_EINVAL; }

    HostPlan *hp = new (std::nothrow) HostPlan();
    if (!hp) { set_error("out of host memory"); return GPW_ENOMEM; }
    try {
        std::memcpy(hp->cell, cell, sizeof(double) * 9);
        double det;
        if (!reciprocal_vectors(cell, hp->binv, &det)) { delete hp; set_error("gpw_build_pairs: singular cell (|det| < 1e-12)"); return GPW_EINVAL; }
        hp->omega = std::fabs(det);
        // binv[c*3+i] = component c of b_i, so that u_i = sum_c r_c binv[c*3+i]
        for (int i = 0; i < 3; i++)
            hp->bnorm[i] = std::sqrt(hp->binv[0 * 3 + i] * hp->binv[0 * 3 + i] + hp->binv[1 * 3 + i] * hp->binv[1 * 3 + i] +
                                     hp->binv[2 * 3 + i] * hp->binv[2 * 3 + i]);
        hp->natm = natm; hp->nshl = nshl; hp->nprim = nprim; hp->nlevel = nlevel; hp->hermi = hermi;
        hp->tau = tau; hp->rel_cutoff = rel_cutoff;
        hp->ao_loc.resize(nshl + 1);
        hp->ao_loc[0] = 0;
        for (int s = 0; s < nshl; s++) hp->ao_loc[s + 1] = hp->ao_loc[s] + ncart(shl_l[s]);
        hp->nao = hp->ao_loc[nshl];

        // ---- level geometry (T5: E_alpha = 0.5 min_i (pi N_i |b_i|)^2) ----
        hp->lev.resize(nlevel);
        hp->S.resize(nlevel);
        for (int a = 0; a < nlevel; a++) {
            LevelGeom &g = hp->lev[a];
            std::memset(&g, 0, sizeof(g));
            double e = 1e300;
            for (int i = 0; i < 3; i++) {
                g.N[i] = mesh[a * 3 + i];
                g.T[i] = g.N[i] / TILE;
                const double gg = M_PI * g.N[i] * hp->bnorm[i];
                e = std::min(e, 0.5 * gg * gg);
            }
            g.ecut = e;
            g.ntile = g.T[0] * g.T[1] * g.T[2];
            const int BR[3] = {BR1, BR2, BR3};
            for (int i = 0; i < 3; i++) g.B[i] = (g.T[i] + BR[i] - 1) / BR[i];
            g.nbrick = g.B[0] * g.B[1] * g.B[2];
            g.dV = hp->omega / ((double)g.N[0] * g.N[1] * g.N[2]);
            for (int c = 0; c < 3; c++)
                for (int i = 0; i < 3; i++) {
                    g.H[c * 3 + i] = cell[i * 3 + c] / g.N[i];
                    g.Hinv[i * 3 + c] = hp->binv[c * 3 + i] * g.N[i];
                }
            const int pr[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
            for (int k = 0; k < 6; k++) {
                double s = 0;
                for (int c = 0; c < 3; c++) s += g.H[c * 3 + pr[k][0]] * g.H[c * 3 + pr[k][1]];
                g.Gm[k] = s;
            }
            build_S(g.H, hp->S[a]);
        }
        // orthogonal lattice vectors (exact zeros, e.g. a diagonal cell matrix): the kernels' ORTHO variants
        hp->ortho = true;
        for (int a = 0; a < nlevel; a++)
            for (int k = 3; k < 6; k++)
                if (hp->lev[a].Gm[k] != 0.0) hp->ortho = false;
        hp->hdiag = true;
        for (int i = 0; i < 9; i++)
            if (i % 4 != 0 && cell[i] != 0.0) hp->hdiag = false;
        for (int s = 0; s < nshl; s++) hp->max_l = std::max(hp->max_l, shl_l[s]);

        // circumradius of a block about its centre (points at +-1.5 steps per axis)
        for (int a = 0; a < nlevel; a++) {
            double m = 0;
            for (int sg = 0; sg < 4; sg++) {
                double v[3];
                for (int x = 0; x < 3; x++)
                    v[x] = 1.5 * (hp->lev[a].H[x * 3 + 0] + ((sg & 1) ? -1 : 1) * hp->lev[a].H[x * 3 + 1] + ((sg & 2) ? -1 : 1) * hp->lev[a].H[x * 3 + 2]);
                m = std::max(m, std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
            }
            hp->circ[a] = m;
        }
        // ---- T1 radii ----
        std::vector<double> prad(nprim, 0.0);
        std::vector<int> prim_shl(nprim, -1);
        for (int s = 0; s < nshl; s++)
            for (int k = 0; k < shl_nprim[s]; k++) {
                const int p = shl_prim_off[s] + k;
                prad[p] = prim_radius(shl_l[s], prim_exp[p], prim_coef[p], tau);
                prim_shl[p] = s;
            }
        // the primitives as the device pair screen reads them (pairs_device.cu)
        hp->prims.resize(nprim);
        for (int p = 0; p < nprim; p++) {
            DevPrim &d = hp->prims[p];
            std::memset(&d, 0, sizeof(d));
            const int s = prim_shl[p];
            if (s < 0) continue;   // a gap in the primitive table: radius 0, never paired
            for (int x = 0; x < 3; x++) d.A[x] = xyz[3 * shl_atom[s] + x];
            d.exp = prim_exp[p]; d.coef = prim_coef[p]; d.rad = prad[p];
            d.shl = s; d.l = shl_l[s]; d.ao = hp->ao_loc[s]; d.atom = shl_atom[s];
        }
        if (!on_host) {   // with a device, pairs and lists are built there (pairs_device.cu, plan_device.cu)
            hp->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
            *out = hp;
            return GPW_OK;
        }

        // ---- T2..T5: enumerate pairs (a, b, T), parallel over shell a ----
        int nthread = (int)std::thread::hardware_concurrency();
        if (nthread < 1) nthread = 1;
        if (nthread > 64) nthread = 64;
        std::vector<std::vector<HostTask>> per_shell(nshl);
        std::atomic<int> too_sharp(0);
        // T3-T5 for one candidate image of primitive q next to primitive p; false if the pair is dropped
        auto screen = [&](const DevPrim &p, const DevPrim &q, const int *img, HostTask &t) -> bool {
            double sep2 = 0.0;
            for (int x = 0; x < 3; x++) {
                const double shift = img[0] * cell[0 * 3 + x] + img[1] * cell[1 * 3 + x] + img[2] * cell[2 * 3 + x];
                t.A[x] = p.A[x];
                t.Bt[x] = q.A[x] + shift;
                sep2 += (t.A[x] - t.Bt[x]) * (t.A[x] - t.Bt[x]);
            }
            if (!(std::sqrt(sep2) < p.rad + q.rad)) return false;                       // T2
            t.ap = p.exp + q.exp;                                                       // T3
            double dA = 0.0, dB = 0.0;
            for (int x = 0; x < 3; x++) {
                t.P[x] = (p.exp * t.A[x] + q.exp * t.Bt[x]) / t.ap;
                dA += (t.P[x] - t.A[x]) * (t.P[x] - t.A[x]);
                dB += (t.P[x] - t.Bt[x]) * (t.P[x] - t.Bt[x]);
            }
            const double gauss = std::exp(-(p.exp * q.exp / t.ap) * sep2);
            t.pref = p.coef * q.coef * gauss;
            t.R = pair_radius(p.l, q.l, t.ap, std::fabs(p.coef * q.coef) * gauss, std::sqrt(dA), std::sqrt(dB), tau);   // T4
            if (t.R <= 0.0) return false;
            t.level = 0;                                                                // T5
            for (int a = nlevel - 1; a >= 0; a--)
                if (hp->lev[a].ecut >= rel_cutoff * t.ap) { t.level = a; break; }
            // The kernels anchor the Gaussian recursion (Eq. 24-25) at the corner of a visited block: its value there,
            // exp(-a_p d^2) with d up to R + one block diagonal, must not underflow.
            const double reach = t.R + 2.0 * hp->circ[t.level];
            if (t.ap * reach * reach > 600.0) { too_sharp = 1; return false; }
            return true;
        };
        parallel_chunks(nshl, 1, nthread, [&](long, long lo, long hi, int) {
            for (long sa = lo; sa < hi; sa++)
                for (int sb = 0; sb < nshl; sb++)
                    for (int ka = 0; ka < shl_nprim[sa]; ka++)
                        for (int kb = 0; kb < shl_nprim[sb]; kb++) {
                            const int pa = shl_prim_off[sa] + ka, pb = shl_prim_off[sb] + kb;
                            if (hermi && pa < pb) continue;   // canonical unordered set (A14)
                            const DevPrim &p = hp->prims[pa], &q = hp->prims[pb];
                            if (p.rad <= 0.0 || q.rad <= 0.0) continue;
                            // T2: the lattice vectors that can bring q within r_p + r_q of p, |f_i - t_i| <= (r_p + r_q) |b_i|
                            int first[3], last[3];
                            for (int i = 0; i < 3; i++) {
                                const double f = (p.A[0] - q.A[0]) * hp->binv[0 * 3 + i] + (p.A[1] - q.A[1]) * hp->binv[1 * 3 + i] +
                                                 (p.A[2] - q.A[2]) * hp->binv[2 * 3 + i];
                                const double w = (p.rad + q.rad) * hp->bnorm[i];
                                first[i] = (int)std::ceil(f - w);
                                last[i] = (int)std::floor(f + w);
                            }
                            int img[3];
                            for (img[0] = first[0]; img[0] <= last[0]; img[0]++)
                                for (img[1] = first[1]; img[1] <= last[1]; img[1]++)
                                    for (img[2] = first[2]; img[2] <= last[2]; img[2]++) {
                                        const bool zero = img[0] == 0 && img[1] == 0 && img[2] == 0;
                                        const bool negative = img[0] < 0 || (img[0] == 0 && (img[1] < 0 || (img[1] == 0 && img[2] < 0)));
                                        if (hermi && pa == pb && negative) continue;   // of (T, -T) keep the lexicographically positive one
                                        HostTask t;
                                        if (!screen(p, q, img, t)) continue;
                                        t.shl_a = (int)sa; t.prim_a = pa; t.shl_b = sb; t.prim_b = pb;
                                        t.T[0] = img[0]; t.T[1] = img[1]; t.T[2] = img[2];
                                        t.la = p.l; t.lb = q.l;
                                        t.sym = (hermi && !(pa == pb && zero)) ? 1 : 0;
                                        per_shell[sa].push_back(t);
                                    }
                        }
        });
        if (too_sharp) {
            delete hp;
            set_error("gpw_build_pairs: a primitive pair is far too sharp for the finest mesh (a_p (R_t + block diagonal)^2 > 600: "
                      "the Gaussian underflows at the corner of its own grid blocks); use a finer level 0");
            return GPW_EUNSUPPORTED;
        }
        size_t nt = 0;
        for (auto &v : per_shell) nt += v.size();
        if (nt > 2000000000ull) { delete hp; set_error("gpw_build_pairs: more than 2^31 pairs"); return GPW_EUNSUPPORTED; }
        // counting sort by class (level, L, la), keeping enumeration order inside a class: per shell the number of
        // its pairs in every class, prefix sums over (class, shell), then every shell scatters its own pairs.
        // (The kernels need (level, L); la inside keeps the lanes of the pre/post-pass on the same loop bounds.)
        constexpr int NCLS = GPW_MAX_LEVEL * 8 * 4;
        auto cls_of = [](const HostTask &t) { return (t.level * 8 + t.la + t.lb) * 4 + t.la; };
        std::vector<long> start((size_t)nshl * NCLS, 0);
        parallel_chunks(nshl, 16, nthread, [&](long, long lo, long hi, int) {
            for (long sa = lo; sa < hi; sa++)
                for (const HostTask &t : per_shell[sa]) start[(size_t)sa * NCLS + cls_of(t)]++;
        });
        long cls_first[NCLS + 1];
        {
            long run = 0;
            for (int c = 0; c < NCLS; c++) {
                cls_first[c] = run;
                for (long sa = 0; sa < nshl; sa++) {
                    const long n = start[(size_t)sa * NCLS + c];
                    start[(size_t)sa * NCLS + c] = run;
                    run += n;
                }
            }
            cls_first[NCLS] = run;
        }
        hp->task.resize(nt);
        parallel_chunks(nshl, 16, nthread, [&](long, long lo, long hi, int) {
            for (long sa = lo; sa < hi; sa++) {
                long *pos = &start[(size_t)sa * NCLS];
                for (const HostTask &t : per_shell[sa]) hp->task[(size_t)pos[cls_of(t)]++] = t;
                std::vector<HostTask>().swap(per_shell[sa]);
            }
        });
        const long ntask = (long)hp->task.size();
        hp->ntask = ntask;
        hp->taskK.resize(ntask); hp->taskP.resize(ntask);
        // inside a class (level, L) the workspace offset is affine in the pair index: coef_base + i * ncoef_pad(L + off)
        long long coff[NOFF] = {0};
        for (int c = 0; c < NCLS; c += 4) {
            const long n = cls_first[c + 4] - cls_first[c];
            const int level = c / 32, L = (c / 4) % 8;
            if (n == 0 || L > MAXLP) continue;
            for (int off = 0; off < NOFF; off++) {
                hp->coef_base[off][level][L] = coff[off] - (long long)cls_first[c] * ncoef_pad(L + off);
                coff[off] += (long long)n * ncoef_pad(L + off);
            }
            hp->ntask_level[level] += n;
            hp->max_L = std::max(hp->max_L, L);
        }
        parallel_chunks(ntask, 4096, nthread, [&](long, long lo, long hi, int) {
            for (long i = lo; i < hi; i++) {
                const HostTask &t = hp->task[i];
                const LevelGeom &g = hp->lev[t.level];
                const int L = t.la + t.lb;
                const long long off = hp->coef_base[0][t.level][L] + (long long)i * ncoef_pad(L);
                TaskK &k = hp->taskK[i];
                for (int a = 0; a < 3; a++)
                    k.nP[a] = (t.P[0] * hp->binv[0 * 3 + a] + t.P[1] * hp->binv[1 * 3 + a] + t.P[2] * hp->binv[2 * 3 + a]) * g.N[a];
                k.ap = t.ap;
                k.c22 = std::exp(-2.0 * t.ap * g.Gm[1]);
                k.c23 = std::exp(-2.0 * t.ap * g.Gm[5]);
                k.c33 = std::exp(-2.0 * t.ap * g.Gm[2]);
                k.coef_off = off;
                TaskP &p = hp->taskP[i];
                for (int x = 0; x < 3; x++) { p.PA[x] = t.P[x] - t.A[x]; p.PB[x] = t.P[x] - t.Bt[x]; }
                p.pref = t.pref;
                p.aa = prim_exp[t.prim_a]; p.ab = prim_exp[t.prim_b];
                p.ao_a = hp->ao_loc[t.shl_a]; p.ao_b = hp->ao_loc[t.shl_b];
                p.atom_a = shl_atom[t.shl_a]; p.atom_b = shl_atom[t.shl_b];
                p.la = (short)t.la; p.lb = (short)t.lb; p.level = (short)t.level; p.sym = (short)t.sym;
            }
        });
        for (int off = 0; off < NOFF; off++) hp->ncoef_total[off] = coff[off];
        for (int a = 0; a < nlevel; a++) { hp->big_lo[a] = cls_first[(a * 8 + 5) * 4]; hp->big_hi[a] = cls_first[(a * 8 + 7) * 4]; }
        // ---- T6: blocks of every pair ----
        std::vector<long long> lev_tile0(nlevel + 1, 0);
        for (int a = 0; a < nlevel; a++) lev_tile0[a + 1] = lev_tile0[a] + hp->lev[a].ntile;
        const long long ntile_all = lev_tile0[nlevel];
        std::vector<long long> lev_brick0(nlevel + 1, 0);
        for (int a = 0; a < nlevel; a++) lev_brick0[a + 1] = lev_brick0[a] + hp->lev[a].nbrick;
        const long long nbrick_all = lev_brick0[nlevel];
        const double *circ = hp->circ;
        const long chunk = 256;
        const long nchunk = (ntask + chunk - 1) / chunk;
        std::vector<std::vector<RawVisit>> raw(nchunk);
        std::vector<std::vector<RawEntry>> rawb(nchunk);
        std::atomic<int> wrap_overflow(0);
        parallel_chunks(ntask, chunk, nthread, [&](long c, long lo, long hi, int) {
            std::vector<RawVisit> &rv = raw[c];
            std::vector<RawEntry> &rb = rawb[c];
            for (long ti = lo; ti < hi; ti++) {
                const size_t rb0 = rb.size();   // this pair's entries start here
                const HostTask &t = hp->task[ti];
                const LevelGeom &g = hp->lev[t.level];
                const int *N = g.N;
                int blo[3], bhi[3];
                for (int i = 0; i < 3; i++) {
                    const double u = t.P[0] * hp->binv[0 * 3 + i] + t.P[1] * hp->binv[1 * 3 + i] + t.P[2] * hp->binv[2 * 3 + i];
                    const double w = t.R * hp->bnorm[i] * N[i];
                    blo[i] = block_of((int)std::ceil(u * N[i] - w));
                    bhi[i] = block_of((int)std::floor(u * N[i] + w));
                }
                const double R2 = t.R * t.R;
                const double rc = circ[t.level];
                for (int b1 = blo[0]; b1 <= bhi[0]; b1++)
                    for (int b2 = blo[1]; b2 <= bhi[1]; b2++)
                        for (int b3 = blo[2]; b3 <= bhi[2]; b3++) {
                            if (!sphere_meets_block(cell, N, t.P, t.R, R2, rc, b1, b2, b3)) continue;
                            const Folded f1 = fold(b1, g.T[0]), f2 = fold(b2, g.T[1]), f3 = fold(b3, g.T[2]);
                            const int w1 = f1.stored, w2 = f2.stored, w3 = f3.stored;
                            const int s1 = f1.wraps, s2 = f2.wraps, s3 = f3.wraps;
                            if (s1 < -127 || s1 > 127 || s2 < -127 || s2 > 127 || s3 < -127 || s3 > 127) { wrap_overflow = 1; continue; }
                            RawVisit v;
                            v.key = lev_tile0[t.level] + ((long long)w1 * g.T[1] + w2) * g.T[2] + w3;
                            v.task = (int)ti;
                            v.s[0] = (signed char)s1; v.s[1] = (signed char)s2; v.s[2] = (signed char)s3;
                            v.L = (unsigned char)(t.la + t.lb);
                            rv.push_back(v);
                            // the same visit in the brick lists of the integration kernel
                            const long long bkey = lev_brick0[t.level] +
                                ((long long)(w1 / BR1) * g.B[1] + (w2 / BR2)) * g.B[2] + (w3 / BR3);
                            const unsigned bit = 1u << ((w2 % BR2) * BR3 + (w3 % BR3));
                            size_t e = rb0;
                            for (; e < rb.size(); e++)
                                if (rb[e].key == bkey && rb[e].s[0] == v.s[0] && rb[e].s[1] == v.s[1] && rb[e].s[2] == v.s[2]) break;
                            if (e == rb.size()) {
                                RawEntry ne;
                                ne.key = bkey; ne.task = (int)ti; ne.L = v.L; ne.mask = 0;
                                ne.s[0] = v.s[0]; ne.s[1] = v.s[1]; ne.s[2] = v.s[2];
                                rb.push_back(ne);
                            }
                            rb[e].mask |= bit;
                        }
            }
        });
        if (wrap_overflow) { delete hp; set_error("gpw_build_pairs: a pair wraps the cell more than 127 times"); return GPW_EUNSUPPORTED; }

        // counting sort by block; chunks are in pair order, pairs are in (level, L) order, so every
        // block's list comes out sorted by L
        std::vector<long long> cnt(ntile_all + 1, 0);
        std::vector<unsigned> segcnt((size_t)ntile_all * 8, 0);
        long long nvis = 0;
        for (auto &rv : raw) {
            nvis += (long long)rv.size();
            for (const RawVisit &v : rv) { cnt[v.key + 1]++; segcnt[(size_t)v.key * 8 + v.L]++; }
        }
        for (long long i = 0; i < ntile_all; i++) cnt[i + 1] += cnt[i];
        hp->visit.resize((size_t)nvis);
        {
            std::vector<long long> cur(cnt.begin(), cnt.end() - 1);
            for (auto &rv : raw) {
                for (const RawVisit &v : rv) {
                    Visit &o = hp->visit[(size_t)cur[v.key]++];
                    o.task = v.task; o.s[0] = v.s[0]; o.s[1] = v.s[1]; o.s[2] = v.s[2]; o.pad = 0;
                    const HostTask &t = hp->task[v.task];
                    hp->nvisit_level[t.level]++;
                    hp->nvisit_class[t.level][t.la][t.lb]++;
                }
                std::vector<RawVisit>().swap(rv);
            }
        }
        hp->tile_base.resize(nlevel);
        hp->seg.resize(nlevel);
        for (int a = 0; a < nlevel; a++) {
            const int ntl = hp->lev[a].ntile;
            hp->tile_base[a].assign(cnt.begin() + lev_tile0[a], cnt.begin() + lev_tile0[a] + ntl + 1);
            hp->seg[a].resize((size_t)ntl * 8);
            for (int tl = 0; tl < ntl; tl++) {
                unsigned acc = 0;
                for (int L = 0; L < 8; L++) {
                    hp->seg[a][(size_t)tl * 8 + L] = acc;
                    acc += segcnt[(size_t)(lev_tile0[a] + tl) * 8 + L];
                }
            }
        }
        // ---- brick lists of the integration kernel (counting sort by brick, pair order kept) ----
        {
            std::vector<long long> bcnt(nbrick_all + 1, 0);
            long long nent = 0;
            for (auto &rb : rawb) {
                nent += (long long)rb.size();
                for (const RawEntry &e : rb) bcnt[e.key + 1]++;
            }
            for (long long i = 0; i < nbrick_all; i++) bcnt[i + 1] += bcnt[i];
            hp->bentry.resize((size_t)nent);
            std::vector<long long> cur(bcnt.begin(), bcnt.end() - 1);
            for (auto &rb : rawb) {
                for (const RawEntry &e : rb) {
                    BEntry &o = hp->bentry[(size_t)cur[e.key]++];
                    o.task = e.task; o.s[0] = e.s[0]; o.s[1] = e.s[1]; o.s[2] = e.s[2]; o.L = e.L; o.mask = e.mask; o.pad = 0;
                }
                std::vector<RawEntry>().swap(rb);
            }
            hp->brick_base.resize(nlevel);
            for (int a = 0; a < nlevel; a++)
                hp->brick_base[a].assign(bcnt.begin() + lev_brick0[a], bcnt.begin() + lev_brick0[a] + hp->lev[a].nbrick + 1);
            // inside a brick: by L (the kernel's code path), then by decreasing number of visited blocks so
            // that the eight lane groups of a warp, which take consecutive entries, finish together
            parallel_chunks(nbrick_all, 64, nthread, [&](long, long lo, long hi, int) {
                for (long b = lo; b < hi; b++)
                    std::stable_sort(hp->bentry.begin() + bcnt[b], hp->bentry.begin() + bcnt[b + 1],
                                     [](const BEntry &x, const BEntry &y) {
                                         if (x.L != y.L) return x.L < y.L;
                                         return __builtin_popcount(x.mask) > __builtin_popcount(y.mask);
                                     });
            });
            const unsigned BITEM_MAX = 768;
            std::vector<std::pair<long long, BItem>> tmp;
            for (int a = 0; a < nlevel; a++) {
                const int nb = hp->lev[a].nbrick;
                for (int b = 0; b < nb; b++) {
                    const long long base = hp->brick_base[a][b];
                    const unsigned n = (unsigned)(hp->brick_base[a][b + 1] - base);
                    if (!n) continue;
                    BItem proto;
                    std::memset(&proto, 0, sizeof(proto));
                    proto.level = a; proto.brick = b; proto.base = base;
                    {
                        unsigned cntL[8] = {0};
                        for (unsigned e = 0; e < n; e++) cntL[hp->bentry[(size_t)(base + e)].L]++;
                        unsigned acc = 0;
                        for (int L = 0; L < 8; L++) { proto.seg[L] = acc; acc += cntL[L]; }
                    }
                    const unsigned nparts = (n + BITEM_MAX - 1) / BITEM_MAX;
                    for (unsigned p = 0; p < nparts; p++) {
                        BItem it = proto;
                        it.lo = (unsigned)((unsigned long long)n * p / nparts);
                        it.hi = (unsigned)((unsigned long long)n * (p + 1) / nparts);
                        long long work = 0;
                        for (unsigned e = it.lo; e < it.hi; e++) {
                            const BEntry &be = hp->bentry[(size_t)(base + e)];
                            work += (long long)__builtin_popcount(be.mask) * (4 + be.L);
                        }
                        tmp.emplace_back(work, it);
                    }
                }
            }
            std::stable_sort(tmp.begin(), tmp.end(), [](const std::pair<long long, BItem> &x, const std::pair<long long, BItem> &y) { return x.first > y.first; });
            hp->bitem.reserve(tmp.size());
            for (auto &x : tmp) hp->bitem.push_back(x.second);
        }
        // ---- work items: every block's list cut into ranges of at most ITEM_MAX visits ----
        const unsigned ITEM_MAX = 384;
        for (int a = 0; a < nlevel; a++) {
            const int ntl = hp->lev[a].ntile;
            for (int tl = 0; tl < ntl; tl++) {
                const unsigned n = (unsigned)(hp->tile_base[a][tl + 1] - hp->tile_base[a][tl]);
                if (!n) continue;
                const unsigned nparts = (n + ITEM_MAX - 1) / ITEM_MAX;
                for (unsigned p = 0; p < nparts; p++) {
                    Item it;
                    it.level = a; it.tile = tl;
                    it.lo = (unsigned)((unsigned long long)n * p / nparts);
                    it.hi = (unsigned)((unsigned long long)n * (p + 1) / nparts);
                    it.single = nparts == 1; it.pad = 0;
                    it.vstart = hp->tile_base[a][tl] + it.lo;
                    hp->item.push_back(it);
                }
            }
        }
        std::stable_sort(hp->item.begin(), hp->item.end(),
                         [](const Item &x, const Item &y) { return (x.hi - x.lo) > (y.hi - y.lo); });
        hp->nitem = (long)hp->item.size();
        hp->nbitem = (long)hp->bitem.size();
        hp->nvisit_total = (long long)hp->visit.size();
    } catch (const std::bad_alloc &) {
        delete hp;
        set_error("gpw_build_pairs: out of host memory");
        return GPW_ENOMEM;
    }
    hp->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    *out = hp;
    return GPW_OK;
}

}  // namespace gpw
