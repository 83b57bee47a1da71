/*
 * gpw_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct evaluation of what the multigrid
 * Gaussian-Plane-Wave hot path computes, written from the paper only
 * (arxiv 2603.24881, text in /root/reference/PAPER.md) plus the readings
 * listed in DESIGN.md ("Readings of the paper").  It shares no code with the
 * CUDA path under paper_2603_24881_b200/csrc and is imported only by tests/,
 * __graft_entry__.smoke() and the cpu_baseline / --impl reference legs of
 * bench.py.
 *
 * What it computes (the TRUNCATED definition, T1..T8):
 *   T1  primitive cutoff radius          PAPER.md:134-138  Eq. (20)
 *   T2  pair enumeration, single lattice sum + folding      PAPER.md:123-132  Eq. (18)-(19)
 *   T3  Gaussian product centre P and exponent a_p          PAPER.md:153-155  Eq. (23)
 *   T4  pair radius "determined through Eq. (20) for each Gaussian pair"
 *   T5  level assignment by pair exponent
 *   T6  4x4x4 grid blocks ("tiles") of a pair
 *   T7  rho(r) += sum D_ij phi_i(r) phi_j(r-T)              PAPER.md:41   Eq. (3)
 *       F_ij   += dV v(r) phi_i(r) phi_j(r-T)               PAPER.md:45   Eq. (4), dV from Eq. (29)
 *   T8  deriv=1: exact real-space gradient of Eq. (3) and Eq. (4)+(11)
 *   T10 deriv=2 (meta-GGA): a fifth component, the kinetic-energy density
 *       tau(r) = 1/2 sum D_ij grad phi_i . grad phi_j                     PAPER.md:100-103  Eq. (15)
 *       F_ij  += dV v_tau(r) 1/2 grad phi_i . grad phi_j                  PAPER.md:105-107  Eq. (16) with the 1/2 of
 *                                                                        PAPER.md:265-268 (reading A25)
 *   T11 nuclear gradient of E = sum_alpha dV sum_r [v0 rho + w . grad rho] at fixed v, w and fixed visit set:
 *       dE/dR_A = dV sum_r sum_ij D_ij [v0 + w . grad_r] d/dR_A (phi_i phi_j)     PAPER.md:272-309  Alg. 3
 *
 * There is no product theorem, no recursion (Eq. 24-25), no factorisation and
 * no blocking in the evaluation: phi_a and phi_b are evaluated separately with
 * a direct exp() at every grid point of every visited tile, in the order the
 * definition states, and summed in long double.
 *
 * Pins (tests/, -m "not gpu"): untruncated brute force over all lattice images
 * (oracle/dense.py), analytic periodic overlap for v = 1 (oracle/overlap.py),
 * electron count Tr(D S), adjointness <rho[D],v> = Tr(D F[v]), the closed form
 * for one s primitive, translation covariance, finite-difference and FFT
 * gradients.  See DESIGN.md "Pins".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXL 3
#define ORC_MAXNC 10 /* (l+1)(l+2)/2 for l = 3 */

typedef struct {
    int shl_a, prim_a, shl_b, prim_b; /* shell index, global primitive index */
    int T[3];                         /* lattice translation of b */
    int level;
    double R;                         /* pair radius (T4) */
    double A[3], Bt[3];               /* centre of a; centre of b shifted by T */
    double P[3];
    double aa, ab, ca, cb;            /* exponents and coefficients */
    int la, lb, ao_a, ao_b;
    /* visits: unwrapped tile coordinates (beta_1,beta_2,beta_3) */
    long nvis;
    int *vis;
} orc_task;

typedef struct {
    double cell[9], binv[9]; /* binv[c*3+i] = component c of b_i: u_i = sum_c r_c binv[c*3+i] */
    double bnorm[3], omega;
    int natm, nshl, nprim, nlevel, nao;
    double *xyz;
    int *shl_atom, *shl_l, *shl_nprim, *shl_prim_off, *ao_loc;
    double *prim_exp, *prim_coef, *prim_rad;
    int *mesh;       /* [nlevel][3] */
    double *ecut;    /* [nlevel] E_alpha of T5 */
    double tau, rel_cutoff;
    long ntask;
    orc_task *task;
    int visits_built; /* 0 = none, 1 = all */
    long last_counts[8 * 16]; /* (ordered pair, tile) visits evaluated by the last eval call, [level][la][lb] */
} orc_ctx;

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- T1: largest root of r^2 |coef| r^l exp(-a r^2) = tau (Eq. 20) -------- */
double orc_prim_radius(int l, double a, double coef, double tau)
{
    double C = log(fabs(coef)) - log(tau);
    double r = sqrt((C > 1.0 ? C : 1.0) / a) + 5.0;
    for (int it = 0; it < 40; it++) {
        double arg = (C + (l + 2) * log(r)) / a;
        if (arg <= 0.0) return 0.0;
        r = sqrt(arg);
    }
    return r;
}

/* ---- T4: largest root of r^2 kappa (r+dA)^la (r+dB)^lb exp(-a_p r^2) = tau - */
double orc_pair_radius(int la, int lb, double ap, double kappa, double dA, double dB, double tau)
{
    double C = log(kappa) - log(tau);
    double r = sqrt((C > 1.0 ? C : 1.0) / ap) + dA + dB + 5.0;
    for (int it = 0; it < 40; it++) {
        double arg = (C + 2.0 * log(r) + la * log(r + dA) + lb * log(r + dB)) / ap;
        if (arg <= 0.0) return 0.0;
        r = sqrt(arg);
    }
    return r;
}

static int invert3(const double *m, double *inv, double *det_out)
{
    double det = m[0] * (m[4] * m[8] - m[5] * m[7]) - m[1] * (m[3] * m[8] - m[5] * m[6]) +
                 m[2] * (m[3] * m[7] - m[4] * m[6]);
    *det_out = det;
    if (fabs(det) < 1e-12) return -1;
    inv[0] = (m[4] * m[8] - m[5] * m[7]) / det;
    inv[1] = (m[2] * m[7] - m[1] * m[8]) / det;
    inv[2] = (m[1] * m[5] - m[2] * m[4]) / det;
    inv[3] = (m[5] * m[6] - m[3] * m[8]) / det;
    inv[4] = (m[0] * m[8] - m[2] * m[6]) / det;
    inv[5] = (m[2] * m[3] - m[0] * m[5]) / det;
    inv[6] = (m[3] * m[7] - m[4] * m[6]) / det;
    inv[7] = (m[1] * m[6] - m[0] * m[7]) / det;
    inv[8] = (m[0] * m[4] - m[1] * m[3]) / det;
    return 0;
}

static int floordiv(int n, int d) { return n >= 0 ? n / d : -((-n + d - 1) / d); }
static int posmod(int n, int d) { int m = n % d; return m < 0 ? m + d : m; }

void orc_free(orc_ctx *c)
{
    if (!c) return;
    if (c->task) {
        for (long t = 0; t < c->ntask; t++) free(c->task[t].vis);
        free(c->task);
    }
    free(c->xyz); free(c->shl_atom); free(c->shl_l); free(c->shl_nprim); free(c->shl_prim_off);
    free(c->ao_loc); free(c->prim_exp); free(c->prim_coef); free(c->prim_rad); free(c->mesh);
    free(c->ecut);
    free(c);
}

static void *dupmem(const void *p, size_t n)
{
    void *q = malloc(n ? n : 1);
    memcpy(q, p, n);
    return q;
}

/* T2..T5: enumerate ORDERED primitive pairs (a, b, T). */
orc_ctx *orc_create(const double *cell, int natm, const double *xyz, int nshl, const int *shl_atom,
                    const int *shl_l, const int *shl_nprim, const int *shl_prim_off,
                    const double *prim_exp, const double *prim_coef, int nlevel, const int *mesh,
                    double tau, double rel_cutoff)
{
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    memcpy(c->cell, cell, 9 * sizeof(double));
    double det;
    if (invert3(cell, c->binv, &det)) { free(c); return NULL; }
    c->omega = fabs(det);
    for (int i = 0; i < 3; i++)
        c->bnorm[i] = sqrt(c->binv[0 * 3 + i] * c->binv[0 * 3 + i] + c->binv[1 * 3 + i] * c->binv[1 * 3 + i] +
                           c->binv[2 * 3 + i] * c->binv[2 * 3 + i]);
    c->natm = natm; c->nshl = nshl; c->nlevel = nlevel; c->tau = tau; c->rel_cutoff = rel_cutoff;
    int nprim = 0;
    for (int s = 0; s < nshl; s++)
        if (shl_prim_off[s] + shl_nprim[s] > nprim) nprim = shl_prim_off[s] + shl_nprim[s];
    c->nprim = nprim;
    c->xyz = (double *)dupmem(xyz, sizeof(double) * 3 * natm);
    c->shl_atom = (int *)dupmem(shl_atom, sizeof(int) * nshl);
    c->shl_l = (int *)dupmem(shl_l, sizeof(int) * nshl);
    c->shl_nprim = (int *)dupmem(shl_nprim, sizeof(int) * nshl);
    c->shl_prim_off = (int *)dupmem(shl_prim_off, sizeof(int) * nshl);
    c->prim_exp = (double *)dupmem(prim_exp, sizeof(double) * nprim);
    c->prim_coef = (double *)dupmem(prim_coef, sizeof(double) * nprim);
    c->mesh = (int *)dupmem(mesh, sizeof(int) * 3 * nlevel);
    c->ao_loc = (int *)malloc(sizeof(int) * (nshl + 1));
    c->ao_loc[0] = 0;
    for (int s = 0; s < nshl; s++) c->ao_loc[s + 1] = c->ao_loc[s] + ncart(shl_l[s]);
    c->nao = c->ao_loc[nshl];
    /* T1 */
    c->prim_rad = (double *)malloc(sizeof(double) * (nprim ? nprim : 1));
    for (int s = 0; s < nshl; s++)
        for (int k = 0; k < shl_nprim[s]; k++) {
            int p = shl_prim_off[s] + k;
            c->prim_rad[p] = orc_prim_radius(shl_l[s], prim_exp[p], prim_coef[p], tau);
        }
    /* T5: E_alpha = 0.5 min_i (pi N_i |b_i|)^2 */
    c->ecut = (double *)malloc(sizeof(double) * nlevel);
    for (int a = 0; a < nlevel; a++) {
        double e = 1e300;
        for (int i = 0; i < 3; i++) {
            double g = M_PI * mesh[a * 3 + i] * c->bnorm[i];
            if (0.5 * g * g < e) e = 0.5 * g * g;
        }
        c->ecut[a] = e;
    }
    /* T2 */
    long cap = 1024, nt = 0;
    orc_task *tk = (orc_task *)malloc(sizeof(orc_task) * cap);
    for (int sa = 0; sa < nshl; sa++)
        for (int sb = 0; sb < nshl; sb++)
            for (int ka = 0; ka < shl_nprim[sa]; ka++)
                for (int kb = 0; kb < shl_nprim[sb]; kb++) {
                    int pa = shl_prim_off[sa] + ka, pb = shl_prim_off[sb] + kb;
                    double ra = c->prim_rad[pa], rb = c->prim_rad[pb];
                    if (ra <= 0.0 || rb <= 0.0) continue;
                    const double *A = xyz + 3 * shl_atom[sa], *B = xyz + 3 * shl_atom[sb];
                    double rsum = ra + rb;
                    double d[3] = {A[0] - B[0], A[1] - B[1], A[2] - B[2]};
                    int tlo[3], thi[3];
                    for (int i = 0; i < 3; i++) {
                        double f = d[0] * c->binv[0 * 3 + i] + d[1] * c->binv[1 * 3 + i] + d[2] * c->binv[2 * 3 + i];
                        double w = rsum * c->bnorm[i];
                        tlo[i] = (int)ceil(f - w);
                        thi[i] = (int)floor(f + w);
                    }
                    for (int t0 = tlo[0]; t0 <= thi[0]; t0++)
                        for (int t1 = tlo[1]; t1 <= thi[1]; t1++)
                            for (int t2 = tlo[2]; t2 <= thi[2]; t2++) {
                                double Tv[3], Bt[3], dd = 0.0;
                                for (int x = 0; x < 3; x++) {
                                    Tv[x] = t0 * cell[0 * 3 + x] + t1 * cell[1 * 3 + x] + t2 * cell[2 * 3 + x];
                                    Bt[x] = B[x] + Tv[x];
                                    dd += (A[x] - Bt[x]) * (A[x] - Bt[x]);
                                }
                                if (!(sqrt(dd) < rsum)) continue;
                                /* T3 */
                                double aa = prim_exp[pa], ab = prim_exp[pb], ap = aa + ab;
                                double P[3], dA = 0.0, dB = 0.0;
                                for (int x = 0; x < 3; x++) {
                                    P[x] = (aa * A[x] + ab * Bt[x]) / ap;
                                    dA += (P[x] - A[x]) * (P[x] - A[x]);
                                    dB += (P[x] - Bt[x]) * (P[x] - Bt[x]);
                                }
                                dA = sqrt(dA); dB = sqrt(dB);
                                double kappa = fabs(prim_coef[pa] * prim_coef[pb]) * exp(-(aa * ab / ap) * dd);
                                /* T4 */
                                double R = orc_pair_radius(shl_l[sa], shl_l[sb], ap, kappa, dA, dB, tau);
                                if (R <= 0.0) continue;
                                /* T5: coarsest level with E_alpha >= rel_cutoff a_p, else level 0 */
                                int lev = 0;
                                for (int a = nlevel - 1; a >= 0; a--)
                                    if (c->ecut[a] >= rel_cutoff * ap) { lev = a; break; }
                                if (nt == cap) { cap *= 2; tk = (orc_task *)realloc(tk, sizeof(orc_task) * cap); }
                                orc_task *t = tk + nt++;
                                memset(t, 0, sizeof(*t));
                                t->shl_a = sa; t->prim_a = pa; t->shl_b = sb; t->prim_b = pb;
                                t->T[0] = t0; t->T[1] = t1; t->T[2] = t2;
                                t->level = lev; t->R = R;
                                for (int x = 0; x < 3; x++) { t->A[x] = A[x]; t->Bt[x] = Bt[x]; t->P[x] = P[x]; }
                                t->aa = aa; t->ab = ab; t->ca = prim_coef[pa]; t->cb = prim_coef[pb];
                                t->la = shl_l[sa]; t->lb = shl_l[sb];
                                t->ao_a = c->ao_loc[sa]; t->ao_b = c->ao_loc[sb];
                            }
                }
    c->task = tk; c->ntask = nt;
    return c;
}

long orc_ntask(const orc_ctx *c) { return c->ntask; }
int orc_nao(const orc_ctx *c) { return c->nao; }

/* ints: [ntask][8] = shl_a, prim_a, shl_b, prim_b, T0, T1, T2, level; R: [ntask] */
void orc_get_tasks(const orc_ctx *c, int *ints, double *R)
{
    for (long t = 0; t < c->ntask; t++) {
        const orc_task *k = c->task + t;
        int *o = ints + 8 * t;
        o[0] = k->shl_a; o[1] = k->prim_a; o[2] = k->shl_b; o[3] = k->prim_b;
        o[4] = k->T[0]; o[5] = k->T[1]; o[6] = k->T[2]; o[7] = k->level;
        R[t] = k->R;
    }
}

/* position of unwrapped grid index n on a level: r_n = sum_i (n_i/N_i) a_i  (u_0 = 0) */
static void grid_pos(const orc_ctx *c, const int *N, int n1, int n2, int n3, double *r)
{
    double u1 = (double)n1 / N[0], u2 = (double)n2 / N[1], u3 = (double)n3 / N[2];
    for (int x = 0; x < 3; x++) r[x] = u1 * c->cell[0 * 3 + x] + u2 * c->cell[1 * 3 + x] + u3 * c->cell[2 * 3 + x];
}

/* T6: list the tiles of one task.  A tile is visited iff at least one of its 64
 * points lies within R of P.  mask (may be NULL): per stored tile of this level,
 * only tiles with mask != 0 are recorded.  Returns the number of visits; if
 * store != 0 the unwrapped tile coordinates are appended to t->vis. */
static long task_tiles(const orc_ctx *c, orc_task *t, const unsigned char *mask, int store)
{
    const int *N = c->mesh + 3 * t->level;
    int lo[3], hi[3];
    for (int i = 0; i < 3; i++) {
        double u = t->P[0] * c->binv[0 * 3 + i] + t->P[1] * c->binv[1 * 3 + i] + t->P[2] * c->binv[2 * 3 + i];
        double w = t->R * c->bnorm[i] * N[i];
        int nlo = (int)ceil(u * N[i] - w), nhi = (int)floor(u * N[i] + w);
        lo[i] = floordiv(nlo, 4);
        hi[i] = floordiv(nhi, 4);
    }
    int T1 = N[0] / 4, T2 = N[1] / 4, T3 = N[2] / 4;
    long n = 0, cap = 0;
    double R2 = t->R * t->R;
    for (int b1 = lo[0]; b1 <= hi[0]; b1++)
        for (int b2 = lo[1]; b2 <= hi[1]; b2++)
            for (int b3 = lo[2]; b3 <= hi[2]; b3++) {
                if (mask) {
                    long id = ((long)posmod(b1, T1) * T2 + posmod(b2, T2)) * T3 + posmod(b3, T3);
                    if (!mask[id]) continue;
                }
                int hit = 0;
                for (int i = 0; i < 4 && !hit; i++)
                    for (int j = 0; j < 4 && !hit; j++)
                        for (int k = 0; k < 4 && !hit; k++) {
                            double r[3];
                            grid_pos(c, N, 4 * b1 + i, 4 * b2 + j, 4 * b3 + k, r);
                            double d2 = (r[0] - t->P[0]) * (r[0] - t->P[0]) + (r[1] - t->P[1]) * (r[1] - t->P[1]) +
                                        (r[2] - t->P[2]) * (r[2] - t->P[2]);
                            if (d2 <= R2) hit = 1;
                        }
                if (!hit) continue;
                if (store) {
                    if (n == cap) { cap = cap ? 2 * cap : 64; t->vis = (int *)realloc(t->vis, sizeof(int) * 3 * cap); }
                    t->vis[3 * n] = b1; t->vis[3 * n + 1] = b2; t->vis[3 * n + 2] = b3;
                }
                n++;
            }
    if (store) t->nvis = n;
    return n;
}

static void clear_visits(orc_ctx *c)
{
    for (long t = 0; t < c->ntask; t++) { free(c->task[t].vis); c->task[t].vis = NULL; c->task[t].nvis = 0; }
    c->visits_built = 0;
}

/* counts[level][la][lb] (4x4 per level) = number of (ordered task, tile) visits */
void orc_visit_counts(orc_ctx *c, long *counts)
{
    memset(counts, 0, sizeof(long) * c->nlevel * 16);
    long *nv = (long *)malloc(sizeof(long) * (c->ntask ? c->ntask : 1));
#pragma omp parallel for schedule(dynamic, 16)
    for (long t = 0; t < c->ntask; t++) nv[t] = task_tiles(c, c->task + t, NULL, 0);
    for (long t = 0; t < c->ntask; t++)
        counts[c->task[t].level * 16 + c->task[t].la * 4 + c->task[t].lb] += nv[t];
    free(nv);
}

/* Values and Cartesian gradients of every component of one primitive shell at
 * displacement d = r - centre.  Eq. (21)-(22); derivative:
 * d/dx [x^l e^{-a x^2}] = (l x^{l-1} - 2 a x^{l+1}) e^{-a x^2}.
 * out[i][0] = value, out[i][1..3] = d/dx, d/dy, d/dz.
 * Component order: decreasing lx, then decreasing ly (reading A2). */
static void shell_values(int l, double a, double coef, const double *d, int deriv, double out[][4])
{
    double e = coef * exp(-a * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
    double pw[3][ORC_MAXL + 2];
    for (int x = 0; x < 3; x++) {
        pw[x][0] = 1.0;
        for (int k = 1; k <= l + 1; k++) pw[x][k] = pw[x][k - 1] * d[x];
    }
    int i = 0;
    for (int lx = l; lx >= 0; lx--)
        for (int ly = l - lx; ly >= 0; ly--) {
            int lz = l - lx - ly;
            int lc[3] = {lx, ly, lz};
            out[i][0] = pw[0][lx] * pw[1][ly] * pw[2][lz] * e;
            if (deriv) {
                for (int x = 0; x < 3; x++) {
                    double dp = -2.0 * a * pw[x][lc[x] + 1];
                    if (lc[x] > 0) dp += lc[x] * pw[x][lc[x] - 1];
                    double prod = dp;
                    for (int y = 0; y < 3; y++)
                        if (y != x) prod *= pw[y][lc[y]];
                    out[i][1 + x] = prod * e;
                }
            }
            i++;
        }
}

/* Second derivatives of every component of one primitive shell (needed by T11 with deriv = 1):
 * out[i][x][y] = d^2/dx dy [x^lx y^ly z^lz e^{-a r^2}] coef, from the 1-D factors
 *   f0 = t^l,  f1 = l t^(l-1) - 2a t^(l+1),  f2 = l(l-1) t^(l-2) - 2a(2l+1) t^l + 4a^2 t^(l+2)
 * (each times the common Gaussian). */
static void shell_hessian(int l, double a, double coef, const double *d, double out[][3][3])
{
    double e = coef * exp(-a * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
    double pw[3][ORC_MAXL + 3];
    for (int x = 0; x < 3; x++) {
        pw[x][0] = 1.0;
        for (int k = 1; k <= l + 2; k++) pw[x][k] = pw[x][k - 1] * d[x];
    }
    int i = 0;
    for (int lx = l; lx >= 0; lx--)
        for (int ly = l - lx; ly >= 0; ly--) {
            int lz = l - lx - ly;
            int lc[3] = {lx, ly, lz};
            double f0[3], f1[3], f2[3];
            for (int x = 0; x < 3; x++) {
                int n = lc[x];
                f0[x] = pw[x][n];
                f1[x] = -2.0 * a * pw[x][n + 1] + (n > 0 ? n * pw[x][n - 1] : 0.0);
                f2[x] = 4.0 * a * a * pw[x][n + 2] - 2.0 * a * (2 * n + 1) * pw[x][n] + (n > 1 ? n * (n - 1) * pw[x][n - 2] : 0.0);
            }
            for (int x = 0; x < 3; x++)
                for (int y = 0; y < 3; y++) {
                    double prod = 1.0;
                    for (int z = 0; z < 3; z++)
                        prod *= (z == x && z == y) ? f2[z] : ((z == x || z == y) ? f1[z] : f0[z]);
                    out[i][x][y] = prod * e;
                }
            i++;
        }
}

static void build_visits(orc_ctx *c, const unsigned char *const *tile_mask, const unsigned char *pair_mask)
{
    clear_visits(c);
#pragma omp parallel for schedule(dynamic, 16)
    for (long t = 0; t < c->ntask; t++) {
        orc_task *k = c->task + t;
        if (pair_mask && !pair_mask[(long)k->shl_a * c->nshl + k->shl_b]) continue;
        const unsigned char *m = tile_mask ? tile_mask[k->level] : NULL;
        if (tile_mask && !m) continue; /* level not sampled */
        task_tiles(c, k, m, 1);
    }
    c->visits_built = 1;
    memset(c->last_counts, 0, sizeof(c->last_counts));
    for (long t = 0; t < c->ntask; t++)
        c->last_counts[c->task[t].level * 16 + c->task[t].la * 4 + c->task[t].lb] += c->task[t].nvis;
}

/* All (ordered task, tile) visits of T6 as rows (task index, beta_1, beta_2, beta_3) with UNWRAPPED tile
 * coordinates; buf may be NULL (count only).  Returns the number of visits. */
long orc_export_visits(orc_ctx *c, long cap, int *buf)
{
    build_visits(c, NULL, NULL);
    long n = 0;
    for (long t = 0; t < c->ntask; t++)
        for (long v = 0; v < c->task[t].nvis; v++, n++)
            if (buf && n < cap) {
                buf[4 * n] = (int)t;
                buf[4 * n + 1] = c->task[t].vis[3 * v];
                buf[4 * n + 2] = c->task[t].vis[3 * v + 1];
                buf[4 * n + 3] = c->task[t].vis[3 * v + 2];
            }
    clear_visits(c);
    return n;
}

/* bookkeeping only (used to size the timed CPU baseline): visits the last eval call evaluated */
void orc_last_visit_counts(const orc_ctx *c, long *counts)
{
    memcpy(counts, c->last_counts, sizeof(long) * c->nlevel * 16);
}

/* T7/T8 collocation.  D: [nao][nao] row-major.  rho[level]: [ncomp][N1][N2][N3],
 * overwritten.  tile_mask: NULL = everything; else per level a byte per stored
 * tile (NULL entry = skip the level); only marked tiles are evaluated, the rest
 * of the array is left zero. */
int orc_eval_rho(orc_ctx *c, const double *D, int deriv, double *const *rho, const unsigned char *const *tile_mask)
{
    int ncomp = deriv == 0 ? 1 : (deriv == 1 ? 4 : 5);
    build_visits(c, tile_mask, NULL);
    for (int lev = 0; lev < c->nlevel; lev++) {
        const int *N = c->mesh + 3 * lev;
        long ng = (long)N[0] * N[1] * N[2];
        memset(rho[lev], 0, sizeof(double) * ng * ncomp);
        int T1 = N[0] / 4, T2 = N[1] / 4, T3 = N[2] / 4;
        long ntile = (long)T1 * T2 * T3;
        /* CSR: stored tile -> (task, unwrapped tile) */
        long *off = (long *)calloc(ntile + 1, sizeof(long));
        for (long t = 0; t < c->ntask; t++) {
            orc_task *k = c->task + t;
            if (k->level != lev) continue;
            for (long v = 0; v < k->nvis; v++) {
                long id = ((long)posmod(k->vis[3 * v], T1) * T2 + posmod(k->vis[3 * v + 1], T2)) * T3 + posmod(k->vis[3 * v + 2], T3);
                off[id + 1]++;
            }
        }
        for (long i = 0; i < ntile; i++) off[i + 1] += off[i];
        long nv = off[ntile];
        long *vt = (long *)malloc(sizeof(long) * (nv ? nv : 1));
        int *vb = (int *)malloc(sizeof(int) * 3 * (nv ? nv : 1));
        long *cur = (long *)malloc(sizeof(long) * (ntile + 1));
        memcpy(cur, off, sizeof(long) * (ntile + 1));
        for (long t = 0; t < c->ntask; t++) {
            orc_task *k = c->task + t;
            if (k->level != lev) continue;
            for (long v = 0; v < k->nvis; v++) {
                long id = ((long)posmod(k->vis[3 * v], T1) * T2 + posmod(k->vis[3 * v + 1], T2)) * T3 + posmod(k->vis[3 * v + 2], T3);
                long p = cur[id]++;
                vt[p] = t;
                vb[3 * p] = k->vis[3 * v]; vb[3 * p + 1] = k->vis[3 * v + 1]; vb[3 * p + 2] = k->vis[3 * v + 2];
            }
        }
        free(cur);
#pragma omp parallel for schedule(dynamic, 4)
        for (long id = 0; id < ntile; id++) {
            if (off[id + 1] == off[id]) continue;
            long double acc[5][64];
            memset(acc, 0, sizeof(acc));
            for (long p = off[id]; p < off[id + 1]; p++) {
                const orc_task *k = c->task + vt[p];
                int nca = ncart(k->la), ncb = ncart(k->lb);
                double fa[ORC_MAXNC][4], fb[ORC_MAXNC][4];
                for (int i = 0; i < 4; i++)
                    for (int j = 0; j < 4; j++)
                        for (int q = 0; q < 4; q++) {
                            double r[3], da[3], db[3];
                            grid_pos(c, N, 4 * vb[3 * p] + i, 4 * vb[3 * p + 1] + j, 4 * vb[3 * p + 2] + q, r);
                            for (int x = 0; x < 3; x++) { da[x] = r[x] - k->A[x]; db[x] = r[x] - k->Bt[x]; }
                            shell_values(k->la, k->aa, k->ca, da, deriv, fa);
                            shell_values(k->lb, k->ab, k->cb, db, deriv, fb);
                            int pt = (i * 4 + j) * 4 + q;
                            for (int ia = 0; ia < nca; ia++)
                                for (int ib = 0; ib < ncb; ib++) {
                                    double d = D[(long)(k->ao_a + ia) * c->nao + k->ao_b + ib];
                                    acc[0][pt] += (long double)(d * fa[ia][0] * fb[ib][0]);
                                    if (deriv)
                                        for (int x = 1; x < 4; x++)
                                            acc[x][pt] += (long double)(d * (fa[ia][x] * fb[ib][0] + fa[ia][0] * fb[ib][x]));
                                    if (deriv == 2) /* Eq. (15): tau = 1/2 sum D grad phi_a . grad phi_b */
                                        acc[4][pt] += (long double)(0.5 * d * (fa[ia][1] * fb[ib][1] + fa[ia][2] * fb[ib][2] + fa[ia][3] * fb[ib][3]));
                                }
                        }
            }
            int w1 = (int)(id / ((long)T2 * T3)), w2 = (int)((id / T3) % T2), w3 = (int)(id % T3);
            for (int cc = 0; cc < ncomp; cc++)
                for (int i = 0; i < 4; i++)
                    for (int j = 0; j < 4; j++)
                        for (int q = 0; q < 4; q++)
                            rho[lev][cc * ng + ((long)(4 * w1 + i) * N[1] + 4 * w2 + j) * N[2] + 4 * w3 + q] =
                                (double)acc[cc][(i * 4 + j) * 4 + q];
        }
        free(off); free(vt); free(vb);
    }
    clear_visits(c);
    return 0;
}

/* T7/T8 integration.  v[level]: [ncomp][N1][N2][N3].  F: [nao][nao] row-major,
 * overwritten, includes dV = Omega / (N1 N2 N3) (Eq. 29).  pair_mask: NULL or
 * [nshl][nshl] bytes; only marked (shell a, shell b) blocks are computed. */
int orc_eval_mat(orc_ctx *c, const double *const *v, int deriv, double *F, const unsigned char *pair_mask)
{
    build_visits(c, NULL, pair_mask);
    memset(F, 0, sizeof(double) * (size_t)c->nao * c->nao);
    /* tasks were generated with (shell a, shell b) outermost: equal pairs are contiguous */
    long ng_cap = 0;
    (void)ng_cap;
    long *gstart = (long *)malloc(sizeof(long) * (c->ntask + 1));
    long ngroup = 0;
    for (long t = 0; t < c->ntask; t++)
        if (t == 0 || c->task[t].shl_a != c->task[t - 1].shl_a || c->task[t].shl_b != c->task[t - 1].shl_b)
            gstart[ngroup++] = t;
    gstart[ngroup] = c->ntask;
#pragma omp parallel for schedule(dynamic, 1)
    for (long g = 0; g < ngroup; g++) {
        const orc_task *k0 = c->task + gstart[g];
        int nca = ncart(k0->la), ncb = ncart(k0->lb);
        long double acc[ORC_MAXNC][ORC_MAXNC];
        memset(acc, 0, sizeof(acc));
        for (long t = gstart[g]; t < gstart[g + 1]; t++) {
            const orc_task *k = c->task + t;
            const int *N = c->mesh + 3 * k->level;
            long ng = (long)N[0] * N[1] * N[2];
            double dV = c->omega / (double)ng;
            const double *vl = v[k->level];
            double fa[ORC_MAXNC][4], fb[ORC_MAXNC][4];
            for (long p = 0; p < k->nvis; p++)
                for (int i = 0; i < 4; i++)
                    for (int j = 0; j < 4; j++)
                        for (int q = 0; q < 4; q++) {
                            int n1 = 4 * k->vis[3 * p] + i, n2 = 4 * k->vis[3 * p + 1] + j, n3 = 4 * k->vis[3 * p + 2] + q;
                            double r[3], da[3], db[3];
                            grid_pos(c, N, n1, n2, n3, r);
                            for (int x = 0; x < 3; x++) { da[x] = r[x] - k->A[x]; db[x] = r[x] - k->Bt[x]; }
                            shell_values(k->la, k->aa, k->ca, da, deriv, fa);
                            shell_values(k->lb, k->ab, k->cb, db, deriv, fb);
                            long m = ((long)posmod(n1, N[0]) * N[1] + posmod(n2, N[1])) * N[2] + posmod(n3, N[2]);
                            double v0 = vl[m];
                            for (int ia = 0; ia < nca; ia++)
                                for (int ib = 0; ib < ncb; ib++) {
                                    double s = v0 * fa[ia][0] * fb[ib][0];
                                    if (deriv)
                                        for (int x = 1; x < 4; x++)
                                            s += vl[x * ng + m] * (fa[ia][x] * fb[ib][0] + fa[ia][0] * fb[ib][x]);
                                    if (deriv == 2) /* Eq. (16) with the 1/2 of PAPER.md:265-268 */
                                        s += vl[4 * ng + m] * 0.5 * (fa[ia][1] * fb[ib][1] + fa[ia][2] * fb[ib][2] + fa[ia][3] * fb[ib][3]);
                                    acc[ia][ib] += (long double)(dV * s);
                                }
                        }
        }
        for (int ia = 0; ia < nca; ia++)
            for (int ib = 0; ib < ncb; ib++)
                F[(long)(k0->ao_a + ia) * c->nao + k0->ao_b + ib] = (double)acc[ia][ib];
    }
    free(gstart);
    clear_visits(c);
    return 0;
}


/* T11 nuclear gradient (Alg. 3).  E = sum_alpha dV_alpha sum_r [v0 rho_alpha + w . grad rho_alpha]
 * with rho_alpha the collocated density of T7; v (and w for deriv = 1) are held fixed, and so is the visit set.
 * grad[A][c] = dE/dR_{A,c}.  A basis function centred on atom A depends on R_A through r - R_A only, so
 * d/dR_{A,c} phi_i = -d_c phi_i; for deriv = 1 the second derivatives d_x d_c phi_i enter through
 * d/dR_{A,c} d_x (phi_i phi_j) = -(d_x d_c phi_i phi_j + d_c phi_i d_x phi_j)  (phi_i on A)
 * and likewise for phi_j on B.  A lattice image B + T moves with B.  v[level]: [ncomp][N1][N2][N3]. */
int orc_eval_grad(orc_ctx *c, const double *const *v, int deriv, const double *D, double *grad)
{
    if (deriv != 0 && deriv != 1) return -1;
    build_visits(c, NULL, NULL);
    int natm = c->natm;
    int nth = orc_num_threads();
    long double *part = (long double *)calloc((size_t)nth * 3 * natm, sizeof(long double));
#pragma omp parallel for schedule(dynamic, 4)
    for (long t = 0; t < c->ntask; t++) {
#ifdef _OPENMP
        long double *g = part + (size_t)omp_get_thread_num() * 3 * natm;
#else
        long double *g = part;
#endif
        const orc_task *k = c->task + t;
        const int *N = c->mesh + 3 * k->level;
        long ng = (long)N[0] * N[1] * N[2];
        double dV = c->omega / (double)ng;
        const double *vl = v[k->level];
        int nca = ncart(k->la), ncb = ncart(k->lb);
        int atom_a = c->shl_atom[k->shl_a], atom_b = c->shl_atom[k->shl_b];
        double fa[ORC_MAXNC][4], fb[ORC_MAXNC][4], ha[ORC_MAXNC][3][3], hb[ORC_MAXNC][3][3];
        for (long p = 0; p < k->nvis; p++)
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++)
                    for (int q = 0; q < 4; q++) {
                        int n1 = 4 * k->vis[3 * p] + i, n2 = 4 * k->vis[3 * p + 1] + j, n3 = 4 * k->vis[3 * p + 2] + q;
                        double r[3], da[3], db[3];
                        grid_pos(c, N, n1, n2, n3, r);
                        for (int x = 0; x < 3; x++) { da[x] = r[x] - k->A[x]; db[x] = r[x] - k->Bt[x]; }
                        shell_values(k->la, k->aa, k->ca, da, 1, fa);
                        shell_values(k->lb, k->ab, k->cb, db, 1, fb);
                        if (deriv) {
                            shell_hessian(k->la, k->aa, k->ca, da, ha);
                            shell_hessian(k->lb, k->ab, k->cb, db, hb);
                        }
                        long m = ((long)posmod(n1, N[0]) * N[1] + posmod(n2, N[1])) * N[2] + posmod(n3, N[2]);
                        double v0 = vl[m];
                        for (int ia = 0; ia < nca; ia++)
                            for (int ib = 0; ib < ncb; ib++) {
                                double d = D[(long)(k->ao_a + ia) * c->nao + k->ao_b + ib] * dV;
                                for (int cc = 0; cc < 3; cc++) {
                                    /* d/dR_A: phi_a -> -d_c phi_a ;  d/dR_B: phi_b -> -d_c phi_b */
                                    double ga = -v0 * fa[ia][1 + cc] * fb[ib][0];
                                    double gb = -v0 * fa[ia][0] * fb[ib][1 + cc];
                                    if (deriv)
                                        for (int x = 0; x < 3; x++) {
                                            double w = vl[(1 + x) * ng + m];
                                            ga -= w * (ha[ia][x][cc] * fb[ib][0] + fa[ia][1 + cc] * fb[ib][1 + x]);
                                            gb -= w * (fa[ia][1 + x] * fb[ib][1 + cc] + fa[ia][0] * hb[ib][x][cc]);
                                        }
                                    g[3 * atom_a + cc] += (long double)(d * ga);
                                    g[3 * atom_b + cc] += (long double)(d * gb);
                                }
                            }
                    }
    }
    for (int i = 0; i < 3 * natm; i++) {
        long double s = 0;
        for (int th = 0; th < nth; th++) s += part[(size_t)th * 3 * natm + i];
        grad[i] = (double)s;
    }
    free(part);
    clear_visits(c);
    return 0;
}
