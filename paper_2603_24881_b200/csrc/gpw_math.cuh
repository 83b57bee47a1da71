// Per-thread arithmetic of the collocation / integration path, written as __host__ __device__
// templates so that the identical code can be stepped on the host while developing.
//
// Formulation:  for one primitive pair the product of Eq. (23) is
//     sum_ij D_ij phi_a,i(r) phi_b,j(r - T) = Q(r - P) exp(-a_p |r - P|^2)
// with Q a polynomial of total degree L = la + lb.  A pre-pass expands Q about the Gaussian-product
// centre P (binomial expansion, Eq. 26-27) and rewrites it in grid-index coordinates
// u = n - n_P (r - P = H u, H = grid step matrix), which keeps one code path for orthorhombic and
// non-orthogonal cells (the paper's A.30-A.33 split).  A lane owns a slab of 4 x 4 grid
// points at its own n1: the polynomial is collapsed in u1 once per slab, in u2 once per row and swept by
// Horner in u3 per point.  The Gaussian on the slab follows the recursion of Eq. (24)-(25)
// from its value at the slab corner and two first-step ratios.  Integration is the exact transpose: row sums,
// partial moments at fixed u1, then the expansion in u1.
#pragma once
#include "gpw_internal.h"

#if defined(__CUDACC__)
#define GPW_HD __host__ __device__ __forceinline__
#else
#define GPW_HD inline
#endif

namespace gpw {

// position of u1^kx u2^ky u3^kz in a pair's polynomial of degree L (kz-major, then ky, then kx)
GPW_HD constexpr int cidx(int L, int kx, int ky, int kz) {
    int o = 0;
    for (int z = 0; z < kz; z++) o += (L - z + 1) * (L - z + 2) / 2;
    for (int y = 0; y < ky; y++) o += (L - kz - y + 1);
    return o + kx;
}
// position of a degree-d monomial X^a Y^b Z^c in the degree-graded order (degree blocks, inside a block
// decreasing a then decreasing b)
GPW_HD constexpr int gidx(int a, int b, int c) {
    const int d = a + b + c;
    const int r = d - a;
    return d * (d + 1) * (d + 2) / 6 + r * (r + 1) / 2 + (r - b);
}

GPW_HD void cart_of(int l, int i, int &lx, int &ly, int &lz) {
    // component i of a shell: decreasing lx, then decreasing ly
    int n = 0;
    for (int x = l; x >= 0; x--)
        for (int y = l - x; y >= 0; y--) {
            if (n == i) { lx = x; ly = y; lz = l - x - y; return; }
            n++;
        }
    lx = ly = lz = 0;
}

// 1-D binomial tables: Tt[x][i][j][k] = coefficient of X^k in (X + PA_x)^i (X + PB_x)^j   (Eq. 26-27)
struct BinomTables {
    double t[3][MAXL + 1][MAXL + 1][MAXLP + 1];
};

GPW_HD void build_binom(const TaskP &p, BinomTables &B) {
    const int la = p.la, lb = p.lb;
    for (int x = 0; x < 3; x++) {
        for (int i = 0; i <= la; i++)
            for (int j = 0; j <= lb; j++) {
                double *cur = B.t[x][i][j];
                for (int k = 0; k <= MAXLP; k++) cur[k] = 0.0;
                if (i == 0 && j == 0) { cur[0] = 1.0; continue; }
                const double *prev = i > 0 ? B.t[x][i - 1][j] : B.t[x][i][j - 1];
                const double off = i > 0 ? p.PA[x] : p.PB[x];
                for (int k = 0; k <= i + j; k++) cur[k] = (k > 0 ? prev[k - 1] : 0.0) + off * prev[k];
            }
    }
}

// Pre-pass: polynomial of one pair from its block of the density matrix.
//   out[cidx(L, k)] = pref * sum_ij Dsym_ij [coefficient of u^k in (r-A)^i (r-B-T)^j]
// S: this level's Cartesian -> grid-index monomial maps (degree blocks).
GPW_HD void pair_poly_from_D(const TaskP &p, const double *D, int nao, const double *S, double *out) {
    const int la = p.la, lb = p.lb, L = la + lb;
    BinomTables B;
    build_binom(p, B);
    double Cg[ncoef(MAXLP)];
    const int nc = ncoef(L);
    for (int k = 0; k < nc; k++) Cg[k] = 0.0;
    const int nca = ncart(la), ncb = ncart(lb);
    for (int i = 0; i < nca; i++) {
        int ix, iy, iz;
        cart_of(la, i, ix, iy, iz);
        for (int j = 0; j < ncb; j++) {
            int jx, jy, jz;
            cart_of(lb, j, jx, jy, jz);
            double d = D[(long long)(p.ao_a + i) * nao + p.ao_b + j];
            if (p.sym) d += D[(long long)(p.ao_b + j) * nao + p.ao_a + i];
            for (int kx = 0; kx <= ix + jx; kx++) {
                const double tx = d * B.t[0][ix][jx][kx];
                for (int ky = 0; ky <= iy + jy; ky++) {
                    const double txy = tx * B.t[1][iy][jy][ky];
                    for (int kz = 0; kz <= iz + jz; kz++) Cg[gidx(kx, ky, kz)] += txy * B.t[2][iz][jz][kz];
                }
            }
        }
    }
    // Cartesian -> grid-index coordinates, degree by degree, into the Horner order
    for (int d = 0; d <= L; d++) {
        const int nd = (d + 1) * (d + 2) / 2;
        const double *Sd = S + s_block_off(d);
        const double *Cd = Cg + d * (d + 1) * (d + 2) / 6;
        int row = 0;
        for (int a = d; a >= 0; a--)
            for (int b = d - a; b >= 0; b--, row++) {
                double s = 0.0;
                for (int col = 0; col < nd; col++) s += Sd[row * nd + col] * Cd[col];
                out[cidx(L, a, b, d - a - b)] = p.pref * s;
            }
    }
}

// Post-pass: F block of one pair from its moment vector  m[cidx(L,k)] = sum_r w(r) G(r) u^k.
//   Fblk[i*ncb + j] = pref * dV * sum_k [coefficient of u^k in (r-A)^i (r-B-T)^j] m[k]
GPW_HD void pair_block_from_moments(const TaskP &p, const double *m, const double *S, double dV, double *Fblk) {
    const int la = p.la, lb = p.lb, L = la + lb;
    BinomTables B;
    build_binom(p, B);
    double Cg[ncoef(MAXLP)];
    for (int d = 0; d <= L; d++) {
        const int nd = (d + 1) * (d + 2) / 2;
        const double *Sd = S + s_block_off(d);
        double *Cd = Cg + d * (d + 1) * (d + 2) / 6;
        for (int col = 0; col < nd; col++) Cd[col] = 0.0;
        int row = 0;
        for (int a = d; a >= 0; a--)
            for (int b = d - a; b >= 0; b--, row++) {
                const double mv = m[cidx(L, a, b, d - a - b)];
                for (int col = 0; col < nd; col++) Cd[col] += Sd[row * nd + col] * mv;
            }
    }
    const int nca = ncart(la), ncb = ncart(lb);
    const double scale = p.pref * dV;
    for (int i = 0; i < nca; i++) {
        int ix, iy, iz;
        cart_of(la, i, ix, iy, iz);
        for (int j = 0; j < ncb; j++) {
            int jx, jy, jz;
            cart_of(lb, j, jx, jy, jz);
            double s = 0.0;
            for (int kx = 0; kx <= ix + jx; kx++)
                for (int ky = 0; ky <= iy + jy; ky++) {
                    const double txy = B.t[0][ix][jx][kx] * B.t[1][iy][jy][ky];
                    for (int kz = 0; kz <= iz + jz; kz++) s += txy * B.t[2][iz][jz][kz] * Cg[gidx(kx, ky, kz)];
                }
            Fblk[i * ncb + j] = scale * s;
        }
    }
}

// ------------------------------------------------------------------------------------------ slab form
// A lane owns the slab of 4 x 4 grid points (rows j along n2, points t along n3) at its own n1.  The
// polynomial is collapsed once per slab in u1 (b[ky][kz]), once per row in u2 (a[kz]) and swept by Horner
// in u3 per point; the Gaussian is one exp() at the slab corner plus two first-step ratios, everything
// else follows by the recursion of Eq. (24)-(25) with the constant second-order ratios c22, c23, c33.

// number of (ky,kz) with ky + kz <= L, and the position of (ky,kz) among them (kz-major)
GPW_HD constexpr int npair2(int L) { return L < 0 ? 0 : (L + 1) * (L + 2) / 2; }
GPW_HD constexpr int bidx(int L, int ky, int kz) {
    int o = 0;
    for (int z = 0; z < kz; z++) o += L - z + 1;
    return o + ky;
}

// Gaussian at the slab corner and the first-step ratios along n2 and n3.
//   g0 = exp(-E(u1,u20,u30)),  r2 = G(j=1,t=0)/G(0,0),  r3 = G(0,1)/G(0,0)
// Every intermediate of the recursion is a true Gaussian value or a true ratio of neighbouring values, so
// it stays inside the FP64 range as long as q u^2 < 700 over the visited blocks (q = a_p h^2 <= ~1 for the
// sharpest pairs routed to level 0 by reading A23, u <= R_t/h + 7 grid steps: two orders of magnitude of
// margin on every config).  ORTHO: the level's step vectors are mutually orthogonal (Gm is diagonal).
struct SlabGauss { double g0, r2, r3; };
template <bool ORTHO = false>
GPW_HD SlabGauss slab_gauss(const double *q, double u1, double u20, double u30) {
    SlabGauss G;
    if constexpr (ORTHO) {
        const double E0 = fma(q[0] * u1, u1, fma(q[1] * u20, u20, q[2] * u30 * u30));
        G.g0 = exp(-E0);
        G.r2 = exp(-(q[1] * fma(2.0, u20, 1.0)));
        G.r3 = exp(-(q[2] * fma(2.0, u30, 1.0)));
    } else {
        const double E0 = q[0] * u1 * u1 + q[1] * u20 * u20 + q[2] * u30 * u30 +
                          2.0 * (q[3] * u1 * u20 + (q[4] * u1 + q[5] * u20) * u30);
        const double s2 = 2.0 * (q[3] * u1 + q[1] * u20 + q[5] * u30) + q[1];
        const double s3 = 2.0 * (q[4] * u1 + q[5] * u20 + q[2] * u30) + q[2];
        G.g0 = exp(-E0); G.r2 = exp(-s2); G.r3 = exp(-s3);
    }
    return G;
}
// Collocation of one pair on one slab.  acc[NCOMP][16] (index j*4+t); for DERIV the gradient is
// accumulated in grid-index (covariant) components:  d/du_i [Q G] = G (dQ/du_i + p_i Q),  p = -2 (q u).
// ORTHO: the Gaussian along n3 relative to the row start (g3) and p_3 are the same for the four rows, p_1
// is constant on the slab and p_2 on a row.
template <int L, int DERIV, bool ORTHO = false>
GPW_HD void colloc_slab(const double *__restrict__ c, const double *q, double c22, double c23, double c33,
                        const SlabGauss SG, double u1, double u20, double u30, double (*acc)[16]) {
    constexpr int NB = npair2(L), NBX = npair2(L - 1);
    double b[NB], bx[NBX > 0 ? NBX : 1];
#pragma unroll
    for (int kz = 0; kz <= L; kz++)
#pragma unroll
        for (int ky = 0; ky <= L - kz; ky++) {
            const int n = L - kz - ky;          // degree in u1
            double p = c[cidx(L, n, ky, kz)], dp = 0.0;
#pragma unroll
            for (int kx = n - 1; kx >= 0; kx--) {
                if (DERIV) dp = kx == n - 1 ? p : fma(dp, u1, p);
                p = fma(p, u1, c[cidx(L, kx, ky, kz)]);
            }
            b[bidx(L, ky, kz)] = p;
            if (DERIV && ky + kz <= L - 1) bx[bidx(L - 1, ky, kz)] = dp;
        }
    double grow = SG.g0, r2 = SG.r2, r3row = SG.r3;
    // p = -2 (q u) at the row start, its step per row and per point
    double qr1 = 0.0, qr2 = 0.0, qr3 = 0.0;
    if (DERIV) {
        if constexpr (ORTHO) {
            qr1 = -2.0 * (q[0] * u1); qr2 = -2.0 * (q[1] * u20); qr3 = -2.0 * (q[2] * u30);
        } else {
            qr1 = -2.0 * (q[0] * u1 + q[3] * u20 + q[4] * u30);
            qr2 = -2.0 * (q[3] * u1 + q[1] * u20 + q[5] * u30);
            qr3 = -2.0 * (q[4] * u1 + q[5] * u20 + q[2] * u30);
        }
    }
    // ORTHO: Gaussian along n3 relative to the row start, and p_3 per point -- shared by the four rows
    double g3[4] = {1.0, 1.0, 1.0, 1.0}, p3t[4] = {0.0, 0.0, 0.0, 0.0};
    if constexpr (ORTHO) {
        double r = SG.r3;
        g3[1] = r; r *= c33; g3[2] = g3[1] * r; r *= c33; g3[3] = g3[2] * r;
        if (DERIV) {
#pragma unroll
            for (int t = 0; t < 4; t++) p3t[t] = fma(-2.0 * q[2], (double)t, qr3);
        }
    }
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const double u2 = u20 + j;
        double a[L + 1], ax[L > 0 ? L : 1], ay[L > 0 ? L : 1];
#pragma unroll
        for (int kz = 0; kz <= L; kz++) {
            const int n = L - kz;               // degree in u2
            double s = b[bidx(L, n, kz)], sy = 0.0;
#pragma unroll
            for (int ky = n - 1; ky >= 0; ky--) {
                if (DERIV) sy = ky == n - 1 ? s : fma(sy, u2, s);
                s = fma(s, u2, b[bidx(L, ky, kz)]);
            }
            a[kz] = s;
            if (DERIV && kz < L) {
                ay[kz] = sy;
                double sx = bx[bidx(L - 1, n - 1, kz)];
#pragma unroll
                for (int ky = n - 2; ky >= 0; ky--) sx = fma(sx, u2, bx[bidx(L - 1, ky, kz)]);
                ax[kz] = sx;
            }
        }
        double g = grow, r = r3row;
        double p1 = qr1, p2 = qr2, p3 = qr3;
#pragma unroll
        for (int t = 0; t < 4; t++) {
            const double u3 = u30 + t;
            if constexpr (ORTHO) { g = t == 0 ? grow : grow * g3[t]; p3 = p3t[t]; }
            double Q = a[L], Qz = 0.0;
#pragma unroll
            for (int kz = L - 1; kz >= 0; kz--) {
                if (DERIV) Qz = kz == L - 1 ? Q : fma(Qz, u3, Q);
                Q = fma(Q, u3, a[kz]);
            }
            acc[0][j * 4 + t] = fma(g, Q, acc[0][j * 4 + t]);
            if constexpr (DERIV != 0) {
                if constexpr (L > 0) {
                    double Qx = ax[L - 1], Qy = ay[L - 1];
#pragma unroll
                    for (int kz = L - 2; kz >= 0; kz--) { Qx = fma(Qx, u3, ax[kz]); Qy = fma(Qy, u3, ay[kz]); }
                    acc[1][j * 4 + t] = fma(g, fma(Q, p1, Qx), acc[1][j * 4 + t]);
                    acc[2][j * 4 + t] = fma(g, fma(Q, p2, Qy), acc[2][j * 4 + t]);
                    acc[3][j * 4 + t] = fma(g, fma(Q, p3, Qz), acc[3][j * 4 + t]);
                } else {
                    const double w = g * Q;
                    acc[1][j * 4 + t] = fma(w, p1, acc[1][j * 4 + t]);
                    acc[2][j * 4 + t] = fma(w, p2, acc[2][j * 4 + t]);
                    acc[3][j * 4 + t] = fma(w, p3, acc[3][j * 4 + t]);
                }
                if constexpr (!ORTHO) { p1 -= 2.0 * q[4]; p2 -= 2.0 * q[5]; p3 -= 2.0 * q[2]; }
            }
            if constexpr (!ORTHO) { g *= r; r *= c33; }
        }
        grow *= r2; r2 *= c22;
        if constexpr (!ORTHO) r3row *= c23;
        if (DERIV) {
            if constexpr (ORTHO) { qr2 -= 2.0 * q[1]; }
            else { qr1 -= 2.0 * q[3]; qr2 -= 2.0 * q[1]; qr3 -= 2.0 * q[5]; }
        }
    }
}

// Integration of one pair on one slab (exact transpose of colloc_slab), in two parts.
//
// integ_slab_rows: the u3 and u2 sweeps.  Accumulates the slab's partial moments at fixed u1,
//     B0[bidx(L,ky,kz)]   += sum_{j,t} g (v0 + z . p) u2^ky u3^kz   + derivative terms in u2, u3
//     B1[bidx(L-1,ky,kz)] += sum_{j,t} g z1 u2^ky u3^kz              (DERIV; multiplies d/du1)
// with p = -2 (q u) (the Gaussian's logarithmic gradient) and z the vector field in grid-index
// (contravariant) components.  vrow(comp, j, out[4]) delivers the four values of row j of component comp.
// A lane of the integration kernel keeps B0 / B1 over ALL blocks of a brick entry: the brick is one block
// thick along n1, so the lane's u1 is the same for every block.
// ORTHO: the Gaussian separates, G = gx(u1) gy(u2) gz(u3).  The caller passes rowg[j] = gx gy(u20 + j),
// the offsets toff[t] of the lane's four points along n3 (a permutation of 0..3: the order in which the
// caller delivers them) and g3[t] = gz(u30 + toff[t]) (SG is not used); the table T[kz][t] = g3[t] u3_t^kz
// is the same for the four rows and the row's factor multiplies the row sums instead of every point.
//
// integ_expand_u1: m[cidx(L,kx,ky,kz)] (+)= B0 u1^kx + kx u1^(kx-1) B1 -- once per entry.
template <int L, int DERIV, bool ORTHO = false, class VRow>
GPW_HD void integ_slab_rows(VRow &&vrow, const double *q, double c22, double c23, double c33,
                            const SlabGauss SG, double u1, double u20, double u30, double *B0, double *B1,
                            const double *rowg = nullptr, const double *g3 = nullptr, const double *toff = nullptr) {
    constexpr int NCOMP = DERIV ? 4 : 1;
    double grow = SG.g0, r2 = SG.r2, r3row = SG.r3;
    double qr1 = 0.0, qr2 = 0.0, qr3 = 0.0;
    if (DERIV) {
        if constexpr (ORTHO) {
            qr1 = -2.0 * (q[0] * u1); qr2 = -2.0 * (q[1] * u20); qr3 = -2.0 * (q[2] * u30);
        } else {
            qr1 = -2.0 * (q[0] * u1 + q[3] * u20 + q[4] * u30);
            qr2 = -2.0 * (q[3] * u1 + q[1] * u20 + q[5] * u30);
            qr3 = -2.0 * (q[4] * u1 + q[5] * u20 + q[2] * u30);
        }
    }
    double T[L + 1][4], p3t[4] = {0.0, 0.0, 0.0, 0.0};
    if constexpr (ORTHO) {
#pragma unroll
        for (int t = 0; t < 4; t++) T[0][t] = g3[t];
#pragma unroll
        for (int kz = 1; kz <= L; kz++)
#pragma unroll
            for (int t = 0; t < 4; t++) T[kz][t] = T[kz - 1][t] * (u30 + toff[t]);
        if (DERIV) {
#pragma unroll
            for (int t = 0; t < 4; t++) p3t[t] = fma(-2.0 * q[2], toff[t], qr3);
        }
    }
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const double u2 = u20 + j;
        double vv[NCOMP][4];
#pragma unroll
        for (int k = 0; k < NCOMP; k++) vrow(k, j, vv[k]);
        double A0[L + 1], A1[L > 0 ? L : 1], A2[L > 0 ? L : 1], A3[L > 0 ? L : 1];
        if constexpr (ORTHO) {
            // row sums without the row's Gaussian factor (it multiplies pw2 below)
            double w0[4];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                w0[t] = vv[0][t];
                if constexpr (DERIV != 0) w0[t] = fma(vv[1][t], qr1, fma(vv[2][t], qr2, fma(vv[3][t], p3t[t], w0[t])));
            }
#pragma unroll
            for (int kz = 0; kz <= L; kz++) {
                A0[kz] = fma(T[kz][3], w0[3], fma(T[kz][2], w0[2], fma(T[kz][1], w0[1], T[kz][0] * w0[0])));
                if (DERIV && kz < L) {
                    A1[kz] = fma(T[kz][3], vv[1][3], fma(T[kz][2], vv[1][2], fma(T[kz][1], vv[1][1], T[kz][0] * vv[1][0])));
                    A2[kz] = fma(T[kz][3], vv[2][3], fma(T[kz][2], vv[2][2], fma(T[kz][1], vv[2][1], T[kz][0] * vv[2][0])));
                    A3[kz] = fma(T[kz][3], vv[3][3], fma(T[kz][2], vv[3][2], fma(T[kz][1], vv[3][1], T[kz][0] * vv[3][0])));
                }
            }
        } else {
#pragma unroll
            for (int kz = 0; kz <= L; kz++) A0[kz] = 0.0;
#pragma unroll
            for (int kz = 0; kz < L; kz++) { A1[kz] = 0.0; A2[kz] = 0.0; A3[kz] = 0.0; }
            double g = grow, r = r3row;
            double p1 = qr1, p2 = qr2, p3 = qr3;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const double u3 = u30 + t;
                double g0 = vv[0][t], g1 = 0.0, g2 = 0.0, g3 = 0.0;
                if constexpr (DERIV != 0) {
                    const double z1 = vv[1][t], z2 = vv[2][t], z3 = vv[3][t];
                    g0 = fma(z1, p1, fma(z2, p2, fma(z3, p3, g0)));
                    g1 = g * z1; g2 = g * z2; g3 = g * z3;
                    p1 -= 2.0 * q[4]; p2 -= 2.0 * q[5]; p3 -= 2.0 * q[2];
                }
                g0 *= g;
                double pw = 1.0;
#pragma unroll
                for (int kz = 0; kz <= L; kz++) {
                    if (kz == 0) {
                        A0[0] += g0;
                        if (DERIV && L > 0) { A1[0] += g1; A2[0] += g2; A3[0] += g3; }
                    } else {
                        A0[kz] = fma(g0, pw, A0[kz]);
                        if (DERIV && kz < L) { A1[kz] = fma(g1, pw, A1[kz]); A2[kz] = fma(g2, pw, A2[kz]); A3[kz] = fma(g3, pw, A3[kz]); }
                    }
                    if (kz < L) pw = kz == 0 ? u3 : pw * u3;
                }
                g *= r; r *= c33;
            }
        }
        if (DERIV) {
#pragma unroll
            for (int kz = 1; kz <= L; kz++) A0[kz] = fma((double)kz, A3[kz - 1], A0[kz]);
        }
        // powers of u2 (ORTHO: times the row's Gaussian factor)
        double pw2[L + 1];
        pw2[0] = ORTHO ? rowg[j] : 1.0;
#pragma unroll
        for (int k = 1; k <= L; k++) pw2[k] = (k == 1 && !ORTHO) ? u2 : pw2[k - 1] * u2;
#pragma unroll
        for (int kz = 0; kz <= L; kz++)
#pragma unroll
            for (int ky = 0; ky <= L - kz; ky++) {
                if (ky == 0 && !ORTHO) B0[bidx(L, 0, kz)] += A0[kz];
                else B0[bidx(L, ky, kz)] = fma(A0[kz], pw2[ky], B0[bidx(L, ky, kz)]);
                if (DERIV && ky > 0) B0[bidx(L, ky, kz)] = fma(A2[kz], ky * pw2[ky - 1], B0[bidx(L, ky, kz)]);
                if (DERIV && ky + kz <= L - 1) {
                    if (ky == 0 && !ORTHO) B1[bidx(L - 1, 0, kz)] += A1[kz];
                    else B1[bidx(L - 1, ky, kz)] = fma(A1[kz], pw2[ky], B1[bidx(L - 1, ky, kz)]);
                }
            }
        if constexpr (!ORTHO) { grow *= r2; r2 *= c22; r3row *= c23; }
        if (DERIV) {
            if constexpr (ORTHO) { qr2 -= 2.0 * q[1]; }
            else { qr1 -= 2.0 * q[3]; qr2 -= 2.0 * q[1]; qr3 -= 2.0 * q[5]; }
        }
    }
}

// contribution of this lane's B0 / B1 to moment (kx,ky,kz):  B0 u1^kx + kx u1^(kx-1) B1
template <int L, int DERIV>
GPW_HD double integ_expand_term(const double *B0, const double *B1, const double *pw1, int kx, int ky, int kz) {
    double s = kx == 0 ? B0[bidx(L, ky, kz)] : B0[bidx(L, ky, kz)] * pw1[kx];
    if (DERIV && kx > 0) s += B1[bidx(L - 1, ky, kz)] * (kx * pw1[kx - 1]);
    return s;
}

}  // namespace gpw
