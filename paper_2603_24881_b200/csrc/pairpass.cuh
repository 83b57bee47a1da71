// Pre- and post-pass of the grid kernels: pair block of D -> pair polynomial, pair moments -> block of F / atom forces.
//
// For one primitive pair the product of Eq. (23) is a polynomial times one Gaussian about P:
//     sum_ij D_ij phi_a,i(r) phi_b,j(r - T) = pref Q(X) exp(-a_p |X|^2),   X = r - P,
// and the grid kernels work with Q in grid-index coordinates u (X = H u).  The pre-pass builds Q from the pair's
// block of D, the post-pass maps the pair's moments m[k] = sum_r w(r) G(r) u^k back to the block of F; the
// derivative variants (kinetic-energy density, Eq. 15-16; nuclear gradient, Alg. 3
// PAPER.md:272-309) differ only in the polynomial: degree L + 2 and L + 1.
//
// Form (tensor-product expansion of Eq. 26-27, done by Taylor shifts one axis at a time; no
// binomial tables, no per-thread arrays).  With Y = r - A = X + PA and Z = r - B - T = Y + s, s = PB - PA:
//   1. q_i(Z) = sum_j D_ij Z^j                      the rows of the D block are homogeneous polynomials of degree lb
//   2. q'_i(Y) = q_i(Y + s)                         Taylor shift, one axis at a time
//   3. R(Y) = sum_i Y^i q'_i(Y)                     index shift and sum ("gather")
//   4. Q(X) = R(X + PA)                             Taylor shift
//   5. coefficients in u: per degree d the map S_d  (orthogonal cells: a diagonal scaling)
// The kinetic-energy density 1/2 grad phi_i . grad phi_j replaces step 3 by a five-point stencil per axis c:
//   (d_c - 2 a_a Y_c) Y^i . (d_c - 2 a_b (Y_c + s_c)) Y^n / 2 =
//        i_c n_c / 2 Y^(i+n-2e_c) - a_b s_c i_c Y^(i+n-e_c) - (a_b i_c + a_a n_c) Y^(i+n)
//        + 2 a_a a_b s_c Y^(i+n+e_c) + 2 a_a a_b Y^(i+n+2e_c)
// The post-pass is the exact transpose, step by step in reverse; the nuclear gradient contracts q' (steps 1-2)
// with the Y-moments (steps 5^T, 4^T) through d/dA_c phi_i = -(i_c Y^(i-e_c) - 2 a_a Y^(i+e_c)) e^.. and
// d/dB_c phi_j = -(d_c - 2 a_b (Y_c + s_c)) q'.
//
// A group of PP_G lanes works on one pair; all arrays live in the group's shared memory, dependencies inside the
// group are ordered by __syncwarp(group mask).  The same code runs on the host with a group of one lane.
#pragma once
#include "gpw_internal.h"

#if defined(__CUDACC__)
#define PP_HD __host__ __device__ __forceinline__
#else
#define PP_HD inline
#endif

namespace gpw {
namespace pp {

constexpr int PP_G = 8;   // lanes per pair

enum Mode : int {
    PRE_DENS = 1,    // D -> polynomial of degree L           (gpw_eval_rho)
    PRE_TAU = 2,     // D -> polynomial of degree L + 2       (gpw_eval_rho, deriv = 2)
    POST_MAT = 4,    // moments of degree L -> F              (gpw_eval_mat)
    POST_TAU = 8,    // moments of degree L + 2 -> F          (gpw_eval_mat, deriv = 2)
    POST_GRAD = 16   // D and moments of degree L + 1 -> atom gradients   (gpw_eval_grad)
};

struct PassArgs {
    const TaskP *tp;
    int ntask, nao, hdiag, mode;                      // hdiag: every level's step matrix H is diagonal (S_d diagonal)
    // the pairs a launch of the group form works on: nsel pairs in up to GPW_MAX_LEVEL ranges, pair number j of the
    // selection being sel_lo[r] + (j - sel_cum[r]) for sel_cum[r] <= j < sel_cum[r + 1]
    int nsel;
    int sel_cum[GPW_MAX_LEVEL + 1];
    int sel_lo[GPW_MAX_LEVEL];
    int big_lo[GPW_MAX_LEVEL], big_n[GPW_MAX_LEVEL];   // per level: the pairs with la + lb >= 5
    int lmin_hot;                                     // PRE_DENS / POST_MAT only for pairs with la + lb >= lmin_hot (the others
                                                      // are done by the register form, pairpass_reg.cuh)
    const double *S_all;                              // [nlevel][S_TOTAL] Cartesian -> grid-index monomial maps
    long long base[NOFF][GPW_MAX_LEVEL][8];           // workspace offset of pair t of class (level, L) = base + t * ncoef_pad(L + off)
    double dV[GPW_MAX_LEVEL];
    const double *D;                                  // [nao][nao]
    double *rec[NOFF];                                // collocation records: 8-double header + polynomial per pair
    const double *mom[NOFF];                          // moment workspaces
    double *F;                                        // [nao][nao]
    double *grad;                                     // [natm][3]
};

// Index tables of the polynomials of degree n <= MAXDEG (kept in shared memory by the kernel: the index arithmetic
// they replace -- tetrahedral numbers, divisions -- was 80 % of the instructions of the first version of this pass).
//   zt[n * 9 + kz]    position of the first coefficient with exponent kz:  tet(n + 1) - tet(n + 1 - kz)
//   lt[tet(n) + i]    line i of a polynomial of degree n: (ky | kz << 8), kz-major -- also the (a, b) with a + b <= n
//   gt[goff(n) + k]   position (in the kz-major order) of monomial k of the degree-graded order (degree blocks, inside a
//                     block decreasing x, then decreasing y -- the order of the maps S_d)
//   mt[goff(n) + k]   exponents of coefficient k of the kz-major order: x | y << 4 | z << 8
constexpr int tet_c(int m) { return m * (m + 1) * (m + 2) / 6; }
constexpr int goff_c(int n) { int o = 0; for (int m = 0; m < n; m++) o += ncoef(m); return o; }
constexpr int NTAB = goff_c(MAXDEG + 1);   // 495
struct Tables {
    unsigned char zt[(MAXDEG + 1) * 9];
    unsigned char gt[NTAB];
    unsigned short lt[ncoef(MAXDEG)];
    unsigned short mt[NTAB];
};
inline void fill_tables(Tables &T) {
    for (int n = 0; n <= MAXDEG; n++) {
        for (int kz = 0; kz <= n; kz++) T.zt[n * 9 + kz] = (unsigned char)(tet_c(n + 1) - tet_c(n + 1 - kz));
        int i = 0, k = 0;
        for (int kz = 0; kz <= n; kz++)
            for (int ky = 0; ky <= n - kz; ky++) {
                T.lt[tet_c(n) + i++] = (unsigned short)(ky | kz << 8);
                for (int kx = 0; kx <= n - kz - ky; kx++) T.mt[goff_c(n) + k++] = (unsigned short)(kx | ky << 4 | kz << 8);
            }
        int gk = 0;
        for (int d = 0; d <= n; d++)
            for (int a = d; a >= 0; a--)
                for (int b = d - a; b >= 0; b--) {
                    const int c = d - a - b;
                    T.gt[goff_c(n) + gk++] = (unsigned char)(tet_c(n + 1) - tet_c(n + 1 - c) + b * (n - c + 1) - b * (b - 1) / 2 + a);
                }
    }
}

struct Grp {
    int gl;          // lane within the group
    int G;           // lanes in the group (PP_G on the device, 1 on the host)
    unsigned mask;   // the group's lanes
    const Tables *tab;
};

PP_HD void gsync(const Grp &g) {
#if defined(__CUDA_ARCH__)
    __syncwarp(g.mask);
#else
    (void)g;
#endif
}
PP_HD void add_to(double *p, double v) {
#if defined(__CUDA_ARCH__)
    atomicAdd(p, v);
#else
    *p += v;
#endif
}
PP_HD double gsum(double v, const Grp &g) {
#if defined(__CUDA_ARCH__)
    v += __shfl_xor_sync(g.mask, v, 1);
    v += __shfl_xor_sync(g.mask, v, 2);
    v += __shfl_xor_sync(g.mask, v, 4);
#else
    (void)g;
#endif
    return v;
}

PP_HD constexpr int tet(int m) { return m * (m + 1) * (m + 2) / 6; }
PP_HD int goff(int n) { return n * (n + 1) * (n + 2) * (n + 3) / 24; }   // sum_{m<n} ncoef(m)
// position of x^kx y^ky z^kz in a polynomial of total degree <= n: kz-major, then ky, then kx (= cidx of gpw_math.cuh)
PP_HD int pidx(const Grp &g, int n, int kx, int ky, int kz) {
    return g.tab->zt[n * 9 + kz] + ky * (n - kz + 1) - ((ky * (ky - 1)) >> 1) + kx;
}
// coefficient (kx,ky,kz) of a polynomial of degree <= n, zero outside its support
PP_HD double pget(const Grp &g, const double *p, int n, int kx, int ky, int kz) {
    return (kx < 0 || ky < 0 || kz < 0 || kx + ky + kz > n) ? 0.0 : p[pidx(g, n, kx, ky, kz)];
}
// floor(e / d) for the small non-negative e of this file (e < 4096, d <= 32), by a reciprocal computed once per pair
PP_HD int recip16(int d) { return 65536 / d + 1; }
PP_HD int divr(int e, int r) { return (e * r) >> 16; }
// offset of the degree block S_d: sum_{e<d} ((e+1)(e+2)/2)^2 (= s_block_off(d), in closed form)
PP_HD int sblock(int d) { return d * (d + 1) * (d + 2) * (3 * d * d + 6 * d + 1) / 60; }
// row / column of monomial (a,b,c) inside the degree block S_d, d = a + b + c: decreasing a, then decreasing b
PP_HD int gidx_in_block(int a, int b, int d) {
    const int r = d - a;
    return r * (r + 1) / 2 + (r - b);
}

// One line of a polynomial of degree <= n along `axis`, the other two exponents being (a, b) in the order
// (y,z), (x,z), (x,y): Taylor shift c(x) -> c(x + s) in place, or its transpose (moments of x^j -> moments of (x+s)^j).
template <int NMAX, bool TRANS>
PP_HD void shift_line(const Grp &g, double *p, int n, int axis, int a, int b, double s) {
    const int m = n - a - b + 1;   // entries of the line
    double c[NMAX + 1];
    int ad[NMAX + 1];
    // addresses along the line, by differences of pidx: x: 1;  y: (n - kz + 1) - ky;  z: tri(n + 1 - kz) - ky
    ad[0] = axis == 0 ? pidx(g, n, 0, a, b) : (axis == 1 ? pidx(g, n, a, 0, b) : pidx(g, n, a, b, 0));
#pragma unroll
    for (int j = 0; j < NMAX; j++)
        ad[j + 1] = ad[j] + (axis == 0 ? 1 : (axis == 1 ? (n - b + 1) - j : (n + 1 - j) * (n + 2 - j) / 2 - b));
#pragma unroll
    for (int j = 0; j <= NMAX; j++) c[j] = j < m ? p[ad[j]] : 0.0;
    if (!TRANS) {
#pragma unroll
        for (int i = 0; i < NMAX; i++)
#pragma unroll
            for (int j = NMAX - 1; j >= i; j--) c[j] = fma(s, c[j + 1], c[j]);
    } else {
#pragma unroll
        for (int i = NMAX - 1; i >= 0; i--)
#pragma unroll
            for (int j = i; j < NMAX; j++) c[j + 1] = fma(s, c[j], c[j + 1]);
    }
#pragma unroll
    for (int j = 0; j <= NMAX; j++)
        if (j < m) p[ad[j]] = c[j];
}

// Taylor shift (or its transpose) of npoly polynomials of degree <= n, `stride` doubles apart, by the vector s.
template <bool TRANS>
PP_HD void shift_polys(double *p, int npoly, int stride, int n, const double *s, const Grp &g) {
    if (n == 0) return;
    const int nl = n * (n + 1) / 2;   // lines with at least two entries: (a, b), a + b < n
#pragma unroll
    for (int axis = 0; axis < 3; axis++) {
        const int rnl = recip16(nl);
        for (int e = g.gl; e < npoly * nl; e += g.G) {
            const int ip = divr(e, rnl);
            const int ab = g.tab->lt[tet(n - 1) + (e - ip * nl)];   // the lines (a, b), a + b <= n - 1
            const int a = ab & 0xff, b = ab >> 8;
            double *q = p + ip * stride;
            if (n <= 3) shift_line<3, TRANS>(g, q, n, axis, a, b, s[axis]);
            else if (n <= 6) shift_line<6, TRANS>(g, q, n, axis, a, b, s[axis]);
            else shift_line<MAXDEG, TRANS>(g, q, n, axis, a, b, s[axis]);
        }
        gsync(g);
    }
}

// Cartesian component i of a shell of angular momentum l -> exponents (decreasing lx, then decreasing ly)
PP_HD void comp_of(int l, int i, int &lx, int &ly, int &lz) {
    int n = 0;
    lx = ly = lz = 0;
    for (int x = l; x >= 0; x--)
        for (int y = l - x; y >= 0; y--, n++)
            if (n == i) { lx = x; ly = y; lz = l - x - y; }
}

// All of one pair.  q: [ncart(la)][NQ] doubles, R: ncoef(L + 2) doubles (the group's shared memory).
template <int NQ>
PP_HD void pair_pass(const PassArgs &A, int t, double *q, double *R, const Grp &g) {
    const TaskP p = A.tp[t];
    const int la = p.la, lb = p.lb, L = la + lb;
    const int nca = ncart(la), ncb = ncart(lb);
    const int nq = ncoef(lb);
    const double *S = A.S_all + (size_t)p.level * S_TOTAL;
    const double s[3] = {p.PB[0] - p.PA[0], p.PB[1] - p.PA[1], p.PB[2] - p.PA[2]};
    int mode = A.mode;
    if (L < A.lmin_hot) mode &= ~(PRE_DENS | POST_MAT);
    if (mode == 0) return;

    // S_d between Cartesian coefficients / moments about P (in R, degree <= n) and grid-index ones (in global memory)
    // Coefficient k of the kz-major order has exponents mt[k]; inside its degree block d it is row gidx_in_block of S_d,
    // and column `col` of that block is coefficient gt[tet(d) + col] of the kz-major order.
    const Tables &T = *g.tab;
    auto cart_to_grid = [&](int n, double scale, double *out) {   // out[k_u] = scale sum_col S[row k_u][col] R[col]
        const unsigned short *mt = T.mt + goff(n);
        const unsigned char *gt = T.gt + goff(n);
        for (int k = g.gl; k < ncoef(n); k += g.G) {
            const int kx = mt[k] & 15, ky = (mt[k] >> 4) & 15, kz = mt[k] >> 8;
            const int d = kx + ky + kz, nd = (d + 1) * (d + 2) / 2;
            const double *Sd = S + sblock(d);
            const int row = gidx_in_block(kx, ky, d);
            double v;
            if (A.hdiag) v = Sd[row * nd + row] * R[k];
            else {
                v = 0.0;
                const unsigned char *gd = gt + tet(d);
                const double *Sr = Sd + row * nd;
                for (int col = 0; col < nd; col++) v = fma(Sr[col], R[gd[col]], v);
            }
            out[k] = scale * v;
        }
    };
    auto grid_to_cart = [&](int n, double scale, const double *m) {   // R[col] = scale sum_row S[row][col] m[row]
        const unsigned short *mt = T.mt + goff(n);
        const unsigned char *gt = T.gt + goff(n);
        for (int k = g.gl; k < ncoef(n); k += g.G) {
            const int kx = mt[k] & 15, ky = (mt[k] >> 4) & 15, kz = mt[k] >> 8;
            const int d = kx + ky + kz, nd = (d + 1) * (d + 2) / 2;
            const double *Sd = S + sblock(d);
            const int col = gidx_in_block(kx, ky, d);
            double v;
            if (A.hdiag) v = Sd[col * nd + col] * m[k];
            else {
                v = 0.0;
                const unsigned char *gd = gt + tet(d);
                for (int row = 0; row < nd; row++) v = fma(Sd[row * nd + col], m[gd[row]], v);
            }
            R[k] = scale * v;
        }
        gsync(g);
    };
    const int rncb = recip16(ncb), rnq = recip16(nq);

    // ---- steps 1-2 (pre-pass, gradient): q'_i(Y) from the D block ----
    if (mode & (PRE_DENS | PRE_TAU | POST_GRAD)) {
        for (int e = g.gl; e < nca * NQ; e += g.G) q[e] = 0.0;
        gsync(g);
        for (int e = g.gl; e < nca * ncb; e += g.G) {
            const int i = divr(e, rncb), j = e - i * ncb;
            int jx, jy, jz;
            comp_of(lb, j, jx, jy, jz);
            double d = A.D[(size_t)(p.ao_a + i) * A.nao + p.ao_b + j];
            if (p.sym) d += A.D[(size_t)(p.ao_b + j) * A.nao + p.ao_a + i];
            q[i * NQ + pidx(g, lb, jx, jy, jz)] = d;
        }
        gsync(g);
        shift_polys<false>(q, nca, NQ, lb, s, g);
    }

    // ---- step 3: R(Y) = sum_i Y^i q'_i(Y) (density), or the kinetic-energy stencil; steps 4-5 ----
    auto finish_pre = [&](int off) {
        const int n = L + off;
        gsync(g);
        shift_polys<false>(R, 1, 0, n, p.PA, g);
        double *out = A.rec[off] + A.base[off][p.level][L] + (long long)t * (ncoef_pad(n) + 8) + 8;
        cart_to_grid(n, p.pref, out);
        gsync(g);   // R is reused
    };
    if (mode & PRE_DENS) {
        // line (ky, kz) of R: component i adds its line (ky - iy, kz - iz) of q'_i, shifted by ix
        const int n = L;
        for (int e = g.gl; e < (n + 1) * (n + 2) / 2; e += g.G) {
            const int ky = T.lt[tet(n) + e] & 0xff, kz = T.lt[tet(n) + e] >> 8;
            double acc[MAXLP + 1];
#pragma unroll
            for (int kx = 0; kx <= MAXLP; kx++) acc[kx] = 0.0;
            int i = 0;
            for (int ix = la; ix >= 0; ix--)
                for (int iy = la - ix; iy >= 0; iy--, i++) {
                    const int ny = ky - iy, nz = kz - (la - ix - iy);
                    if (ny < 0 || nz < 0 || ny + nz > lb) continue;
                    const double *ql = q + i * NQ + pidx(g, lb, 0, ny, nz) - ix;   // ql[kx] = q'_i[kx - ix, ny, nz]
                    const int hi = ix + lb - ny - nz;
#pragma unroll
                    for (int kx = 0; kx <= MAXLP; kx++)
                        if (kx >= ix && kx <= hi) acc[kx] += ql[kx];
                }
            double *Rl = R + pidx(g, n, 0, ky, kz);
#pragma unroll
            for (int kx = 0; kx <= MAXLP; kx++)
                if (kx <= n - ky - kz) Rl[kx] = acc[kx];
        }
        finish_pre(0);
    }
    if (mode & PRE_TAU) {
        const int n = L + 2;
        const double aab2 = 2.0 * p.aa * p.ab;
        const unsigned short *mtn = T.mt + goff(n);
        for (int k = g.gl; k < ncoef(n); k += g.G) {
            const int kx = mtn[k] & 15, ky = (mtn[k] >> 4) & 15, kz = mtn[k] >> 8;
            {
                double v = 0.0;
                int i = 0;
                for (int ix = la; ix >= 0; ix--)
                    for (int iy = la - ix; iy >= 0; iy--, i++) {
                        const double *qi = q + i * NQ;
                        const int ic[3] = {ix, iy, la - ix - iy};
                        const int n0[3] = {kx - ix, ky - iy, kz - ic[2]};   // n = k - i
                        const double q0 = pget(g, qi, lb, n0[0], n0[1], n0[2]);
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                            const double qm2 = pget(g, qi, lb, n0[0] - 2 * e0, n0[1] - 2 * e1, n0[2] - 2 * e2);
                            const double qm1 = pget(g, qi, lb, n0[0] - e0, n0[1] - e1, n0[2] - e2);
                            const double qp1 = pget(g, qi, lb, n0[0] + e0, n0[1] + e1, n0[2] + e2);
                            const double qp2 = pget(g, qi, lb, n0[0] + 2 * e0, n0[1] + 2 * e1, n0[2] + 2 * e2);
                            v += aab2 * (qm2 + s[c] * qm1) - (p.ab * ic[c] + p.aa * n0[c]) * q0 -
                                 p.ab * s[c] * ic[c] * qp1 + 0.5 * ic[c] * (n0[c] + 2) * qp2;
                        }
                    }
                R[k] = v;
            }
        }
        finish_pre(2);
    }

    // ---- post-pass ----
    if (mode & (POST_MAT | POST_TAU)) {
        const double scale = p.pref * A.dV[p.level];
        bool first = true;
        if (mode & POST_MAT) {
            grid_to_cart(L, scale, A.mom[0] + A.base[0][p.level][L] + (long long)t * ncoef_pad(L));
            shift_polys<true>(R, 1, 0, L, p.PA, g);
            const int nlq = (lb + 1) * (lb + 2) / 2, rnlq = recip16(nlq);
            for (int e = g.gl; e < nca * nlq; e += g.G) {   // q^_i[n] = R^[i + n], one line (ny, nz) of q^_i at a time
                const int i = divr(e, rnlq), l = e - i * nlq;
                const int ny = T.lt[tet(lb) + l] & 0xff, nz = T.lt[tet(lb) + l] >> 8;
                int ix, iy, iz;
                comp_of(la, i, ix, iy, iz);
                double *ql = q + i * NQ + pidx(g, lb, 0, ny, nz);
                const double *Rl = R + pidx(g, L, ix, iy + ny, iz + nz);
                for (int nx = 0; nx <= lb - ny - nz; nx++) ql[nx] = Rl[nx];
            }
            first = false;
            gsync(g);   // R is reused
        }
        if (mode & POST_TAU) {
            const int n = L + 2;
            grid_to_cart(n, scale, A.mom[2] + A.base[2][p.level][L] + (long long)t * ncoef_pad(n));
            shift_polys<true>(R, 1, 0, n, p.PA, g);
            const double aab2 = 2.0 * p.aa * p.ab;
            for (int e = g.gl; e < nca * nq; e += g.G) {
                const int i = divr(e, rnq), k = e - i * nq;
                int ic[3];
                comp_of(la, i, ic[0], ic[1], ic[2]);
                const int mk = T.mt[goff(lb) + k];
                const int nn[3] = {mk & 15, (mk >> 4) & 15, mk >> 8};
                const int m0[3] = {ic[0] + nn[0], ic[1] + nn[1], ic[2] + nn[2]};   // i + n
                const double r0 = pget(g, R, n, m0[0], m0[1], m0[2]);
                double v = 0.0;
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                    const double rp2 = pget(g, R, n, m0[0] + 2 * e0, m0[1] + 2 * e1, m0[2] + 2 * e2);
                    const double rp1 = pget(g, R, n, m0[0] + e0, m0[1] + e1, m0[2] + e2);
                    const double rm1 = pget(g, R, n, m0[0] - e0, m0[1] - e1, m0[2] - e2);
                    const double rm2 = pget(g, R, n, m0[0] - 2 * e0, m0[1] - 2 * e1, m0[2] - 2 * e2);
                    v += aab2 * (rp2 + s[c] * rp1) - (p.ab * ic[c] + p.aa * nn[c]) * r0 - p.ab * s[c] * ic[c] * rm1 +
                         0.5 * ic[c] * nn[c] * rm2;
                }
                if (first) q[i * NQ + k] = v;
                else q[i * NQ + k] += v;
            }
            gsync(g);
        }
        shift_polys<true>(q, nca, NQ, lb, s, g);
        for (int e = g.gl; e < nca * ncb; e += g.G) {
            const int i = divr(e, rncb), j = e - i * ncb;
            int jx, jy, jz;
            comp_of(lb, j, jx, jy, jz);
            const double x = q[i * NQ + pidx(g, lb, jx, jy, jz)];
            add_to(A.F + (size_t)(p.ao_a + i) * A.nao + p.ao_b + j, x);
            if (p.sym) add_to(A.F + (size_t)(p.ao_b + j) * A.nao + p.ao_a + i, x);
        }
    }
    if (mode & POST_GRAD) {
        const int n = L + 1;
        grid_to_cart(n, p.pref * A.dV[p.level], A.mom[1] + A.base[1][p.level][L] + (long long)t * ncoef_pad(n));
        shift_polys<true>(R, 1, 0, n, p.PA, g);
        double gA[3] = {0.0, 0.0, 0.0}, gB[3] = {0.0, 0.0, 0.0};
        for (int e = g.gl; e < nca * nq; e += g.G) {
            const int i = divr(e, rnq), k = e - i * nq;
            int ic[3];
            comp_of(la, i, ic[0], ic[1], ic[2]);
            const int mk = T.mt[goff(lb) + k];
            const int nn[3] = {mk & 15, (mk >> 4) & 15, mk >> 8};
            const double qv = q[i * NQ + k];
            const int m0[3] = {ic[0] + nn[0], ic[1] + nn[1], ic[2] + nn[2]};
            const double r0 = pget(g, R, n, m0[0], m0[1], m0[2]);
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                const double rp1 = pget(g, R, n, m0[0] + e0, m0[1] + e1, m0[2] + e2);
                const double rm1 = pget(g, R, n, m0[0] - e0, m0[1] - e1, m0[2] - e2);
                gA[c] -= qv * (ic[c] * rm1 - 2.0 * p.aa * rp1);
                gB[c] -= qv * (nn[c] * rm1 - 2.0 * p.ab * (rp1 + s[c] * r0));
            }
        }
#pragma unroll
        for (int c = 0; c < 3; c++) {
            gA[c] = gsum(gA[c], g);
            gB[c] = gsum(gB[c], g);
        }
        if (g.gl == 0) {
#pragma unroll
            for (int c = 0; c < 3; c++) {
                add_to(A.grad + 3 * (size_t)p.atom_a + c, gA[c]);
                add_to(A.grad + 3 * (size_t)p.atom_b + c, gB[c]);
            }
        }
    }
}

}  // namespace pp
}  // namespace gpw
