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

struct Grp {
    int gl;          // lane within the group
    int G;           // lanes in the group (PP_G on the device, 1 on the host)
    unsigned mask;   // the group's lanes
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
// position of x^kx y^ky z^kz in a polynomial of total degree <= n: kz-major, then ky, then kx (= cidx of gpw_math.cuh)
PP_HD int pidx(int n, int kx, int ky, int kz) {
    return tet(n + 1) - tet(n + 1 - kz) + ky * (n - kz + 1) - ky * (ky - 1) / 2 + kx;
}
// coefficient (kx,ky,kz) of a polynomial of degree <= n, zero outside its support
PP_HD double pget(const double *p, int n, int kx, int ky, int kz) {
    return (kx < 0 || ky < 0 || kz < 0 || kx + ky + kz > n) ? 0.0 : p[pidx(n, kx, ky, kz)];
}
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
PP_HD void shift_line(double *p, int n, int axis, int a, int b, double s) {
    const int m = n - a - b + 1;   // entries of the line
    double c[NMAX + 1];
    int ad[NMAX + 1];
    // addresses along the line, by differences of pidx: x: 1;  y: (n - kz + 1) - ky;  z: tri(n + 1 - kz) - ky
    ad[0] = axis == 0 ? pidx(n, 0, a, b) : (axis == 1 ? pidx(n, a, 0, b) : pidx(n, a, b, 0));
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
        for (int e = g.gl; e < npoly * nl; e += g.G) {
            const int ip = e / nl;
            int a = e - ip * nl, b = 0;
            while (a >= n - b) { a -= n - b; b++; }
            double *q = p + ip * stride;
            if (n <= 3) shift_line<3, TRANS>(q, n, axis, a, b, s[axis]);
            else if (n <= 6) shift_line<6, TRANS>(q, n, axis, a, b, s[axis]);
            else shift_line<MAXDEG, TRANS>(q, n, axis, a, b, s[axis]);
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
    auto cart_to_grid = [&](int n, double scale, double *out) {   // out[k_u] = scale sum_col S[row k_u][col] R[col]
        const int n1 = n + 1;
        for (int e = g.gl; e < n1 * n1; e += g.G) {
            const int ky = e % n1, kz = e / n1;
            for (int kx = 0; kx <= n - ky - kz; kx++) {
                const int d = kx + ky + kz, nd = (d + 1) * (d + 2) / 2;
                const double *Sd = S + sblock(d);
                const int row = gidx_in_block(kx, ky, d);
                double v;
                if (A.hdiag) v = Sd[row * nd + row] * R[pidx(n, kx, ky, kz)];
                else {
                    v = 0.0;
                    int col = 0;
                    for (int a = d; a >= 0; a--)
                        for (int b = d - a; b >= 0; b--, col++) v = fma(Sd[row * nd + col], R[pidx(n, a, b, d - a - b)], v);
                }
                out[pidx(n, kx, ky, kz)] = scale * v;
            }
        }
    };
    auto grid_to_cart = [&](int n, double scale, const double *m) {   // R[col] = scale sum_row S[row][col] m[row]
        const int n1 = n + 1;
        for (int e = g.gl; e < n1 * n1; e += g.G) {
            const int ky = e % n1, kz = e / n1;
            for (int kx = 0; kx <= n - ky - kz; kx++) {
                const int d = kx + ky + kz, nd = (d + 1) * (d + 2) / 2;
                const double *Sd = S + sblock(d);
                const int col = gidx_in_block(kx, ky, d);
                double v;
                if (A.hdiag) v = Sd[col * nd + col] * m[pidx(n, kx, ky, kz)];
                else {
                    v = 0.0;
                    int row = 0;
                    for (int a = d; a >= 0; a--)
                        for (int b = d - a; b >= 0; b--, row++) v = fma(Sd[row * nd + col], m[pidx(n, a, b, d - a - b)], v);
                }
                R[pidx(n, kx, ky, kz)] = scale * v;
            }
        }
        gsync(g);
    };

    // ---- steps 1-2 (pre-pass, gradient): q'_i(Y) from the D block ----
    if (mode & (PRE_DENS | PRE_TAU | POST_GRAD)) {
        for (int e = g.gl; e < nca * NQ; e += g.G) q[e] = 0.0;
        gsync(g);
        for (int e = g.gl; e < nca * ncb; e += g.G) {
            const int i = e / ncb, j = e - i * ncb;
            int jx, jy, jz;
            comp_of(lb, j, jx, jy, jz);
            double d = A.D[(size_t)(p.ao_a + i) * A.nao + p.ao_b + j];
            if (p.sym) d += A.D[(size_t)(p.ao_b + j) * A.nao + p.ao_a + i];
            q[i * NQ + pidx(lb, jx, jy, jz)] = d;
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
        const int n = L, n1 = n + 1;
        for (int e = g.gl; e < n1 * n1; e += g.G) {
            const int ky = e % n1, kz = e / n1;
            if (ky + kz > n) continue;
            double acc[MAXLP + 1];
#pragma unroll
            for (int kx = 0; kx <= MAXLP; kx++) acc[kx] = 0.0;
            int i = 0;
            for (int ix = la; ix >= 0; ix--)
                for (int iy = la - ix; iy >= 0; iy--, i++) {
                    const int ny = ky - iy, nz = kz - (la - ix - iy);
                    if (ny < 0 || nz < 0 || ny + nz > lb) continue;
                    const double *ql = q + i * NQ + pidx(lb, 0, ny, nz) - ix;   // ql[kx] = q'_i[kx - ix, ny, nz]
                    const int hi = ix + lb - ny - nz;
#pragma unroll
                    for (int kx = 0; kx <= MAXLP; kx++)
                        if (kx >= ix && kx <= hi) acc[kx] += ql[kx];
                }
            double *Rl = R + pidx(n, 0, ky, kz);
#pragma unroll
            for (int kx = 0; kx <= MAXLP; kx++)
                if (kx <= n - ky - kz) Rl[kx] = acc[kx];
        }
        finish_pre(0);
    }
    if (mode & PRE_TAU) {
        const int n = L + 2, n1 = n + 1;
        const double aab2 = 2.0 * p.aa * p.ab;
        for (int e = g.gl; e < n1 * n1; e += g.G) {
            const int ky = e % n1, kz = e / n1;
            for (int kx = 0; kx <= n - ky - kz; kx++) {
                double v = 0.0;
                int i = 0;
                for (int ix = la; ix >= 0; ix--)
                    for (int iy = la - ix; iy >= 0; iy--, i++) {
                        const double *qi = q + i * NQ;
                        const int ic[3] = {ix, iy, la - ix - iy};
                        const int n0[3] = {kx - ix, ky - iy, kz - ic[2]};   // n = k - i
                        const double q0 = pget(qi, lb, n0[0], n0[1], n0[2]);
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                            const double qm2 = pget(qi, lb, n0[0] - 2 * e0, n0[1] - 2 * e1, n0[2] - 2 * e2);
                            const double qm1 = pget(qi, lb, n0[0] - e0, n0[1] - e1, n0[2] - e2);
                            const double qp1 = pget(qi, lb, n0[0] + e0, n0[1] + e1, n0[2] + e2);
                            const double qp2 = pget(qi, lb, n0[0] + 2 * e0, n0[1] + 2 * e1, n0[2] + 2 * e2);
                            v += aab2 * (qm2 + s[c] * qm1) - (p.ab * ic[c] + p.aa * n0[c]) * q0 -
                                 p.ab * s[c] * ic[c] * qp1 + 0.5 * ic[c] * (n0[c] + 2) * qp2;
                        }
                    }
                R[pidx(n, kx, ky, kz)] = v;
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
            const int lb1 = lb + 1;
            for (int e = g.gl; e < nca * lb1 * lb1; e += g.G) {   // q^_i[n] = R^[i + n], one line (ny, nz) of q^_i at a time
                const int i = e / (lb1 * lb1), l = e - i * lb1 * lb1;
                const int ny = l % lb1, nz = l / lb1;
                if (ny + nz > lb) continue;
                int ix, iy, iz;
                comp_of(la, i, ix, iy, iz);
                double *ql = q + i * NQ + pidx(lb, 0, ny, nz);
                const double *Rl = R + pidx(L, ix, iy + ny, iz + nz);
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
                const int i = e / nq, k = e - i * nq;
                int ic[3];
                comp_of(la, i, ic[0], ic[1], ic[2]);
                int nn[3] = {0, 0, 0}, cnt = 0;
                for (int z = 0; z <= lb; z++)
                    for (int y = 0; y <= lb - z; y++)
                        for (int x = 0; x <= lb - z - y; x++, cnt++)
                            if (cnt == k) { nn[0] = x; nn[1] = y; nn[2] = z; }
                const int m0[3] = {ic[0] + nn[0], ic[1] + nn[1], ic[2] + nn[2]};   // i + n
                const double r0 = pget(R, n, m0[0], m0[1], m0[2]);
                double v = 0.0;
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                    const double rp2 = pget(R, n, m0[0] + 2 * e0, m0[1] + 2 * e1, m0[2] + 2 * e2);
                    const double rp1 = pget(R, n, m0[0] + e0, m0[1] + e1, m0[2] + e2);
                    const double rm1 = pget(R, n, m0[0] - e0, m0[1] - e1, m0[2] - e2);
                    const double rm2 = pget(R, n, m0[0] - 2 * e0, m0[1] - 2 * e1, m0[2] - 2 * e2);
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
            const int i = e / ncb, j = e - i * ncb;
            int jx, jy, jz;
            comp_of(lb, j, jx, jy, jz);
            const double x = q[i * NQ + pidx(lb, jx, jy, jz)];
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
            const int i = e / nq, k = e - i * nq;
            int ic[3];
            comp_of(la, i, ic[0], ic[1], ic[2]);
            int nn[3] = {0, 0, 0}, cnt = 0;
            for (int z = 0; z <= lb; z++)
                for (int y = 0; y <= lb - z; y++)
                    for (int x = 0; x <= lb - z - y; x++, cnt++)
                        if (cnt == k) { nn[0] = x; nn[1] = y; nn[2] = z; }
            const double qv = q[i * NQ + k];
            const int m0[3] = {ic[0] + nn[0], ic[1] + nn[1], ic[2] + nn[2]};
            const double r0 = pget(R, n, m0[0], m0[1], m0[2]);
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const int e0 = c == 0, e1 = c == 1, e2 = c == 2;
                const double rp1 = pget(R, n, m0[0] + e0, m0[1] + e1, m0[2] + e2);
                const double rm1 = pget(R, n, m0[0] - e0, m0[1] - e1, m0[2] - e2);
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
