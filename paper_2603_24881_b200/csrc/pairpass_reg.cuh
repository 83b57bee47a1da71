// Register form of the density pre-pass and the Fock post-pass (degree offset 0, the hot path): one thread per pair,
// everything unrolled over the compile-time class (la, lb), so that every polynomial coefficient has a register of
// its own and no index is computed at run time.  Same five steps as pairpass.cuh (which keeps the general,
// group-cooperative form for the derivative variants of degree L + 1 and L + 2, whose 120 / 165 coefficients do not
// fit one thread's registers):
//   q_i(Z) = sum_j D_ij Z^j  ->  Taylor shift by s = PB - PA  ->  R(Y) += Y^i q'_i(Y)  ->  Taylor shift by PA  ->  S_d
// (Eq. 26-27, one axis at a time), and the exact transpose for the moments.
#pragma once
#include <utility>

#include "gpw_math.cuh"
#include "pairpass.cuh"

namespace gpw {
namespace ppr {

// Cartesian component i of a shell (decreasing lx, then decreasing ly), usable in constant expressions
GPW_HD constexpr int comp_x(int l, int i) {
    int n = 0;
    for (int x = l; x >= 0; x--)
        for (int y = l - x; y >= 0; y--, n++)
            if (n == i) return x;
    return 0;
}
GPW_HD constexpr int comp_y(int l, int i) {
    int n = 0;
    for (int x = l; x >= 0; x--)
        for (int y = l - x; y >= 0; y--, n++)
            if (n == i) return y;
    return 0;
}

// Taylor shift c(x) -> c(x + s) of a polynomial of total degree <= N held in c[cidx(N, ...)], one axis at a time;
// TRANS: the transpose (moments of x^k -> moments of (x + s)^k).
template <int N, bool TRANS>
GPW_HD void shift3(double *c, double sx, double sy, double sz) {
#pragma unroll
    for (int axis = 0; axis < 3; axis++) {
        const double s = axis == 0 ? sx : (axis == 1 ? sy : sz);
#pragma unroll
        for (int b = 0; b <= N; b++)
#pragma unroll
            for (int a = 0; a <= N - b; a++) {
                const int m = N - a - b + 1;   // entries of the line with the other two exponents (a, b)
                auto at = [&](int j) { return axis == 0 ? cidx(N, j, a, b) : (axis == 1 ? cidx(N, a, j, b) : cidx(N, a, b, j)); };
                if (!TRANS) {
#pragma unroll
                    for (int i = 0; i < m - 1; i++)
#pragma unroll
                        for (int j = m - 2; j >= i; j--) c[at(j)] = fma(s, c[at(j + 1)], c[at(j)]);
                } else {
#pragma unroll
                    for (int i = m - 2; i >= 0; i--)
#pragma unroll
                        for (int j = i; j < m - 1; j++) c[at(j + 1)] = fma(s, c[at(j)], c[at(j + 1)]);
                }
            }
    }
}

// out[cidx(L, k_u)] = scale sum_col S_d[row k_u][col] R[col]   (HDIAG: S_d is diagonal)
template <int L, bool HDIAG>
GPW_HD void cart_to_grid(const double *R, const double *__restrict__ S, double scale, double *__restrict__ out) {
#pragma unroll
    for (int d = 0; d <= L; d++) {
        const int nd = (d + 1) * (d + 2) / 2;
        const double *Sd = S + s_block_off(d);
        int row = 0;
#pragma unroll
        for (int a = d; a >= 0; a--)
#pragma unroll
            for (int b = d - a; b >= 0; b--, row++) {
                double v = 0.0;
                if (HDIAG) v = Sd[row * nd + row] * R[cidx(L, a, b, d - a - b)];
                else {
                    int col = 0;
#pragma unroll
                    for (int a2 = d; a2 >= 0; a2--)
#pragma unroll
                        for (int b2 = d - a2; b2 >= 0; b2--, col++) v = fma(Sd[row * nd + col], R[cidx(L, a2, b2, d - a2 - b2)], v);
                }
                out[cidx(L, a, b, d - a - b)] = scale * v;
            }
    }
}
// R[col] = scale sum_row S_d[row][col] m[cidx(L, row)]
template <int L, bool HDIAG>
GPW_HD void grid_to_cart(const double *__restrict__ m, const double *__restrict__ S, double scale, double *R) {
    double mv[ncoef(L)];
#pragma unroll
    for (int k = 0; k < ncoef(L); k++) mv[k] = m[k];
#pragma unroll
    for (int d = 0; d <= L; d++) {
        const int nd = (d + 1) * (d + 2) / 2;
        const double *Sd = S + s_block_off(d);
        int col = 0;
#pragma unroll
        for (int a = d; a >= 0; a--)
#pragma unroll
            for (int b = d - a; b >= 0; b--, col++) {
                double v = 0.0;
                if (HDIAG) v = Sd[col * nd + col] * mv[cidx(L, a, b, d - a - b)];
                else {
                    int row = 0;
#pragma unroll
                    for (int a2 = d; a2 >= 0; a2--)
#pragma unroll
                        for (int b2 = d - a2; b2 >= 0; b2--, row++) v = fma(Sd[row * nd + col], mv[cidx(L, a2, b2, d - a2 - b2)], v);
                }
                R[cidx(L, a, b, d - a - b)] = scale * v;
            }
    }
}

// One component i of shell a (a compile-time index: the loop over i is expanded as a pack, because the compiler does
// not unroll a loop with a body of this size on a pragma alone and the polynomial would drop into local memory).
template <int LA, int LB, int I>
GPW_HD void pre_component(const TaskP &p, const double *__restrict__ D, int nao, double sx, double sy, double sz, double *R) {
    constexpr int L = LA + LB, NCB = ncart(LB);
    constexpr int ix = comp_x(LA, I), iy = comp_y(LA, I), iz = LA - ix - iy;
    double q[ncoef(LB)];
#pragma unroll
    for (int k = 0; k < ncoef(LB); k++) q[k] = 0.0;
    const double *row = D + (size_t)(p.ao_a + I) * nao + p.ao_b;
#pragma unroll
    for (int j = 0; j < NCB; j++) {
        const int jx = comp_x(LB, j), jy = comp_y(LB, j);
        double d = row[j];
        if (p.sym) d += D[(size_t)(p.ao_b + j) * nao + p.ao_a + I];
        q[cidx(LB, jx, jy, LB - jx - jy)] = d;
    }
    shift3<LB, false>(q, sx, sy, sz);
#pragma unroll
    for (int nz = 0; nz <= LB; nz++)
#pragma unroll
        for (int ny = 0; ny <= LB - nz; ny++)
#pragma unroll
            for (int nx = 0; nx <= LB - nz - ny; nx++) R[cidx(L, nx + ix, ny + iy, nz + iz)] += q[cidx(LB, nx, ny, nz)];
}
template <int LA, int LB, int... I>
GPW_HD void pre_components(const TaskP &p, const double *__restrict__ D, int nao, double sx, double sy, double sz, double *R,
                           std::integer_sequence<int, I...>) {
    (pre_component<LA, LB, I>(p, D, nao, sx, sy, sz, R), ...);
}

// Pre-pass of one pair of class (LA, LB): block of D -> polynomial in grid-index coordinates.
template <int LA, int LB, bool HDIAG>
GPW_HD void pre_dens(const TaskP &p, const double *__restrict__ D, int nao, const double *__restrict__ S, double *__restrict__ out) {
    constexpr int L = LA + LB;
    const double sx = p.PB[0] - p.PA[0], sy = p.PB[1] - p.PA[1], sz = p.PB[2] - p.PA[2];
    double R[ncoef(L)];
#pragma unroll
    for (int k = 0; k < ncoef(L); k++) R[k] = 0.0;
    pre_components<LA, LB>(p, D, nao, sx, sy, sz, R, std::make_integer_sequence<int, ncart(LA)>{});
    shift3<L, false>(R, p.PA[0], p.PA[1], p.PA[2]);
    cart_to_grid<L, HDIAG>(R, S, p.pref, out);
}

template <int LA, int LB, int I>
GPW_HD void post_component(const TaskP &p, double sx, double sy, double sz, const double *R, double *F, int nao) {
    constexpr int L = LA + LB, NCB = ncart(LB);
    constexpr int ix = comp_x(LA, I), iy = comp_y(LA, I), iz = LA - ix - iy;
    double q[ncoef(LB)];
#pragma unroll
    for (int nz = 0; nz <= LB; nz++)
#pragma unroll
        for (int ny = 0; ny <= LB - nz; ny++)
#pragma unroll
            for (int nx = 0; nx <= LB - nz - ny; nx++) q[cidx(LB, nx, ny, nz)] = R[cidx(L, nx + ix, ny + iy, nz + iz)];
    shift3<LB, true>(q, sx, sy, sz);
#pragma unroll
    for (int j = 0; j < NCB; j++) {
        const int jx = comp_x(LB, j), jy = comp_y(LB, j);
        const double x = q[cidx(LB, jx, jy, LB - jx - jy)];
        pp::add_to(F + (size_t)(p.ao_a + I) * nao + p.ao_b + j, x);
        if (p.sym) pp::add_to(F + (size_t)(p.ao_b + j) * nao + p.ao_a + I, x);
    }
}
template <int LA, int LB, int... I>
GPW_HD void post_components(const TaskP &p, double sx, double sy, double sz, const double *R, double *F, int nao,
                            std::integer_sequence<int, I...>) {
    (post_component<LA, LB, I>(p, sx, sy, sz, R, F, nao), ...);
}

// Post-pass of one pair: moments (grid-index coordinates) -> block of F, added atomically (mirrored for sym).
template <int LA, int LB, bool HDIAG>
GPW_HD void post_mat(const TaskP &p, const double *__restrict__ m, const double *__restrict__ S, double scale, double *F, int nao) {
    constexpr int L = LA + LB;
    const double sx = p.PB[0] - p.PA[0], sy = p.PB[1] - p.PA[1], sz = p.PB[2] - p.PA[2];
    double R[ncoef(L)];
    grid_to_cart<L, HDIAG>(m, S, scale, R);
    shift3<L, true>(R, p.PA[0], p.PA[1], p.PA[2]);
    post_components<LA, LB>(p, sx, sy, sz, R, F, nao, std::make_integer_sequence<int, ncart(LA)>{});
}

}  // namespace ppr
}  // namespace gpw
