// Inter-level Fourier combination, Eq. (7)-(8), and the G-space operators of the Fock build on the
// finest mesh (Hartree potential Eq. 5-6, gradient Eq. 10, divergence Eq. 14): cuFFT plus pointwise kernels on the
// half spectra.  Off the optimisation target; HBM-bound.
//
//   up:   rho~(G) = sum_alpha [F(rho_alpha)](G) for |G| < G_alpha, evaluated on the finest mesh
//   down: v_alpha = F^-1 of [F(v_fine)](G) restricted to |G| < G_alpha          (the adjoint of up)
// F(f)(G_m) = (1/N_grid) sum_n f(r_n) exp(-i G_m . r_n), G_m = 2 pi sum_i m_i b_i, b_i = columns of
// inverse(cell).  G_alpha = min_i pi N_alpha,i |b_i|; Nyquist planes |m_i| = N_alpha,i/2 are dropped and a
// plane wave with |G| = G_alpha up to rounding (1e-12 relative in |G|^2) counts as ">=" (A17).
//
// Real-to-complex transforms: a level's half spectrum is [N1][N2][N3/2+1]; the kept set is inversion
// symmetric, so Hermitian symmetry survives the cut and the embedding.
#include <cufft.h>

#include <cmath>
#include <string>

#include "gpw_kernels.cuh"

namespace gpw {

struct InterpState {
    int nlevel = 0;
    cufftHandle fwd[GPW_MAX_LEVEL], inv[GPW_MAX_LEVEL];
    bool made[GPW_MAX_LEVEL] = {false};
    cufftDoubleComplex *spec_f = nullptr;   // half spectrum on the finest mesh
    cufftDoubleComplex *spec_a = nullptr;   // half spectrum of one level (sized for the finest)
    void *work = nullptr;                   // cuFFT work area shared by all plans
    size_t work_bytes = 0;
    long bytes = 0;
};

namespace {

struct SpecGeom {
    int Na[3], Nf[3];     // level mesh, finest mesh
    double M[6];          // metric of the reciprocal vectors b_i . b_j, packed 11 22 33 12 13 23
    double cut2;          // (G_alpha / 2 pi)^2 (1 - 1e-12)
    double scale;
};

__device__ __forceinline__ bool kept(const SpecGeom &g, int m1, int m2, int m3) {
    if (2 * abs(m1) >= g.Na[0] || 2 * abs(m2) >= g.Na[1] || 2 * abs(m3) >= g.Na[2]) return false;
    const double a = m1, b = m2, c = m3;
    const double g2 = g.M[0] * a * a + g.M[1] * b * b + g.M[2] * c * c + 2.0 * (g.M[3] * a * b + g.M[4] * a * c + g.M[5] * b * c);
    return g2 < g.cut2;
}

// UP = true:  spec_f[embed(m)] += scale * spec_a[m] for kept m;   UP = false:  spec_a[m] = kept ? scale * spec_f[embed(m)] : 0
template <bool UP>
__global__ void __launch_bounds__(256) k_spectrum_transfer(SpecGeom g, cufftDoubleComplex *__restrict__ spec_f,
                                                           cufftDoubleComplex *__restrict__ spec_a) {
    const int h3 = g.Na[2] / 2 + 1, hf3 = g.Nf[2] / 2 + 1;
    const long long n = (long long)g.Na[0] * g.Na[1] * h3;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int i3 = (int)(i % h3), i2 = (int)((i / h3) % g.Na[1]), i1 = (int)(i / ((long long)h3 * g.Na[1]));
        const int m1 = i1 < g.Na[0] - g.Na[0] / 2 ? i1 : i1 - g.Na[0];
        const int m2 = i2 < g.Na[1] - g.Na[1] / 2 ? i2 : i2 - g.Na[1];
        const int m3 = i3;
        const bool k = kept(g, m1, m2, m3);
        const long long jf = ((long long)(m1 < 0 ? m1 + g.Nf[0] : m1) * g.Nf[1] + (m2 < 0 ? m2 + g.Nf[1] : m2)) * hf3 + m3;
        if (UP) {
            if (k) {
                const cufftDoubleComplex a = spec_a[i];
                cufftDoubleComplex f = spec_f[jf];
                f.x += g.scale * a.x; f.y += g.scale * a.y;
                spec_f[jf] = f;
            }
        } else {
            cufftDoubleComplex o = make_cuDoubleComplex(0.0, 0.0);
            if (k) { const cufftDoubleComplex f = spec_f[jf]; o.x = g.scale * f.x; o.y = g.scale * f.y; }
            spec_a[i] = o;
        }
    }
}

bool fft_ok(cufftResult r, const char *what) {
    if (r == CUFFT_SUCCESS) return true;
    set_error(std::string(what) + ": cuFFT error " + std::to_string((int)r));
    return false;
}
bool cu_ok(cudaError_t e, const char *what) {
    if (e == cudaSuccess) return true;
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return false;
}

size_t half_count(const int *N) { return (size_t)N[0] * N[1] * (N[2] / 2 + 1); }

// plans, scratch spectra and the shared work area, created on first use
int ensure(const HostPlan *hp, InterpState **stp) {
    if (*stp) return GPW_OK;
    InterpState *s = new InterpState();
    s->nlevel = hp->nlevel;
    size_t wmax = 0;
    for (int a = 0; a < hp->nlevel; a++) {
        const int *N = hp->lev[a].N;
        for (int dir = 0; dir < 2; dir++) {
            cufftHandle *h = dir ? &s->inv[a] : &s->fwd[a];
            size_t ws = 0;
            if (!fft_ok(cufftCreate(h), "cufftCreate") || !fft_ok(cufftSetAutoAllocation(*h, 0), "cufftSetAutoAllocation") ||
                !fft_ok(cufftMakePlan3d(*h, N[0], N[1], N[2], dir ? CUFFT_Z2D : CUFFT_D2Z, &ws), "cufftMakePlan3d")) {
                interp_free(s);
                return GPW_ECUDA;
            }
            wmax = ws > wmax ? ws : wmax;
        }
        s->made[a] = true;
    }
    const size_t nb = sizeof(cufftDoubleComplex) * half_count(hp->lev[0].N);
    s->work_bytes = wmax ? wmax : 16;
    if (!cu_ok(cudaMalloc((void **)&s->spec_f, nb), "interp scratch") || !cu_ok(cudaMalloc((void **)&s->spec_a, nb), "interp scratch") ||
        !cu_ok(cudaMalloc(&s->work, s->work_bytes), "interp work area")) {
        interp_free(s);
        return GPW_ECUDA;
    }
    s->bytes = (long)(2 * nb + s->work_bytes);
    for (int a = 0; a < hp->nlevel; a++)
        if (!fft_ok(cufftSetWorkArea(s->fwd[a], s->work), "cufftSetWorkArea") ||
            !fft_ok(cufftSetWorkArea(s->inv[a], s->work), "cufftSetWorkArea")) {
            interp_free(s);
            return GPW_ECUDA;
        }
    *stp = s;
    return GPW_OK;
}

SpecGeom geom(const HostPlan *hp, int a, double scale) {
    SpecGeom g;
    const double *b = hp->binv;   // binv[c*3+i] = component c of b_i (column i of inverse(cell))
    auto dot = [&](int i, int j) { return b[0 * 3 + i] * b[0 * 3 + j] + b[1 * 3 + i] * b[1 * 3 + j] + b[2 * 3 + i] * b[2 * 3 + j]; };
    g.M[0] = dot(0, 0); g.M[1] = dot(1, 1); g.M[2] = dot(2, 2); g.M[3] = dot(0, 1); g.M[4] = dot(0, 2); g.M[5] = dot(1, 2);
    double c2 = 0.0;
    for (int i = 0; i < 3; i++) {
        g.Na[i] = hp->lev[a].N[i];
        g.Nf[i] = hp->lev[0].N[i];
        const double h = 0.5 * g.Na[i];
        const double v = h * h * g.M[i];      // (N_i |b_i| / 2)^2 = (G_alpha,i / 2 pi)^2
        c2 = (i == 0 || v < c2) ? v : c2;
    }
    g.cut2 = c2 * (1.0 - 1e-12);
    g.scale = scale;
    return g;
}

int grid_for(size_t n) { return (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8); }

// ---- G-space operators on the finest mesh (Eq. 5-6, Eq. 10, Eq. 14) ----
// G_m = 2 pi sum_i m_i b_i.  Plane waves on a Nyquist plane (|m_i| = N_i / 2) are dropped (A26): there the
// two aliases +-N_i/2 share one grid function but not one G.
struct GGeom {
    int N[3];
    double B[9];      // B[c*3+i] = 2 pi * component c of b_i
    double scale;     // 1 / N_grid (cuFFT's forward + inverse transforms multiply by N_grid)
};
enum { G_HARTREE = 0, G_GRAD = 1, G_DIV = 2 };

// HARTREE: out = 4 pi / |G|^2 in (0 at G = 0);  GRAD: out = i G_c in;  DIV: out (+)= i G_c in  (accumulate if c > 0)
template <int KIND>
__global__ void __launch_bounds__(256) k_gspace(GGeom g, int c, const cufftDoubleComplex *__restrict__ in,
                                                cufftDoubleComplex *__restrict__ out) {
    const int h3 = g.N[2] / 2 + 1;
    const long long n = (long long)g.N[0] * g.N[1] * h3;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int i3 = (int)(i % h3), i2 = (int)((i / h3) % g.N[1]), i1 = (int)(i / ((long long)h3 * g.N[1]));
        const int m1 = i1 < g.N[0] - g.N[0] / 2 ? i1 : i1 - g.N[0];
        const int m2 = i2 < g.N[1] - g.N[1] / 2 ? i2 : i2 - g.N[1];
        const int m3 = i3;
        const bool nyq = 2 * abs(m1) == g.N[0] || 2 * abs(m2) == g.N[1] || 2 * abs(m3) == g.N[2];
        double G[3];
#pragma unroll
        for (int x = 0; x < 3; x++) G[x] = g.B[x * 3 + 0] * m1 + g.B[x * 3 + 1] * m2 + g.B[x * 3 + 2] * m3;
        const cufftDoubleComplex a = in[i];
        cufftDoubleComplex o = make_cuDoubleComplex(0.0, 0.0);
        if (KIND == G_HARTREE) {
            const double g2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
            if (!nyq && g2 > 0.0) { const double k = 4.0 * M_PI / g2 * g.scale; o.x = k * a.x; o.y = k * a.y; }
        } else {
            const double Gc = c == 0 ? G[0] : (c == 1 ? G[1] : G[2]);
            if (!nyq) { const double k = Gc * g.scale; o.x = -k * a.y; o.y = k * a.x; }   // i G_c (x + i y)
            if (KIND == G_DIV && c > 0) { const cufftDoubleComplex p = out[i]; o.x += p.x; o.y += p.y; }
        }
        out[i] = o;
    }
}

GGeom ggeom(const HostPlan *hp) {
    GGeom g;
    for (int i = 0; i < 3; i++) g.N[i] = hp->lev[0].N[i];
    for (int k = 0; k < 9; k++) g.B[k] = 2.0 * M_PI * hp->binv[k];
    g.scale = 1.0 / ((double)g.N[0] * g.N[1] * g.N[2]);
    return g;
}

}  // namespace

void interp_free(InterpState *s) {
    if (!s) return;
    for (int a = 0; a < s->nlevel; a++)
        if (s->made[a]) { cufftDestroy(s->fwd[a]); cufftDestroy(s->inv[a]); }
    cudaFree(s->spec_f); cudaFree(s->spec_a); cudaFree(s->work);
    delete s;
}

long interp_bytes(const InterpState *s) { return s ? s->bytes : 0; }

int interp_up(const HostPlan *hp, InterpState **stp, const double *const *rho, int ncomp, double *fine, cudaStream_t st) {
    const int rc = ensure(hp, stp);
    if (rc != GPW_OK) return rc;
    InterpState *s = *stp;
    const int *Nf = hp->lev[0].N;
    const size_t nf = (size_t)Nf[0] * Nf[1] * Nf[2];
    for (int k = 0; k < ncomp; k++) {
        if (!cu_ok(cudaMemsetAsync(s->spec_f, 0, sizeof(cufftDoubleComplex) * half_count(Nf), st), "gpw_interp_up: memset")) return GPW_ECUDA;
        for (int a = 0; a < hp->nlevel; a++) {
            const int *N = hp->lev[a].N;
            const size_t na = (size_t)N[0] * N[1] * N[2];
            if (!fft_ok(cufftSetStream(s->fwd[a], st), "cufftSetStream") ||
                !fft_ok(cufftExecD2Z(s->fwd[a], const_cast<double *>(rho[a]) + k * na, s->spec_a), "gpw_interp_up: D2Z")) return GPW_ECUDA;
            const SpecGeom g = geom(hp, a, 1.0 / (double)na);
            k_spectrum_transfer<true><<<grid_for(half_count(N)), 256, 0, st>>>(g, s->spec_f, s->spec_a);
        }
        if (!fft_ok(cufftSetStream(s->inv[0], st), "cufftSetStream") ||
            !fft_ok(cufftExecZ2D(s->inv[0], s->spec_f, fine + k * nf), "gpw_interp_up: Z2D")) return GPW_ECUDA;
    }
    return cu_ok(cudaGetLastError(), "gpw_interp_up") ? GPW_OK : GPW_ECUDA;
}

int gspace_apply(const HostPlan *hp, InterpState **stp, int kind, const double *in, double *out, cudaStream_t st) {
    const int rc = ensure(hp, stp);
    if (rc != GPW_OK) return rc;
    InterpState *s = *stp;
    const int *Nf = hp->lev[0].N;
    const size_t nf = (size_t)Nf[0] * Nf[1] * Nf[2];
    const GGeom g = ggeom(hp);
    const int nblk = grid_for(half_count(Nf));
    if (!fft_ok(cufftSetStream(s->fwd[0], st), "cufftSetStream") || !fft_ok(cufftSetStream(s->inv[0], st), "cufftSetStream")) return GPW_ECUDA;
    if (kind == G_HARTREE) {
        if (!fft_ok(cufftExecD2Z(s->fwd[0], const_cast<double *>(in), s->spec_f), "gpw_hartree: D2Z")) return GPW_ECUDA;
        k_gspace<G_HARTREE><<<nblk, 256, 0, st>>>(g, 0, s->spec_f, s->spec_a);
        if (!fft_ok(cufftExecZ2D(s->inv[0], s->spec_a, out), "gpw_hartree: Z2D")) return GPW_ECUDA;
    } else if (kind == G_GRAD) {
        if (!fft_ok(cufftExecD2Z(s->fwd[0], const_cast<double *>(in), s->spec_f), "gpw_gspace_gradient: D2Z")) return GPW_ECUDA;
        for (int c = 0; c < 3; c++) {
            k_gspace<G_GRAD><<<nblk, 256, 0, st>>>(g, c, s->spec_f, s->spec_a);
            if (!fft_ok(cufftExecZ2D(s->inv[0], s->spec_a, out + c * nf), "gpw_gspace_gradient: Z2D")) return GPW_ECUDA;
        }
    } else {
        for (int c = 0; c < 3; c++) {
            if (!fft_ok(cufftExecD2Z(s->fwd[0], const_cast<double *>(in) + c * nf, s->spec_a), "gpw_gspace_divergence: D2Z")) return GPW_ECUDA;
            k_gspace<G_DIV><<<nblk, 256, 0, st>>>(g, c, s->spec_a, s->spec_f);
        }
        if (!fft_ok(cufftExecZ2D(s->inv[0], s->spec_f, out), "gpw_gspace_divergence: Z2D")) return GPW_ECUDA;
    }
    return cu_ok(cudaGetLastError(), "G-space operator") ? GPW_OK : GPW_ECUDA;
}

int interp_down(const HostPlan *hp, InterpState **stp, const double *fine, int ncomp, double *const *v, cudaStream_t st) {
    const int rc = ensure(hp, stp);
    if (rc != GPW_OK) return rc;
    InterpState *s = *stp;
    const int *Nf = hp->lev[0].N;
    const size_t nf = (size_t)Nf[0] * Nf[1] * Nf[2];
    for (int k = 0; k < ncomp; k++) {
        if (!fft_ok(cufftSetStream(s->fwd[0], st), "cufftSetStream") ||
            !fft_ok(cufftExecD2Z(s->fwd[0], const_cast<double *>(fine) + k * nf, s->spec_f), "gpw_restrict_down: D2Z")) return GPW_ECUDA;
        for (int a = 0; a < hp->nlevel; a++) {
            const int *N = hp->lev[a].N;
            const size_t na = (size_t)N[0] * N[1] * N[2];
            const SpecGeom g = geom(hp, a, 1.0 / (double)nf);
            k_spectrum_transfer<false><<<grid_for(half_count(N)), 256, 0, st>>>(g, s->spec_f, s->spec_a);
            if (!fft_ok(cufftSetStream(s->inv[a], st), "cufftSetStream") ||
                !fft_ok(cufftExecZ2D(s->inv[a], s->spec_a, v[a] + k * na), "gpw_restrict_down: Z2D")) return GPW_ECUDA;
        }
    }
    return cu_ok(cudaGetLastError(), "gpw_restrict_down") ? GPW_OK : GPW_ECUDA;
}

}  // namespace gpw
