// oracle_bp.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle.cpp header).
//
// Backprojection: the two definitions (B_exact, B_lin) and the step-by-step
// Fourier-gridding algorithm (S5 gridding, S6 2D inverse FFT, S7 deapodise+crop),
// plus literal transposes used by the adjoint pin P8.
//
// Geometry (reading Q9): pixel (ix, iy) is at x = ix - n/2, y = iy - n/2; a ray at
// angle theta through (x, y) hits detector coordinate s = x cos + y sin + c.
// theta is float32 radians; cos/sin are taken in double from the float32 value.
// Angular quadrature weight is pi / nproj (inside C of S4, and explicit in B_lin).

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {

void orc_fft(const cplx* x, cplx* X, int N, int sign);
void orc_neglog(const uint16_t*, const float*, const float*, int, int, int, double*);
void orc_filter_rows(const double*, int, int, int, double*);
void orc_filter_rows_pad(const double*, int, int, int, int, double*);
void orc_spectrum(const double*, int, int, double, cplx*);
void orc_spectrum_fused(const double*, int, int, double, int, int, cplx*);

// Gaussian gridding kernel phi(t) = exp(-alpha t^2), alpha = pi / (sqrt(2) m)   (reading Q7),
// and its continuous transform  Phi^(x) = sqrt(pi/alpha) exp(-pi^2 x^2 / (alpha M^2))  (Q8).
static inline double kernel_alpha(int m) { return PI / (std::sqrt(2.0) * (double)m); }
double orc_kernel_alpha(int m) { return kernel_alpha(m); }

// The (phi, Phi^) pair as one switch, so that a narrower kernel can be swapped in "in both implementations at once"
// (reading Q21).  The kernel argument of every function below is a CODE:
//   m            (1..15)   Gaussian of half-width m, exactly the arithmetic above (unchanged);
//   16 + m                 Kaiser-Bessel window of half-width m (the textbook gridding kernel of the NUFFT literature the
//                          paper's Fourier method cites):
//                            phi(t)  = I0(beta sqrt(1 - (t/m)^2)) / I0(beta)  for |t| < m, else 0,
//                            Phi^(x) = (2m / I0(beta)) sinh(z) / z,  z = sqrt(beta^2 - (2 pi m x / M)^2)   (its exact transform),
//                            beta    = pi sqrt((2m/sigma)^2 (sigma - 1/2)^2 - 0.8),  sigma = 2 the oversampling (Beatty et al. 2005).
static inline int k_half(int code) { return code & 15; }
static inline bool k_is_kb(int code) { return (code >> 4) == 1; }
static inline double kb_beta(int m) { return PI * std::sqrt((double)m * (double)m * 2.25 - 0.8); }
// modified Bessel function of order 0 by its power series sum ((z/2)^2)^k / (k!)^2 (all terms positive: no cancellation)
static double bessel_i0(double z) {
    const double q = 0.25 * z * z;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 200; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    return sum;
}
static double k_phi(int code, double t) {                 // interpolation weight at distance t, zero outside the open box
    const int m = k_half(code);
    if (!(std::fabs(t) < (double)m)) return 0.0;
    if (!k_is_kb(code)) return std::exp(-kernel_alpha(m) * t * t);
    const double beta = kb_beta(m), u = 1.0 - (t / (double)m) * (t / (double)m);
    return bessel_i0(beta * std::sqrt(u > 0.0 ? u : 0.0)) / bessel_i0(beta);
}
static double k_phihat(int code, double x, int M) {       // continuous transform of phi at frequency x / M cycles per cell
    const int m = k_half(code);
    if (!k_is_kb(code)) {
        const double alpha = kernel_alpha(m);
        return std::sqrt(PI / alpha) * std::exp(-PI * PI * x * x / (alpha * (double)M * (double)M));
    }
    const double beta = kb_beta(m), a = 2.0 * PI * (double)m * x / (double)M, z2 = beta * beta - a * a;
    const double z = std::sqrt(std::fabs(z2));
    const double sh = z2 > 0.0 ? (z < 1e-8 ? 1.0 : std::sinh(z) / z) : (z < 1e-8 ? 1.0 : std::sin(z) / z);
    return 2.0 * (double)m * sh / bessel_i0(beta);
}
double orc_kernel_phi(int code, double t) { return k_phi(code, t); }
double orc_kernel_phihat(int code, double x, int M) { return k_phihat(code, x, M); }
double orc_bessel_i0(double z) { return bessel_i0(z); }

// ---------------------------------------------------------------------------
// B_exact: the sum that gridding approximates (adjoint type-1 non-uniform DFT):
//   f[iy][ix] = Re sum_j sum_k G[j][k] exp(2 pi i (k/M) (x cos_j + y sin_j)),  k signed.
// Equals (pi/nproj) sum_j q~_j(s): line summation with exact trigonometric
// interpolation of the filtered row.  O(n^2 nproj M); small n only.
// Complex output (fre, fim) so packed slice pairs can be checked; fim may be NULL.
// ---------------------------------------------------------------------------
void orc_backproject_exact(const cplx* G, const float* theta, int nproj, int n,
                           double* fre, double* fim) {
    const int M = 2 * n;
    std::vector<double> cs(nproj), sn(nproj);
    for (int j = 0; j < nproj; ++j) { cs[j] = std::cos((double)theta[j]); sn[j] = std::sin((double)theta[j]); }
#pragma omp parallel for schedule(dynamic, 1)
    for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
            double x = ix - n / 2, y = iy - n / 2;
            cplx acc = 0.0;
            for (int j = 0; j < nproj; ++j) {
                double t = (x * cs[j] + y * sn[j]) / (double)M;
                for (int k = 0; k < M; ++k) {
                    int ks = (k < M / 2) ? k : k - M;
                    double a = 2.0 * PI * (double)ks * t;
                    acc += G[(size_t)j * M + k] * cplx(std::cos(a), std::sin(a));
                }
            }
            fre[(size_t)iy * n + ix] = acc.real();
            if (fim) fim[(size_t)iy * n + ix] = acc.imag();
        }
}

// ---------------------------------------------------------------------------
// B_lin: "direct discretization of the backprojection line integral" with linear
// interpolation (the paper's LineRec):
//   f = (pi/nproj) sum_j [(1-w) q_j[i0] + w q_j[i0+1]],  s = x cos + y sin + c,
//   i0 = floor(s), w = s - i0, q_j[i] = 0 outside [0, n).
// ---------------------------------------------------------------------------
void orc_backproject_lin(const double* q, const float* theta, int nproj, int n, double center,
                         double* f) {
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
            double x = ix - n / 2, y = iy - n / 2, acc = 0.0;
            for (int j = 0; j < nproj; ++j) {
                double s = x * std::cos((double)theta[j]) + y * std::sin((double)theta[j]) + center;
                double fl = std::floor(s);
                long i0 = (long)fl;
                double w = s - fl;
                double q0 = (i0 >= 0 && i0 < n) ? q[(size_t)j * n + i0] : 0.0;
                double q1 = (i0 + 1 >= 0 && i0 + 1 < n) ? q[(size_t)j * n + i0 + 1] : 0.0;
                acc += (1.0 - w) * q0 + w * q1;
            }
            f[(size_t)iy * n + ix] = acc * PI / (double)nproj;
        }
}

// Literal transpose of B_lin (pixel-driven linear splat), for the adjoint pin P8:
//   (R_lin f)[j][i] = (pi/nproj) sum_pixels f * ((1-w)[i == i0] + w[i == i0+1]).
void orc_project_lin_adjoint(const double* f, const float* theta, int nproj, int n, double center,
                             double* q) {
    std::memset(q, 0, sizeof(double) * (size_t)nproj * n);
    for (int j = 0; j < nproj; ++j)
        for (int iy = 0; iy < n; ++iy)
            for (int ix = 0; ix < n; ++ix) {
                double x = ix - n / 2, y = iy - n / 2;
                double s = x * std::cos((double)theta[j]) + y * std::sin((double)theta[j]) + center;
                double fl = std::floor(s);
                long i0 = (long)fl;
                double w = s - fl, v = f[(size_t)iy * n + ix] * PI / (double)nproj;
                if (i0 >= 0 && i0 < n) q[(size_t)j * n + i0] += (1.0 - w) * v;
                if (i0 + 1 >= 0 && i0 + 1 < n) q[(size_t)j * n + i0 + 1] += w * v;
            }
}

// ---------------------------------------------------------------------------
// S5: polar-to-Cartesian gridding on the 2x oversampled grid.
// For every (j, k): nu = (k cos_j, k sin_j) in grid cells.  Per axis d:
//   taps are the integers l with |l - nu_d| < m  (open box: 2m taps, 2m-1 when nu_d is an
//   integer -- the symmetric choice keeps F Hermitian for real data, so the image is exactly
//   real and two slices can ride one complex transform; reading Q7);  w_d = phi(l - nu_d).
//   F[l2 mod M][l1 mod M] += G[j][k] w_1 w_2          (box truncation, periodic wrap)
// G[nproj][M] (FFT order) -> F[M][M] (FFT order, row index = l2).
// ---------------------------------------------------------------------------
static inline int wrap(long l, int M) { long r = l % M; return (int)(r < 0 ? r + M : r); }

void orc_grid(const cplx* G, const float* theta, int nproj, int n, int code, cplx* F) {
    const int M = 2 * n, m = k_half(code);
    const double alpha = kernel_alpha(m);
    for (size_t i = 0; i < (size_t)M * M; ++i) F[i] = 0.0;
    std::vector<double> w1(2 * m), w2(2 * m);
    for (int j = 0; j < nproj; ++j) {
        double cs = std::cos((double)theta[j]), sn = std::sin((double)theta[j]);
        for (int k = 0; k < M; ++k) {
            int ks = (k < M / 2) ? k : k - M;
            double nu1 = (double)ks * cs, nu2 = (double)ks * sn;
            long l01 = (long)std::floor(nu1), l02 = (long)std::floor(nu2);
            for (int a = -m + 1; a <= m; ++a) {   // candidates floor(nu)-m+1 .. floor(nu)+m
                double t1 = (double)(l01 + a) - nu1, t2 = (double)(l02 + a) - nu2;
                if (k_is_kb(code)) {
                    w1[a + m - 1] = k_phi(code, t1);
                    w2[a + m - 1] = k_phi(code, t2);
                    continue;
                }
                w1[a + m - 1] = (std::fabs(t1) < (double)m) ? std::exp(-alpha * t1 * t1) : 0.0;
                w2[a + m - 1] = (std::fabs(t2) < (double)m) ? std::exp(-alpha * t2 * t2) : 0.0;
            }
            cplx g = G[(size_t)j * M + k];
            for (int a2 = -m + 1; a2 <= m; ++a2) {
                int r = wrap(l02 + a2, M);
                for (int a1 = -m + 1; a1 <= m; ++a1) {
                    int c = wrap(l01 + a1, M);
                    F[(size_t)r * M + c] += g * (w1[a1 + m - 1] * w2[a2 + m - 1]);
                }
            }
        }
    }
}

// Literal transpose of S5 (gather with the same weights), for P8:
//   G*[j][k] = sum_taps w_1 w_2 F[l2 mod M][l1 mod M].
void orc_grid_adjoint(const cplx* F, const float* theta, int nproj, int n, int code, cplx* G) {
    const int M = 2 * n, m = k_half(code);
    const double alpha = kernel_alpha(m);
    for (int j = 0; j < nproj; ++j) {
        double cs = std::cos((double)theta[j]), sn = std::sin((double)theta[j]);
        for (int k = 0; k < M; ++k) {
            int ks = (k < M / 2) ? k : k - M;
            double nu1 = (double)ks * cs, nu2 = (double)ks * sn;
            long l01 = (long)std::floor(nu1), l02 = (long)std::floor(nu2);
            cplx acc = 0.0;
            for (int a2 = -m + 1; a2 <= m; ++a2)
                for (int a1 = -m + 1; a1 <= m; ++a1) {
                    double t1 = (double)(l01 + a1) - nu1, t2 = (double)(l02 + a2) - nu2;
                    if (std::fabs(t1) >= (double)m || std::fabs(t2) >= (double)m) continue;
                    acc += F[(size_t)wrap(l02 + a2, M) * M + wrap(l01 + a1, M)] *
                           (k_is_kb(code) ? k_phi(code, t1) * k_phi(code, t2) : std::exp(-alpha * t1 * t1) * std::exp(-alpha * t2 * t2));
                }
            G[(size_t)j * M + k] = acc;
        }
    }
}

// ---------------------------------------------------------------------------
// S6: 2D inverse FFT, unnormalised:  g[x2][x1] = sum F[l2][l1] e^{+2 pi i (l1 x1 + l2 x2)/M},
// as 1D transforms of the rows then of the columns ("2D FFT as a combination of 1D FFTs",
// PAPER.md:300).  sign = +1 inverse, -1 forward (the forward one serves the adjoint pin).
// ---------------------------------------------------------------------------
void orc_fft2(const cplx* F, int M, int sign, cplx* g) {
    std::vector<cplx> T((size_t)M * M);
#pragma omp parallel
    {
        std::vector<cplx> a(M), b(M);
#pragma omp for schedule(static)
        for (int r = 0; r < M; ++r) orc_fft(F + (size_t)r * M, T.data() + (size_t)r * M, M, sign);
#pragma omp for schedule(static)
        for (int c = 0; c < M; ++c) {
            for (int r = 0; r < M; ++r) a[r] = T[(size_t)r * M + c];
            orc_fft(a.data(), b.data(), M, sign);
            for (int r = 0; r < M; ++r) g[(size_t)r * M + c] = b[r];
        }
    }
}

// ---------------------------------------------------------------------------
// S7: deapodise and crop ("accuracy controls"):
//   f[iy][ix] = g[y mod M][x mod M] / (Phi^(x) Phi^(y)),  x = ix - n/2, y = iy - n/2.
// Real part -> fre; imaginary part (second slice of a packed pair) -> fim if not NULL.
// ---------------------------------------------------------------------------
void orc_deapod_crop(const cplx* g, int n, int code, double* fre, double* fim) {
    const int M = 2 * n, m = k_half(code);
    const double alpha = kernel_alpha(m);
    for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
            double x = ix - n / 2, y = iy - n / 2;
            double px = std::sqrt(PI / alpha) * std::exp(-PI * PI * x * x / (alpha * (double)M * (double)M));
            double py = std::sqrt(PI / alpha) * std::exp(-PI * PI * y * y / (alpha * (double)M * (double)M));
            if (k_is_kb(code)) { px = k_phihat(code, x, M); py = k_phihat(code, y, M); }
            cplx v = g[(size_t)wrap((long)y, M) * M + wrap((long)x, M)] / (px * py);
            fre[(size_t)iy * n + ix] = v.real();
            if (fim) fim[(size_t)iy * n + ix] = v.imag();
        }
}

// Literal transpose of S7 (divide, zero-embed at (y mod M, x mod M)), for P8.
void orc_deapod_crop_adjoint(const double* fre, const double* fim, int n, int code, cplx* g) {
    const int M = 2 * n, m = k_half(code);
    const double alpha = kernel_alpha(m);
    for (size_t i = 0; i < (size_t)M * M; ++i) g[i] = 0.0;
    for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
            double x = ix - n / 2, y = iy - n / 2;
            double px = std::sqrt(PI / alpha) * std::exp(-PI * PI * x * x / (alpha * (double)M * (double)M));
            double py = std::sqrt(PI / alpha) * std::exp(-PI * PI * y * y / (alpha * (double)M * (double)M));
            if (k_is_kb(code)) { px = k_phihat(code, x, M); py = k_phihat(code, y, M); }
            cplx v(fre[(size_t)iy * n + ix], fim ? fim[(size_t)iy * n + ix] : 0.0);
            g[(size_t)wrap((long)y, M) * M + wrap((long)x, M)] = v / (px * py);
        }
}

// B_grid = S5 -> S6 -> S7 on one slice's spectrum.
void orc_backproject_grid(const cplx* G, const float* theta, int nproj, int n, int m,
                          double* fre, double* fim) {
    const int M = 2 * n;
    std::vector<cplx> F((size_t)M * M), g((size_t)M * M);
    orc_grid(G, theta, nproj, n, m, F.data());
    orc_fft2(F.data(), M, +1, g.data());
    orc_deapod_crop(g.data(), n, m, fre, fim);
}

// ---------------------------------------------------------------------------
// Whole chains, slice by slice.  method: 0 = B_grid, 1 = B_exact, 2 = B_lin.
// p[nz][nproj][n] (sinogram after -log) -> out[nz][n][n];  q_out (filtered sinogram,
// [nz][nproj][n]) is written when not NULL.  Slices are independent.
// ---------------------------------------------------------------------------
void orc_fbp_from_sino_pad(const double* p, const float* theta, int nproj, int nz, int n, double center, int filter,
                           int pad, int m, int method, double* out, double* q_out);
void orc_fbp_from_sino(const double* p, const float* theta, int nproj, int nz, int n,
                       double center, int filter, int m, int method, double* out, double* q_out) {
    orc_fbp_from_sino_pad(p, theta, nproj, nz, n, center, filter, 0, m, method, out, q_out);
}
// pad: bit 0 = padding of the filter stage (orc_filter_rows_pad): 0 zeros, 1 edge values;
//      bit 1 = S3 + S4 fused without the crop (orc_spectrum_fused; gridding / exact backprojection only)
void orc_fbp_from_sino_pad(const double* p, const float* theta, int nproj, int nz, int n, double center, int filter,
                           int pad, int m, int method, double* out, double* q_out) {
    const int M = 2 * n;
    // nested parallelism is off by default, so the inner pragmas run serially here
#pragma omp parallel for schedule(dynamic, 1) if (method != 1)
    for (int z = 0; z < nz; ++z) {
        std::vector<double> q((size_t)nproj * n);
        orc_filter_rows_pad(p + (size_t)z * nproj * n, nproj, n, filter, pad & 1, q.data());
        if (q_out) std::memcpy(q_out + (size_t)z * nproj * n, q.data(), sizeof(double) * q.size());
        double* f = out + (size_t)z * n * n;
        if (method == 2) {
            orc_backproject_lin(q.data(), theta, nproj, n, center, f);
        } else {
            std::vector<cplx> G((size_t)nproj * M);
            if (pad & 2) orc_spectrum_fused(p + (size_t)z * nproj * n, nproj, n, center, filter, pad & 1, G.data());
            else orc_spectrum(q.data(), nproj, n, center, G.data());
            if (method == 0) orc_backproject_grid(G.data(), theta, nproj, n, m, f, nullptr);
            else orc_backproject_exact(G.data(), theta, nproj, n, f, nullptr);
        }
    }
}

// raw uint16 counts -> reconstruction (S1..S7).
void orc_recon(const uint16_t* raw, const float* flat, const float* dark, const float* theta,
               int nproj, int nz, int n, double center, int filter, int m, int method, double* out) {
    std::vector<double> p((size_t)nz * nproj * n);
    orc_neglog(raw, flat, dark, nproj, nz, n, p.data());
    orc_fbp_from_sino(p.data(), theta, nproj, nz, n, center, filter, m, method, out, nullptr);
}
void orc_recon_pad(const uint16_t* raw, const float* flat, const float* dark, const float* theta, int nproj, int nz, int n,
                   double center, int filter, int pad, int m, int method, double* out) {
    std::vector<double> p((size_t)nz * nproj * n);
    orc_neglog(raw, flat, dark, nproj, nz, n, p.data());
    orc_fbp_from_sino_pad(p.data(), theta, nproj, nz, n, center, filter, pad, m, method, out, nullptr);
}

}  // extern "C"
