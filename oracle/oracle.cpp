// oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, double-precision CPU statement of what the hot path computes:
// parallel-beam filtered backprojection by Fourier gridding (the paper's
// "FourierRec": "Fourier-based method with exponential functions for
// interpolation in the frequency domain"), plus the two
// definitions it approximates (exact band-limited line summation B_exact and
// the textbook linear-interpolation line summation B_lin = the paper's
// LineRec).  The paper prints no formula; every formula
// here is the classical definition the paper names, in the reading fixed by
// DESIGN.md ("Readings of the paper", Q1..Q17).  Stage names S1..S7 follow
// DESIGN.md / SURVEY.md 8(c).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline/reference
// arm may call this.  It shares no source, header, table or helper with the
// CUDA path under paper_2209_08450_b200/.  No blocking, fusion or reordering
// beyond what each definition states; OpenMP is used only over independent
// slices / image rows ("reconstruction is done independently for different
// slices").
//
// Pins (tests/test_oracle_pins.py): P1 closed-form -log; P2 FFT vs O(N^2) DFT
// and Parseval; P3 filter impulse responses vs closed forms; P4 plane wave;
// P5 analytic ellipsoid phantom (scale, orientation); P6 centre shift;
// P7 gridding vs exact; P8 adjoint identities; P9 slice-pair packing.
// Parity unpinned: the absolute accuracy of FBP against the rasterised phantom
// (Gibbs, finite angles) is reported, not gated.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {

// ---------------------------------------------------------------------------
// Fourier transforms.  orc_dft is the definition  X[k] = sum_i x[i] e^{sign 2 pi i k i / N};
// orc_fft is the textbook iterative radix-2 Cooley-Tukey (N a power of two) the
// chain uses; P2 pins one to the other.
// ---------------------------------------------------------------------------
void orc_dft(const cplx* x, cplx* X, int N, int sign) {
    for (int k = 0; k < N; ++k) {
        cplx acc = 0.0;
        for (int i = 0; i < N; ++i) {
            // reduce k*i mod N first so the angle stays small
            long long r = ((long long)k * i) % N;
            double a = sign * 2.0 * PI * (double)r / (double)N;
            acc += x[i] * cplx(std::cos(a), std::sin(a));
        }
        X[k] = acc;
    }
}

void orc_fft(const cplx* x, cplx* X, int N, int sign) {
    int lg = 0;
    while ((1 << lg) < N) ++lg;
    for (int i = 0; i < N; ++i) {           // bit-reversal permutation
        int r = 0;
        for (int b = 0; b < lg; ++b) if (i & (1 << b)) r |= 1 << (lg - 1 - b);
        X[r] = x[i];
    }
    for (int len = 2; len <= N; len <<= 1) {
        int half = len >> 1;
        for (int s = 0; s < N; s += len)
            for (int t = 0; t < half; ++t) {
                double a = sign * 2.0 * PI * (double)t / (double)len;
                cplx w(std::cos(a), std::sin(a));
                cplx u = X[s + t], v = w * X[s + t + half];
                X[s + t] = u + v;
                X[s + t + half] = u - v;
            }
    }
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// ---------------------------------------------------------------------------
// S1 + S2: dark/flat-field correction and negative logarithm.
//   t = (raw - dark) / max(flat - dark, eps_d);  t = max(t, t_min);  p = -ln t
// eps_d = 1e-3 counts, t_min = 1e-6 (reading Q11).  raw[nproj][nz][n] uint16,
// flat/dark[nz][n] float32 (already averaged), p[nz][nproj][n].
// ---------------------------------------------------------------------------
void orc_neglog(const uint16_t* raw, const float* flat, const float* dark,
                int nproj, int nz, int n, double* p) {
    const double eps_d = 1e-3, t_min = 1e-6;
    for (int z = 0; z < nz; ++z)
        for (int j = 0; j < nproj; ++j)
            for (int i = 0; i < n; ++i) {
                double d = (double)dark[(size_t)z * n + i];
                double f = (double)flat[(size_t)z * n + i];
                double r = (double)raw[((size_t)j * nz + z) * n + i];
                double den = f - d;
                if (den < eps_d) den = eps_d;
                double t = (r - d) / den;
                if (t < t_min) t = t_min;
                p[((size_t)z * nproj + j) * n + i] = -std::log(t);
            }
}

// ---------------------------------------------------------------------------
// Filter table H[k], k = 0..M-1 in FFT order (k >= M/2 means k - M), reading Q4.
//   H = R * W;  R = DFT_M of the band-limited ramp kernel
//       h[0] = 1/4, h[i] = -1/(pi^2 i^2) for odd i, 0 for even i != 0   (i signed, wrapped)
//   W: ramp 1; shepp sin(pi k/M)/(pi k/M); parzen with u = |k|/(M/2):
//       1 - 6u^2(1-u) for u <= 1/2, 2(1-u)^3 for u > 1/2.     H[M/2] := 0.
//   "or other filter": the textbook apodisation windows on the same u,
//       cosine cos(pi u/2), Hann (1 + cos(pi u))/2, Hamming 0.54 + 0.46 cos(pi u).
// filter: 0 ramp, 1 shepp, 2 parzen ("Shepp-Logan, Parzen or other filter"),
//         3 cosine, 4 hann, 5 hamming.
// ---------------------------------------------------------------------------
void orc_filter(int M, int filter, double* H) {
    std::vector<cplx> h(M), R(M);
    for (int i = 0; i < M; ++i) {
        int is = (i < M / 2) ? i : i - M;           // signed index, -M/2 .. M/2-1
        double v = 0.0;
        if (is == 0) v = 0.25;
        else if (is % 2 != 0) v = -1.0 / (PI * PI * (double)is * (double)is);
        h[i] = v;
    }
    orc_dft(h.data(), R.data(), M, -1);
    for (int k = 0; k < M; ++k) {
        int ks = (k < M / 2) ? k : k - M;
        double W = 1.0;
        if (filter == 1) {
            double a = PI * (double)ks / (double)M;
            W = (ks == 0) ? 1.0 : std::sin(a) / a;
        } else if (filter == 2) {
            double u = std::fabs((double)ks) / (double)(M / 2);
            W = (u <= 0.5) ? 1.0 - 6.0 * u * u * (1.0 - u) : 2.0 * (1.0 - u) * (1.0 - u) * (1.0 - u);
        } else if (filter >= 3) {
            double u = std::fabs((double)ks) / (double)(M / 2);
            if (filter == 3) W = std::cos(0.5 * PI * u);
            else if (filter == 4) W = 0.5 * (1.0 + std::cos(PI * u));
            else W = 0.54 + 0.46 * std::cos(PI * u);
        }
        H[k] = R[k].real() * W;
    }
    H[M / 2] = 0.0;
}

// ---------------------------------------------------------------------------
// S3: ramp-type filtering of each detector row by a zero-padded FFT of length
// M = 2n ("one-dimensional filtering"; padding PAPER.md:59, :173).
//   a = [p, 0];  P = FFT(a);  Q = P H;  q = IFFT(Q)/M, kept for 0 <= i < n.
// p, q: [rows][n].
// pad = 1 ("edge"; padding for "samples not fitting into the detector field
// of view"): the n padding samples repeat the nearest detector edge of the periodic length-M row,
//   a[i] = p[n-1] for n <= i < n + n/2,  a[i] = p[0] for n + n/2 <= i < M   (pad = 0: zeros, the default).
// ---------------------------------------------------------------------------
void orc_filter_rows_pad(const double* p, int rows, int n, int filter, int pad, double* q);
void orc_filter_rows(const double* p, int rows, int n, int filter, double* q) {
    orc_filter_rows_pad(p, rows, n, filter, 0, q);
}
void orc_filter_rows_pad(const double* p, int rows, int n, int filter, int pad, double* q) {
    const int M = 2 * n;
    std::vector<double> H(M);
    orc_filter(M, filter, H.data());
#pragma omp parallel
    {
        std::vector<cplx> a(M), P(M), b(M);
#pragma omp for schedule(static)
        for (int r = 0; r < rows; ++r) {
            const double* pr = p + (size_t)r * n;
            for (int i = 0; i < M; ++i) a[i] = (i < n) ? pr[i] : (pad == 0 ? 0.0 : (i < n + n / 2 ? pr[n - 1] : pr[0]));
            orc_fft(a.data(), P.data(), M, -1);
            for (int k = 0; k < M; ++k) P[k] *= H[k];
            orc_fft(P.data(), b.data(), M, +1);
            for (int i = 0; i < n; ++i) q[(size_t)r * n + i] = b[i].real() / (double)M;
        }
    }
}

// ---------------------------------------------------------------------------
// S4: spectrum of the filtered projections on the polar grid (Fourier-slice
// theorem).   b = [q, 0] (length M);  B = FFT(b);
//   G[j][k] = C B_j[k] e^{+2 pi i k c / M},  k signed,  C = pi / (nproj M),  G[j][-M/2] = 0.
// The phase moves the rotation axis (detector coordinate c) to the origin.
// q[nproj][n] -> G[nproj][M] in FFT order.
// ---------------------------------------------------------------------------
void orc_spectrum(const double* q, int nproj, int n, double center, cplx* G) {
    const int M = 2 * n;
    const double C = PI / ((double)nproj * (double)M);
    std::vector<cplx> b(M), B(M);
    for (int j = 0; j < nproj; ++j) {
        for (int i = 0; i < M; ++i) b[i] = (i < n) ? q[(size_t)j * n + i] : 0.0;
        orc_fft(b.data(), B.data(), M, -1);
        for (int k = 0; k < M; ++k) {
            int ks = (k < M / 2) ? k : k - M;
            double a = 2.0 * PI * (double)ks * center / (double)M;
            G[(size_t)j * M + k] = C * B[k] * cplx(std::cos(a), std::sin(a));
        }
        G[(size_t)j * M + M / 2] = 0.0;
    }
}


// ---------------------------------------------------------------------------
// S3 + S4 fused, WITHOUT the crop between them (SURVEY 8(c) "literal vs fused reading", Q6; an option of
// SURVEY 8(f-2), not the default): the filter and the spectrum have the same length M, so
//   G[j][k] = C H[k] P_j[k] e^{+2 pi i k c / M},   P_j = FFT_M(padded row),   G[j][-M/2] = 0.
// It backprojects the UNCROPPED periodic filtered row (tails outside the detector included).
// p[nproj][n] -> G[nproj][M], FFT order; pad as in orc_filter_rows_pad.
// ---------------------------------------------------------------------------
void orc_spectrum_fused(const double* p, int nproj, int n, double center, int filter, int pad, cplx* G) {
    const int M = 2 * n;
    const double C = PI / ((double)nproj * (double)M);
    std::vector<double> H(M);
    orc_filter(M, filter, H.data());
    std::vector<cplx> a(M), P(M);
    for (int j = 0; j < nproj; ++j) {
        const double* pr = p + (size_t)j * n;
        for (int i = 0; i < M; ++i) a[i] = (i < n) ? pr[i] : (pad == 0 ? 0.0 : (i < n + n / 2 ? pr[n - 1] : pr[0]));
        orc_fft(a.data(), P.data(), M, -1);
        for (int k = 0; k < M; ++k) {
            int ks = (k < M / 2) ? k : k - M;
            double ph = 2.0 * PI * (double)ks * center / (double)M;
            G[(size_t)j * M + k] = C * H[k] * P[k] * cplx(std::cos(ph), std::sin(ph));
        }
        G[(size_t)j * M + M / 2] = 0.0;
    }
}

}  // extern "C"
