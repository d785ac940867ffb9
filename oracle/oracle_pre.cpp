// oracle_pre.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle.cpp header).
//
// Optional pre-processing of the sinogram between S2 (-log) and S3 (filter): "pre-processing may include
// ring-removal filtering ... with an analytical formula by V. Titarenko (Titarenko et al., 2010; Titarenko, 2016), zinger
// artifacts reduction (Rivers, 1998)".  The paper names the methods and prints no formula; the readings
// built here are DESIGN.md Q22 (zingers) and Q23 (rings), written out below.  Plain double precision, slice by slice.
//
// Pins (tests/test_oracle_pins.py, P13 / P14): the 3 x 3 median against numpy.median on every window of a small array;
// untouched samples stay bit-identical; injected zingers are the only samples replaced; the ring estimate against a dense
// numpy.linalg.solve of the same normal equations, its null space (a profile linear in the detector index is left alone),
// and the damping of a single bad column.

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <vector>

extern "C" {

// ---------------------------------------------------------------------------
// Zinger removal (reading Q22, after Rivers 1998: a zinger is an isolated bright detector sample, i.e. an isolated LOW
// sample of p = -ln t; it is detected against a median-smoothed copy and replaced by it).  For every sample of every slice
//   med = median of the 3 x 3 neighbourhood in (projection j, detector pixel i) of the ORIGINAL sinogram, indices clamped
//         to the array (edge samples repeat),
//   p'[j][i] = med  if  med - p[j][i] > dif,  else p[j][i].
// p, out: [nz][nproj][n]; out must not alias p.
// ---------------------------------------------------------------------------
void orc_zinger(const double* p, int nz, int nproj, int n, double dif, double* out) {
    for (int z = 0; z < nz; ++z) {
        const double* s = p + (size_t)z * nproj * n;
        double* o = out + (size_t)z * nproj * n;
        for (int j = 0; j < nproj; ++j)
            for (int i = 0; i < n; ++i) {
                double w[9];
                int t = 0;
                for (int dj = -1; dj <= 1; ++dj)
                    for (int di = -1; di <= 1; ++di) {
                        const int jj = std::min(std::max(j + dj, 0), nproj - 1), ii = std::min(std::max(i + di, 0), n - 1);
                        w[t++] = s[(size_t)jj * n + ii];
                    }
                std::sort(w, w + 9);
                const double med = w[4], v = s[(size_t)j * n + i];
                o[(size_t)j * n + i] = (med - v > dif) ? med : v;
            }
    }
}

// ---------------------------------------------------------------------------
// Ring removal by a closed-form Tikhonov estimate (reading Q23, after Titarenko et al. 2010).  A ring is an offset r[i] of
// detector pixel i that is the same in every projection: p[j][i] = u[j][i] + r[i].  With pbar[i] the mean of p[j][i] over
// the projections and D2 the second-difference operator ((D2 v)[i] = v[i] - 2 v[i+1] + v[i+2], i = 0..n-3), the offsets
// are estimated as the minimiser of
//   || D2 (pbar - r) ||^2 + alpha || r ||^2        (the object's mean profile is smooth, the offsets are small),
// whose normal equations have the closed form  (A + alpha I) r = A pbar,  A = D2^T D2  (symmetric, pentadiagonal);
// then p'[j][i] = p[j][i] - r[i] for every projection.  The system is solved by banded Cholesky (LDL^T), O(n).
// p, out: [nz][nproj][n] (out may alias p); r_out: [nz][n] or NULL.
// ---------------------------------------------------------------------------
void orc_ring_ti(const double* p, int nz, int nproj, int n, double alpha, double* out, double* r_out) {
    for (int z = 0; z < nz; ++z) {
        const double* s = p + (size_t)z * nproj * n;
        std::vector<double> pbar(n, 0.0), rhs(n, 0.0), r(n, 0.0);
        for (int i = 0; i < n; ++i) {
            double acc = 0.0;
            for (int j = 0; j < nproj; ++j) acc += s[(size_t)j * n + i];
            pbar[i] = acc / (double)nproj;
        }
        // bands of A = D2^T D2: a0 diagonal, a1 first, a2 second off-diagonal; rhs = D2^T (D2 pbar)
        std::vector<double> a0(n, 0.0), a1(n, 0.0), a2(n, 0.0);
        for (int i = 0; i + 2 < n; ++i) {
            const double d = pbar[i] - 2.0 * pbar[i + 1] + pbar[i + 2];
            rhs[i] += d; rhs[i + 1] -= 2.0 * d; rhs[i + 2] += d;
            a0[i] += 1.0; a0[i + 1] += 4.0; a0[i + 2] += 1.0;
            a1[i] -= 2.0; a1[i + 1] -= 2.0;          // (i, i+1) and (i+1, i+2)
            a2[i] += 1.0;                            // (i, i+2)
        }
        for (int i = 0; i < n; ++i) a0[i] += alpha;
        // LDL^T of the pentadiagonal matrix: L unit lower with sub-diagonals l1, l2
        std::vector<double> d(n), l1(n, 0.0), l2(n, 0.0);
        for (int i = 0; i < n; ++i) {
            double di = a0[i];
            if (i >= 1) di -= l1[i - 1] * l1[i - 1] * d[i - 1];
            if (i >= 2) di -= l2[i - 2] * l2[i - 2] * d[i - 2];
            d[i] = di;
            if (i + 1 < n) {
                double v = a1[i];
                if (i >= 1) v -= l1[i - 1] * l2[i - 1] * d[i - 1];
                l1[i] = v / di;
            }
            if (i + 2 < n) l2[i] = a2[i] / di;
        }
        std::vector<double> y(n);
        for (int i = 0; i < n; ++i) {
            double v = rhs[i];
            if (i >= 1) v -= l1[i - 1] * y[i - 1];
            if (i >= 2) v -= l2[i - 2] * y[i - 2];
            y[i] = v;
        }
        for (int i = n - 1; i >= 0; --i) {
            double v = y[i] / d[i];
            if (i + 1 < n) v -= l1[i] * r[i + 1];
            if (i + 2 < n) v -= l2[i] * r[i + 2];
            r[i] = v;
        }
        double* o = out + (size_t)z * nproj * n;
        for (int j = 0; j < nproj; ++j)
            for (int i = 0; i < n; ++i) o[(size_t)j * n + i] = s[(size_t)j * n + i] - r[i];
        if (r_out)
            for (int i = 0; i < n; ++i) r_out[(size_t)z * n + i] = r[i];
    }
}

}  // extern "C"
