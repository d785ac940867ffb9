// k_grid.cu -- S5: polar -> Cartesian gridding with the separable Gaussian kernel
// phi(t) = exp(-alpha t^2), alpha = pi/(sqrt(2) m), open box |l - nu| < m per axis,
// oversampling 2, periodic in M  ("exponential functions for interpolation
// in the frequency domain", :173 oversampling; readings Q7 in DESIGN.md).
//
// Two implementations:
//  * gather (default, atomics-free, bitwise reproducible): every thread OWNS Cartesian cells
//    and sums the polar samples whose box covers them.  Because the grid side equals the padded
//    row length M, samples on a ray are one grid cell apart, so the samples of projection j
//    near cell l are k = round(l.u_j) + i, |i| <= m sqrt(2) + 1/2, and only projections whose ray
//    passes within m sqrt(2) of the cell matter: an angular window around atan2(l2, l1).
//  * scatter with fp32 atomics (bring-up and cross-check only; fp32 grid only).
#include "tcp_internal.h"

namespace tcpk {

constexpr int GT = 16;   // gather tile side (cells); 256 threads per CTA

// ---------------------------------------------------------------------------------------
template <int MH, class TC>
__global__ void __launch_bounds__(GT* GT) grid_gather_kernel(const TC* __restrict__ spec, TC* __restrict__ grid,
                                                             const double2* __restrict__ trig,
                                                             const float* __restrict__ theta,
                                                             const int* __restrict__ tile_order, int nproj, int M,
                                                             float alpha2) {
    const int n = M >> 1;
    const int tiles_x = M / GT;
    const int tile = tile_order[blockIdx.x];
    const int pair = blockIdx.y;
    const int L1 = (tile % tiles_x) * GT + (threadIdx.x % GT);
    const int L2 = (tile / tiles_x) * GT + (threadIdx.x / GT);
    const int l1 = (L1 < n) ? L1 : L1 - M;   // signed, [-n, n)
    const int l2 = (L2 < n) ? L2 : L2 - M;
    const TC* sp = spec + (size_t)pair * nproj * M;
    constexpr float RMAX = MH * 1.41421356f + 0.01f;      // max distance of a contributing sample
    constexpr int RI = (int)(MH * 1.41421356f + 0.5f);    // |k - round(u)| <= RI
    constexpr float PI_F = 3.14159265358979f;
    const float t0 = theta[0];

    float2 acc = make_float2(0.f, 0.f);
    // periodic images of the cell that samples (|nu| <= n-1) can reach
    const int na1 = (l1 <= -n + MH - 2) ? 2 : ((l1 >= n - MH) ? 2 : 1);
    const int na2 = (l2 <= -n + MH - 2) ? 2 : ((l2 >= n - MH) ? 2 : 1);
    for (int a2 = 0; a2 < na2; ++a2) {
        const int lam2 = (a2 == 0) ? l2 : ((l2 < 0) ? l2 + M : l2 - M);
        for (int a1 = 0; a1 < na1; ++a1) {
            const int lam1 = (a1 == 0) ? l1 : ((l1 < 0) ? l1 + M : l1 - M);
            const float rho = sqrtf((float)lam1 * (float)lam1 + (float)lam2 * (float)lam2);
            if (rho > (float)(n - 1) + RMAX + 1.f) continue;
            int j0 = 0, count = nproj;
            float a = 0.f, width = 4.f * PI_F;
            if (rho > RMAX + 0.5f) {
                const float delta = asinf(fminf(1.f, RMAX / rho)) + 1e-4f;
                if (delta < 0.5f * PI_F - 1e-3f) {
                    const float psi = atan2f((float)lam2, (float)lam1);
                    a = psi - delta - t0;
                    a -= PI_F * floorf(a / PI_F);          // [0, pi)
                    width = 2.f * delta;
                    int lo = 0, hi = nproj;                // first j with theta[j] - t0 >= a
                    while (lo < hi) {
                        int mid = (lo + hi) >> 1;
                        if (theta[mid] - t0 < a) lo = mid + 1; else hi = mid;
                    }
                    j0 = lo;
                }
            }
            for (int cnt = 0; cnt < count; ++cnt) {
                int j = j0 + cnt;
                float wrapped = 0.f;
                if (j >= nproj) { j -= nproj; wrapped = PI_F; }
                if ((theta[j] - t0) + wrapped - a > width) break;
                const double2 cs = trig[j];
                const double u = (double)lam1 * cs.x + (double)lam2 * cs.y;
                const double k0d = rint(u);
                const int k0 = (int)k0d;
                const double ex = fma(k0d, cs.x, -(double)lam1);   // sample k0 relative to the cell
                const double ey = fma(k0d, cs.y, -(double)lam2);
                const TC* row = sp + (size_t)j * M;
#pragma unroll
                for (int i = -RI; i <= RI; ++i) {
                    const int k = k0 + i;
                    const double dxd = fma((double)i, cs.x, ex);
                    const double dyd = fma((double)i, cs.y, ey);
                    if (fabs(dxd) < (double)MH && fabs(dyd) < (double)MH && k > -n && k < n) {
                        const float dx = (float)dxd, dy = (float)dyd;
                        const float w = exp2f(-alpha2 * fmaf(dx, dx, dy * dy));
                        const float2 g = ld_c(row, (size_t)(k & (M - 1)));
                        acc.x = fmaf(w, g.x, acc.x);
                        acc.y = fmaf(w, g.y, acc.y);
                    }
                }
            }
        }
    }
    st_c(grid + (size_t)pair * M * M, (size_t)L2 * M + L1, acc);
}

int launch_grid_gather(const tcp_ctx* c, const float* theta, cudaStream_t st) {
    const double alpha = 3.14159265358979323846 / (1.4142135623730951 * c->m);
    const float alpha2 = (float)(alpha * 1.4426950408889634);
    dim3 grid(c->ntiles, c->npair);
#define LAUNCH(MH, TC)                                                                                          \
    grid_gather_kernel<MH, TC><<<grid, GT * GT, 0, st>>>((const TC*)c->spec, (TC*)c->grid, c->trig, theta,      \
                                                         c->tile_order, c->nproj, c->M, alpha2)
    if (c->m == 3) { if (c->half_store) LAUNCH(3, __half2); else LAUNCH(3, float2); }
    else           { if (c->half_store) LAUNCH(4, __half2); else LAUNCH(4, float2); }
#undef LAUNCH
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

// ---------------------------------------------------------------------------------------
template <int MH>
__global__ void __launch_bounds__(256) grid_scatter_kernel(const float2* __restrict__ spec, float2* __restrict__ grid,
                                                           const double2* __restrict__ trig, int nproj, int M,
                                                           float alpha) {
    const int n = M >> 1;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)nproj * M) return;
    const int pair = blockIdx.y;
    const int j = (int)(idx / M), kk = (int)(idx % M);
    const int k = (kk < n) ? kk : kk - M;
    if (k == -n) return;
    const double2 cs = trig[j];
    const double nu1 = (double)k * cs.x, nu2 = (double)k * cs.y;
    const double f1 = floor(nu1), f2 = floor(nu2);
    const int l01 = (int)f1, l02 = (int)f2;
    float w1[2 * MH], w2[2 * MH];
#pragma unroll
    for (int a = 0; a < 2 * MH; ++a) {
        const double t1 = (double)(a - MH + 1) + (f1 - nu1), t2 = (double)(a - MH + 1) + (f2 - nu2);
        w1[a] = (fabs(t1) < (double)MH) ? expf(-alpha * (float)(t1 * t1)) : 0.f;
        w2[a] = (fabs(t2) < (double)MH) ? expf(-alpha * (float)(t2 * t2)) : 0.f;
    }
    const float2 g = spec[((size_t)pair * nproj + j) * M + kk];
    float2* F = grid + (size_t)pair * M * M;
#pragma unroll
    for (int a2 = 0; a2 < 2 * MH; ++a2) {
        const int r = (l02 + a2 - MH + 1) & (M - 1);
#pragma unroll
        for (int a1 = 0; a1 < 2 * MH; ++a1) {
            const int cc = (l01 + a1 - MH + 1) & (M - 1);
            const float w = w1[a1] * w2[a2];
            if (w != 0.f) {
                atomicAdd(&F[(size_t)r * M + cc].x, g.x * w);
                atomicAdd(&F[(size_t)r * M + cc].y, g.y * w);
            }
        }
    }
}

int launch_grid_scatter(const tcp_ctx* c, cudaStream_t st) {
    if (c->half_store) return set_error(TCP_EUNSUPPORTED, "scatter gridding supports TCP_F32 only");
    TCP_CUDA_CHECK(cudaMemsetAsync(c->grid, 0, (size_t)c->npair * c->M * c->M * sizeof(float2), st));
    const float alpha = (float)(3.14159265358979323846 / (1.4142135623730951 * c->m));
    dim3 grid((unsigned)(((size_t)c->nproj * c->M + 255) / 256), c->npair);
    if (c->m == 3)
        grid_scatter_kernel<3><<<grid, 256, 0, st>>>((const float2*)c->spec, (float2*)c->grid, c->trig, c->nproj, c->M, alpha);
    else
        grid_scatter_kernel<4><<<grid, 256, 0, st>>>((const float2*)c->spec, (float2*)c->grid, c->trig, c->nproj, c->M, alpha);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

}  // namespace tcpk
