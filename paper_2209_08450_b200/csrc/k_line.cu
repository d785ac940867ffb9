// k_line.cu -- the paper's direct line-summation operator ("LineRec"; O(N^4), also
// the operator the paper reuses for laminography): backprojection of the filtered sinogram with linear
// interpolation along the detector,
//   f[iy][ix] = (pi / nproj) sum_j (1 - w) q_j[i0] + w q_j[i0 + 1],
//   s = x cos(theta_j) + y sin(theta_j) + c,  i0 = floor(s),  w = s - i0,  q_j[i] = 0 outside [0, n),
// x = ix - n/2, y = iy - n/2 (reading Q9).  q is the filtered sinogram S3 leaves in the sinogram
// workspace (filter_kernel, k_rows.cu).  Selected by tcp_set_option(TCP_OPT_ALGORITHM, TCP_ALG_LINE).
//
// A thread owns one pixel of ZT slices: the detector coordinate is formed once per projection and shared
// by the slices.  s is needed to ~1e-6 of a detector pixel at |x|, |y| up to 2048 for the 1e-5 gate, so
// it is summed in float-float arithmetic from the float-float trig table (products by FMA residuals,
// sums by two-sum); floor and fraction are then exact to ~1e-7.
#include "tcp_internal.h"

namespace tcpk {

template <class TS, class TO, int ZT>
__global__ void __launch_bounds__(256) line_bp_kernel(const TS* __restrict__ q, TO* __restrict__ out,
                                                      const float4* __restrict__ trigf, int nproj, int n, int nz,
                                                      float center, float scale) {
    const int ix = blockIdx.x * 32 + threadIdx.x, iy = blockIdx.y * 8 + threadIdx.y, z0 = blockIdx.z * ZT;
    const float x = (float)(ix - n / 2), y = (float)(iy - n / 2);
    const size_t zstride = (size_t)nproj * n;
    float acc[ZT];
#pragma unroll
    for (int zz = 0; zz < ZT; ++zz) acc[zz] = 0.f;
    const TS* row = q + (size_t)z0 * zstride;
    for (int j = 0; j < nproj; ++j, row += n) {
        const float4 t = __ldg(&trigf[j]);                       // (cos hi, cos lo, sin hi, sin lo)
        const float p1 = x * t.x, p2 = y * t.z;
        const float e12 = fmaf(x, t.x, -p1) + fmaf(y, t.z, -p2) + fmaf(x, t.y, y * t.w);
        const float a = p1 + p2, ab = a - p1;
        const float ea = (p1 - (a - ab)) + (p2 - ab);
        const float u = a + center, ub = u - a;
        const float eu = (a - (u - ub)) + (center - ub);
        float fl = floorf(u);
        float w = (u - fl) + (e12 + ea + eu);
        if (w < 0.f) { fl -= 1.f; w += 1.f; }
        else if (w >= 1.f) { fl += 1.f; w -= 1.f; }
        const int i0 = (int)fl;
        const bool v0 = (unsigned)i0 < (unsigned)n, v1 = (unsigned)(i0 + 1) < (unsigned)n;
        const TS* r = row;
#pragma unroll
        for (int zz = 0; zz < ZT; ++zz) {
            if (z0 + zz < nz) {
                const float q0 = v0 ? ld_r(r, i0) : 0.f, q1 = v1 ? ld_r(r, i0 + 1) : 0.f;
                acc[zz] += fmaf(w, q1 - q0, q0);
            }
            r += zstride;
        }
    }
#pragma unroll
    for (int zz = 0; zz < ZT; ++zz)
        if (z0 + zz < nz) st_r(out, ((size_t)(z0 + zz) * n + iy) * n + ix, acc[zz] * scale);
}

template <class TS, class TO>
static int launch_line_t(const tcp_ctx* c, void* out, cudaStream_t st) {
    constexpr int ZT = 8;
    dim3 grid(c->n / 32, c->n / 8, (c->nz + ZT - 1) / ZT), block(32, 8);
    line_bp_kernel<TS, TO, ZT><<<grid, block, 0, st>>>((const TS*)c->sino, (TO*)out, c->trigf, c->nproj, c->n, c->nz, c->center,
                                                       (float)(3.14159265358979323846 / (double)c->nproj));
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_line_bp(const tcp_ctx* c, void* out, cudaStream_t st) {
    if (!c->half_store) return launch_line_t<float, float>(c, out, st);
    return c->half_out ? launch_line_t<__half, __half>(c, out, st) : launch_line_t<__half, float>(c, out, st);
}

}  // namespace tcpk
