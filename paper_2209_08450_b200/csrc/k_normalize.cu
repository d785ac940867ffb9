// k_normalize.cu -- S1+S2: dark/flat-field correction, negative logarithm and cast
// (fp16 rule PAPER.md:53: arithmetic in fp32, one rounding to the storage type),
// the frame-averaging helper, and the fp64 cos/sin table of the projection angles.
//
// HBM-bound: 2 B read + B_r written per sample.  Each thread moves 8 detector pixels:
// one 128-bit load of uint16, 2x2 128-bit loads of flat/dark (L2 resident: nz*n floats are
// reused by all nproj projections) and one (half) or two (float) 128-bit stores.  The
// projection-major -> slice-major transpose only permutes whole rows, so both sides stay
// fully coalesced.
#include <algorithm>

#include "tcp_internal.h"

namespace tcpk {

__device__ __forceinline__ float neglog1(float raw, float flat, float dark) {
    const float eps_d = 1e-3f, t_min = 1e-6f;
    const float den = flat - dark;
    // near t = 1 (air) -ln t cancels: use t - 1 = (raw - flat)/den, exact numerator (Sterbenz),
    // and log1p, so p keeps fp32 RELATIVE accuracy even where p ~ 0
    if (den >= eps_d) {
        const float u = (raw - flat) / den;
        if (u > -0.5f) return -log1pf(u);
    }
    const float t = fmaxf((raw - dark) / fmaxf(den, eps_d), t_min);
    return -logf(t);
}

template <class TS>
__global__ void __launch_bounds__(256) normalize_kernel(const uint4* __restrict__ raw, const float4* __restrict__ flat,
                                                        const float4* __restrict__ dark, TS* __restrict__ sino,
                                                        int nproj, int nz, int n8) {
    // one thread per 8 pixels; index space [nproj][nz][n8] in raw order
    const size_t total = (size_t)nproj * nz * n8;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int i8 = (int)(v % n8);
        const size_t row = v / n8;
        const int z = (int)(row % nz);
        const int j = (int)(row / nz);
        const uint4 r = __ldcs(&raw[v]);                       // streamed once
        const size_t fo = ((size_t)z * n8 + i8) * 2;
        const float4 f0 = __ldg(&flat[fo]), f1 = __ldg(&flat[fo + 1]);
        const float4 d0 = __ldg(&dark[fo]), d1 = __ldg(&dark[fo + 1]);
        float p[8];
        p[0] = neglog1((float)(r.x & 0xffffu), f0.x, d0.x);
        p[1] = neglog1((float)(r.x >> 16), f0.y, d0.y);
        p[2] = neglog1((float)(r.y & 0xffffu), f0.z, d0.z);
        p[3] = neglog1((float)(r.y >> 16), f0.w, d0.w);
        p[4] = neglog1((float)(r.z & 0xffffu), f1.x, d1.x);
        p[5] = neglog1((float)(r.z >> 16), f1.y, d1.y);
        p[6] = neglog1((float)(r.w & 0xffffu), f1.z, d1.z);
        p[7] = neglog1((float)(r.w >> 16), f1.w, d1.w);
        const size_t o = (((size_t)z * nproj + j) * n8 + i8) * 8;   // element offset in sino
        float4* dst = reinterpret_cast<float4*>(sino + o);
        dst[0] = make_float4(p[0], p[1], p[2], p[3]);
        dst[1] = make_float4(p[4], p[5], p[6], p[7]);
    }
}

// fp16 storage: the result is rounded to half (2^-11 relative), so the hardware approximations
// (rcp.approx, lg2.approx: ~2^-22) are exact for the purpose and the kernel stays HBM-bound instead of
// ALU-bound.  A thread keeps 1 / (flat - dark) and dark of its 8 pixels in registers and walks JP
// projections of the same detector row, so the flat/dark loads and the reciprocals are amortised.
// fast_rcp, fast_lg2, u16f: tcp_internal.h (shared with the fused loader of rows_kernel)

constexpr int JP = 4;
__global__ void __launch_bounds__(256) normalize_half_kernel(const uint4* __restrict__ raw, const float4* __restrict__ flat,
                                                             const float4* __restrict__ dark, __half* __restrict__ sino,
                                                             int nproj, int nz, int n8) {
    const float eps_d = 1e-3f, t_min = 1e-6f, mln2 = -0.69314718055994531f;
    const int jgroups = (nproj + JP - 1) / JP;
    const size_t total = (size_t)jgroups * nz * n8;             // index space [jgroup][nz][n8]
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int i8 = (int)(v % n8);
        const size_t row = v / n8;
        const int z = (int)(row % nz);
        const int j0 = (int)(row / nz) * JP;
        const size_t fo = ((size_t)z * n8 + i8) * 2;
        const float4 f0 = __ldg(&flat[fo]), f1 = __ldg(&flat[fo + 1]);
        const float4 d0 = __ldg(&dark[fo]), d1 = __ldg(&dark[fo + 1]);
        const float dk[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
        const float fl[8] = {f0.x, f0.y, f0.z, f0.w, f1.x, f1.y, f1.z, f1.w};
        float inv[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) inv[e] = fast_rcp(fmaxf(fl[e] - dk[e], eps_d));
        uint4 r[JP];
#pragma unroll
        for (int q = 0; q < JP; ++q)
            if (j0 + q < nproj) r[q] = __ldcs(&raw[((size_t)(j0 + q) * nz + z) * n8 + i8]);
#pragma unroll
        for (int q = 0; q < JP; ++q) {
            if (j0 + q >= nproj) break;
            const unsigned w[4] = {r[q].x, r[q].y, r[q].z, r[q].w};
            float p[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const unsigned u = (e & 1) ? (w[e >> 1] >> 16) : (w[e >> 1] & 0xffffu);
                p[e] = mln2 * fast_lg2(fmaxf((u16f(u) - dk[e]) * inv[e], t_min));
            }
            const __half2 h0 = __floats2half2_rn(p[0], p[1]), h1 = __floats2half2_rn(p[2], p[3]);
            const __half2 h2 = __floats2half2_rn(p[4], p[5]), h3 = __floats2half2_rn(p[6], p[7]);
            uint4 o4;
            o4.x = *reinterpret_cast<const unsigned*>(&h0);
            o4.y = *reinterpret_cast<const unsigned*>(&h1);
            o4.z = *reinterpret_cast<const unsigned*>(&h2);
            o4.w = *reinterpret_cast<const unsigned*>(&h3);
            *reinterpret_cast<uint4*>(sino + (((size_t)z * nproj + (j0 + q)) * n8 + i8) * 8) = o4;
        }
    }
}

// Detector width ndet not a power of two (tcp_create_det; "padded/unpadded to the power of 2
// sizes"): sample i of the caller's row lands at i + pad_l of a row of n, the rest is air (p = 0).  Scalar
// loads: ndet may be odd.  Same arithmetic as normalize_kernel, one rounding to the storage type.
template <class TS>
__global__ void __launch_bounds__(256) normalize_pad_kernel(const uint16_t* __restrict__ raw, const float* __restrict__ flat,
                                                            const float* __restrict__ dark, TS* __restrict__ sino, int nproj,
                                                            int nz, int n, int ndet, int pad_l) {
    const size_t total = (size_t)nproj * nz * n;                // index space [nproj][nz][n] (padded rows, raw order)
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int ip = (int)(v % n);
        const size_t row = v / n;
        const int z = (int)(row % nz);
        const int j = (int)(row / nz);
        const int i = ip - pad_l;
        float p = 0.f;
        if (i >= 0 && i < ndet)
            p = neglog1((float)raw[((size_t)j * nz + z) * ndet + i], __ldg(&flat[(size_t)z * ndet + i]),
                        __ldg(&dark[(size_t)z * ndet + i]));
        st_r(sino, ((size_t)z * nproj + j) * n + ip, p);
    }
}

// the central ndet x ndet pixels of the padded image [nslices][n][n] -> out [nslices][ndet][ndet]
template <class TO>
__global__ void __launch_bounds__(256) crop_out_kernel(const TO* __restrict__ src, TO* __restrict__ dst, int nslices, int n,
                                                       int ndet, int pad_l) {
    const size_t total = (size_t)nslices * ndet * ndet;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(v % ndet);
        const size_t r = v / ndet;
        const int iy = (int)(r % ndet);
        const size_t z = r / ndet;
        dst[v] = src[(z * n + (iy + pad_l)) * n + (ix + pad_l)];
    }
}

int launch_crop_out(const tcp_ctx* c, int nslices, void* out, cudaStream_t st) {
    const size_t total = (size_t)nslices * c->ndet * c->ndet;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)148 * 8 * 4);
    if (c->half_out)
        crop_out_kernel<__half><<<blocks, 256, 0, st>>>((const __half*)c->out_pad, (__half*)out, nslices, c->n, c->ndet, c->pad_l);
    else
        crop_out_kernel<float><<<blocks, 256, 0, st>>>((const float*)c->out_pad, (float*)out, nslices, c->n, c->ndet, c->pad_l);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_normalize(const tcp_ctx* c, const uint16_t* raw, const float* flat, const float* dark, cudaStream_t st) {
    if (c->ndet != c->n) {
        const size_t total = (size_t)c->nproj * c->nz * c->n;
        const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)148 * 8 * 4);
        if (c->half_store)
            normalize_pad_kernel<__half><<<blocks, 256, 0, st>>>(raw, flat, dark, (__half*)c->sino, c->nproj, c->nz, c->n, c->ndet, c->pad_l);
        else
            normalize_pad_kernel<float><<<blocks, 256, 0, st>>>(raw, flat, dark, (float*)c->sino, c->nproj, c->nz, c->n, c->ndet, c->pad_l);
        TCP_CUDA_CHECK(cudaGetLastError());
        return TCP_OK;
    }
    const int n8 = c->n / 8;
    const int cap = 148 * 8 * 4;                  // a few waves of 8 resident CTAs per SM
    if (c->half_store) {
        const size_t total = (size_t)((c->nproj + JP - 1) / JP) * c->nz * n8;
        int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)cap);
        normalize_half_kernel<<<blocks, 256, 0, st>>>((const uint4*)raw, (const float4*)flat, (const float4*)dark,
                                                      (__half*)c->sino, c->nproj, c->nz, n8);
    } else {
        const size_t total = (size_t)c->nproj * c->nz * n8;
        int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)cap);
        normalize_kernel<float><<<blocks, 256, 0, st>>>((const uint4*)raw, (const float4*)flat, (const float4*)dark,
                                                        (float*)c->sino, c->nproj, c->nz, n8);
    }
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

// mean of K uint16 frames: sum in fp32 (exact below 2^24), one division
__global__ void mean_frames_kernel(const uint16_t* __restrict__ frames, int nframes, size_t npix, float* __restrict__ mean) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npix; i += (size_t)gridDim.x * blockDim.x) {
        float s = 0.f;
        for (int k = 0; k < nframes; ++k) s += (float)frames[(size_t)k * npix + i];
        mean[i] = s / (float)nframes;
    }
}

int launch_mean_frames(const uint16_t* frames, int nframes, int nz, int n, float* mean, cudaStream_t st) {
    const size_t npix = (size_t)nz * n;
    int blocks = (int)((npix + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    mean_frames_kernel<<<blocks, 256, 0, st>>>(frames, nframes, npix, mean);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

// cos/sin of the float32 angles in fp64: k*cos(theta) with
// k up to 4096 must be good to ~1e-6 grid cells for the 1e-5 fp32 gate.
__global__ void trig_kernel(const float* __restrict__ theta, int nproj, double2* __restrict__ trig, float4* __restrict__ trigf,
                            float* __restrict__ wq, const float* __restrict__ flat,
                            const float* __restrict__ dark, float2* __restrict__ fdtab, int nfd) {
    // fused S1+S2 (rows_kernel's loader): per detector pixel of the chunk the reciprocal normalize_half_kernel forms, and dark
    if (flat)
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nfd; i += gridDim.x * blockDim.x) {
            const float dk = dark[i];
            fdtab[i] = make_float2(fast_rcp(fmaxf(flat[i] - dk, 1e-3f)), dk);
        }
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < nproj) {
        // quadrature weight for unequally spaced angles (TCP_OPT_ANGLE_WEIGHTS, reading Q20):
        // trapezoid rule on the periodic angle axis, (theta_{j+1} - theta_{j-1}) / 2 with theta_nproj = theta_0 + pi
        // and theta_{-1} = theta_{nproj-1} - pi, relative to pi/nproj; fp64 from the float32 angles
        {
            const double pi = 3.14159265358979323846264338327950288;
            const double nxt = (j + 1 < nproj) ? (double)theta[j + 1] : (double)theta[0] + pi;
            const double prv = (j > 0) ? (double)theta[j - 1] : (double)theta[nproj - 1] - pi;
            wq[j] = (float)(0.5 * (nxt - prv) * (double)nproj / pi);
        }
        double t = (double)theta[j];
        const double c = cos(t), s = sin(t);
        trig[j] = make_double2(c, s);
        // float-float split (hi + lo = the fp64 value to 2^-48): lets the fp16 gridding kernel form
        // k*cos, k*sin to ~1e-11 cells with fp32 FMAs only
        const float ch = (float)c, sh = (float)s;
        trigf[j] = make_float4(ch, (float)(c - (double)ch), sh, (float)(s - (double)sh));
    }
}

int launch_trig(const tcp_ctx* c, const float* theta, cudaStream_t st, const float* flat, const float* dark) {
    const int nfd = c->nz * c->n;
    const int blocks = flat ? std::max((c->nproj + 127) / 128, std::min((nfd + 127) / 128, 148 * 4)) : (c->nproj + 127) / 128;
    trig_kernel<<<blocks, 128, 0, st>>>(theta, c->nproj, c->trig, c->trigf, c->wq, flat, dark, c->fdtab, nfd);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

}  // namespace tcpk
