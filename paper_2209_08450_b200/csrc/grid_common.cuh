// grid_common.cuh -- pieces shared by the two tile-owned gridding kernels (k_grid_tile.cu: CUDA-core
// FMA path; k_grid_mma.cu: tcgen05 path): tile geometry, chord records, the fp32 chord range test.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

namespace tcpk {

constexpr int TS = 32;          // tile side (cells)
constexpr int NTHR = 256;       // threads per CTA: 16 x 16 blocks of 2 x 2 cells
constexpr int MAXREC = 32;      // records (chords) per batch: one hit-mask bit each

__host__ __device__ constexpr int chord_len(int MH) { return MH == 3 ? 56 : 60; }   // >= (32+2m+.1) sqrt2 + 2
template <class TC> __host__ __device__ constexpr int batch_records() { return sizeof(TC) == 4 ? 24 : 12; }

struct ChordRec {               // one staged chord
    float c, s;                 // cos, sin of the projection (fp32: range tests only)
    float inv;                  // 1 / dominant component
    int pack;                   // kmin (low 16, signed) | count << 16 | dominant axis << 24
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Kaiser-Bessel window (kernel code 16 + m, reading Q21): phi(d) = I0(beta sqrt(u)) / I0(beta), u = 1 - (d/m)^2,
// from a table of phi over u in [0, 1] (KB_NTAB intervals, built in fp64 at create) with linear interpolation:
// |error| <= h^2 / 8 max|phi''(u)| = 4e-7 at beta = 13.9, below the fp32 path's 1e-5 gate.
constexpr int KB_NTAB = 4096;
__device__ __forceinline__ float kb_weight(const float* __restrict__ tab, float d, float inv_m2) {
    const float u = fmaxf(fmaf(-d * d, inv_m2, 1.f), 0.f) * (float)KB_NTAB;
    const int i = min((int)u, KB_NTAB - 1);
    const float a = __ldg(tab + i), b = __ldg(tab + i + 1);
    return fmaf(u - (float)i, b - a, a);
}
// weight of one tap at distance d: Gaussian 2^(-k2 d^2) (kbtab == NULL, k2 = alpha log2 e) or the table (k2 = 1 / m^2)
__device__ __forceinline__ float tap_weight(const float* __restrict__ kbtab, float d, float k2) {
    return kbtab ? kb_weight(kbtab, d, k2) : ex2_approx(-k2 * d * d);
}

template <class TC> __device__ __forceinline__ TC czero();
template <> __device__ __forceinline__ float2 czero<float2>() { return make_float2(0.f, 0.f); }
template <> __device__ __forceinline__ __half2 czero<__half2>() { return __floats2half2_rn(0.f, 0.f); }

// acc += w * g for one complex value; fp16 storage: g is a half2 (re, im) word, w a half
__device__ __forceinline__ void cfma_h(float& re, float& im, unsigned g, unsigned short w) {
    asm("{.reg .b16 lo, hi;\n mov.b32 {lo, hi}, %2;\n fma.rn.f32.f16 %0, lo, %3, %0;\n fma.rn.f32.f16 %1, hi, %3, %1;}"
        : "+f"(re), "+f"(im)
        : "r"(g), "h"(w));
}

// k-range of the samples of a ray (c, s) inside the box [ax, bx) x [ay, by) (already widened by
// the kernel support and a slack), clipped to |k| <= kmaxabs.  fp32: a superset is enough, the
// exact tap decision is taken per sample in fp64.
__device__ __forceinline__ bool chord_range(float c, float s, float ax, float bx, float ay, float by, float kmaxabs,
                                            int& kmin, int& kmax) {
    float lo = -kmaxabs, hi = kmaxabs;
    if (fabsf(c) > 1e-6f) {
        const float t0 = ax / c, t1 = bx / c;
        lo = fmaxf(lo, fminf(t0, t1));
        hi = fminf(hi, fmaxf(t0, t1));
    } else if (!(ax <= 0.01f && bx >= -0.01f)) return false;
    if (fabsf(s) > 1e-6f) {
        const float t0 = ay / s, t1 = by / s;
        lo = fmaxf(lo, fminf(t0, t1));
        hi = fminf(hi, fmaxf(t0, t1));
    } else if (!(ay <= 0.01f && by >= -0.01f)) return false;
    kmin = (int)ceilf(lo);
    kmax = (int)floorf(hi);
    return kmin <= kmax;
}

}  // namespace tcpk
