// k_ifft2.cu -- S6 + S7: unnormalised inverse 2D FFT of the oversampled grid as two passes of
// 1D shared-memory transforms ("2D FFT as a combination of 1D FFTs"), pruned to
// the central n outputs per axis, with deapodisation, crop and cast fused into the second pass
// ("accuracy controls").
//
// pass 1 (columns): for each l1, IFFT over l2 -> x2; keep iy = x2 + n/2 in [0, n);
//                   T[pair][iy][l1].  A CTA owns W adjacent columns, so every global access is
//                   a W-wide segment; lines sit in shared memory with a stride chosen to keep
//                   the W-interleaved accesses bank-conflict free.
// pass 2 (rows):    for each iy, IFFT over l1 -> x1; keep ix = x1 + n/2;
//                   out[2 pair][iy][ix] = Re * deay[iy] * deax[ix], out[2 pair + 1] = Im * ...
#include "fft.cuh"
#include "tcp_internal.h"

namespace tcpk {

#ifndef COLS_BUDGET
#define COLS_BUDGET 16384
#endif
__host__ __device__ constexpr int cols_w(int M) { return (COLS_BUDGET / M) < 2 ? 2 : (COLS_BUDGET / M) < 32 ? (COLS_BUDGET / M) : 32; }   // columns per CTA
__host__ __device__ constexpr int cols_wp(int M) { return cols_w(M) / 2; }                          // column pairs per CTA
// stride between the pair-lines of a CTA, in cpair (16 B) units: a quarter-warp (8 lanes = one
// 128-byte shared-memory wavefront of 16-byte accesses) holds min(WP, 8) lines x 8 / min(WP, 8)
// consecutive elements, so lines must be 8 / min(WP, 8) elements apart modulo 8
__host__ __device__ constexpr int cols_stride(int M) {
    const int wp = cols_wp(M) < 8 ? cols_wp(M) : 8;
    const int want = (8 / wp) % 8;
    return padded_len(M) + (want - padded_len(M) % 8 + 8) % 8;
}

__device__ __forceinline__ cpair ld_c2(const float2* p, size_t i) {
    const float4 v = *reinterpret_cast<const float4*>(p + i);
    return cpair{make_float2(v.x, v.y), make_float2(v.z, v.w)};
}
__device__ __forceinline__ cpair ld_c2(const __half2* p, size_t i) {
    const uint2 v = *reinterpret_cast<const uint2*>(p + i);
    return cpair{__half22float2(*reinterpret_cast<const __half2*>(&v.x)), __half22float2(*reinterpret_cast<const __half2*>(&v.y))};
}
__device__ __forceinline__ void st_c2(float2* p, size_t i, cpair v) {
    *reinterpret_cast<float4*>(p + i) = make_float4(v.a.x, v.a.y, v.b.x, v.b.y);
}
__device__ __forceinline__ void st_c2(__half2* p, size_t i, cpair v) {
    const __half2 a = f2h2_sat(v.a), b = f2h2_sat(v.b);
    *reinterpret_cast<uint2*>(p + i) = make_uint2(*reinterpret_cast<const unsigned*>(&a), *reinterpret_cast<const unsigned*>(&b));
}

// A thread owns one butterfly position of TWO adjacent columns (one 8- or 16-byte global access per
// row, one 16-byte shared-memory access per element): half the memory instructions of a
// column-per-thread layout and two independent dependency chains per thread.
template <int M, class TC>
__global__ void __launch_bounds__(cols_wp(M) * M / 16) ifft_cols_kernel(const TC* __restrict__ grid,
                                                                        TC* __restrict__ pass1,
                                                                        const float2* __restrict__ tw, int strip) {
    constexpr int n = M / 2, W = cols_w(M), WP = cols_wp(M), LS = cols_stride(M);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cpair* smem = reinterpret_cast<cpair*>(smem_raw);
    const int wp = threadIdx.x % WP;          // column pair inside the CTA's strip (fastest: coalescing)
    const int tid = threadIdx.x / WP;         // thread inside the pair's FFT group
    cpair* s = smem + (size_t)wp * LS;
    const int pair = blockIdx.y;
    const int l1 = blockIdx.x * W + 2 * wp;
    // strip-major grid: the CTA's W columns are one contiguous block of M rows x W
    const TC* src = grid + (size_t)pair * M * M + (strip ? (size_t)blockIdx.x * M * W + 2 * wp : (size_t)l1);
    const size_t rstride = strip ? (size_t)W : (size_t)M;
    // pass-1 array, strip-major like the grid: [pair][M/W][n iy][W l1], so that consecutive iy of the CTA's
    // W columns are contiguous (a warp stores 256 contiguous bytes instead of 16-byte pieces 4 M bytes apart)
    TC* dst = pass1 + (size_t)pair * n * M + (size_t)blockIdx.x * n * W + 2 * wp;
    fft_line<M, true>(
        s, tid, tw, [&](int l2) { return ld_c2(src, (size_t)l2 * rstride); },
        [&](int x2, cpair v) {
            // signed x2 in [-n/2, n/2)  <->  FFT index x2 mod M
            if (x2 < n / 2) st_c2(dst, (size_t)(x2 + n / 2) * W, v);
            else if (x2 >= M - n / 2) st_c2(dst, (size_t)(x2 - (M - n / 2)) * W, v);
        });
}

// The same column pass as a persistent kernel for the strip-major grid of the fp16 path: one CTA per SM
// (its lines fill most of the shared memory), so a CTA's global loads are not hidden by another CTA's
// compute.  Here the next strip (a contiguous block of M x W half2) is copied into a staging buffer with
// cp.async while the current strip is transformed, and the first pass reads its inputs from there.
template <int M>
__global__ void __launch_bounds__(cols_wp(M) * M / 16, 1) ifft_cols_pf_kernel(const __half2* __restrict__ grid,
                                                                              __half2* __restrict__ pass1,
                                                                              const float2* __restrict__ tw, int nunits) {
    constexpr int n = M / 2, W = cols_w(M), WP = cols_wp(M), LS = cols_stride(M), NT = WP * M / 16;
    constexpr int CHUNKS = M * W * (int)sizeof(__half2) / 16;       // 16-byte pieces of a strip
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cpair* smem = reinterpret_cast<cpair*>(smem_raw);
    const __half2* stage = reinterpret_cast<const __half2*>(smem_raw + (size_t)WP * LS * sizeof(cpair));
    const uint32_t stage_u32 = (uint32_t)__cvta_generic_to_shared(stage);
    const int wp = threadIdx.x % WP, tid = threadIdx.x / WP;
    cpair* s = smem + (size_t)wp * LS;
    auto prefetch = [&](int unit) {                                  // unit = pair * (M / W) + strip: a contiguous block
        if (unit < nunits) {
            const unsigned char* g = reinterpret_cast<const unsigned char*>(grid + (size_t)unit * M * W);
#pragma unroll
            for (int c = threadIdx.x; c < CHUNKS; c += NT)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(stage_u32 + c * 16), "l"(g + (size_t)c * 16) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    prefetch(blockIdx.x);
#pragma unroll 1
    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        const int pair = unit / (M / W), strip = unit % (M / W);
        __half2* dst = pass1 + (size_t)pair * n * M + (size_t)strip * n * W + 2 * wp;
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        fft_line<M, true>(
            s, tid, tw, [&](int l2) { return ld_c2(stage, (size_t)l2 * W + 2 * wp); },
            [&](int x2, cpair v) {
                if (x2 < n / 2) st_c2(dst, (size_t)(x2 + n / 2) * W, v);
                else if (x2 >= M - n / 2) st_c2(dst, (size_t)(x2 - (M - n / 2)) * W, v);
            },
            [&]() { prefetch(unit + gridDim.x); });
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

template <int M, int ROWS, class TC, class TO>
__global__ void __launch_bounds__(ROWS* M / 16) ifft_rows_kernel(const TC* __restrict__ pass1, TO* __restrict__ out,
                                                                 const float2* __restrict__ tw,
                                                                 const float* __restrict__ deax,
                                                                 const float* __restrict__ deay, int nz) {
    constexpr int n = M / 2, TG = M / 16;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / TG, tid = threadIdx.x % TG;
    float2* s = smem + (size_t)g * padded_len(M);
    const int pair = blockIdx.y;
    const int iy = blockIdx.x * ROWS + g;     // n is a multiple of ROWS
    constexpr int W = cols_w(M);              // strip width of the pass-1 array (ifft_cols_kernel)
    const TC* src = pass1 + (size_t)pair * n * M + (size_t)iy * W;
    const float dy = __ldg(&deay[iy]);
    const int zA = 2 * pair, zB = 2 * pair + 1;
    TO* oA = out + ((size_t)zA * n + iy) * n;
    TO* oB = out + ((size_t)zB * n + iy) * n;
    const bool hasB = zB < nz;
    fft_line<M, true>(
        s, tid, tw, [&](int l1) { return ld_c(src, (size_t)(l1 / W) * n * W + (size_t)(l1 % W)); },
        [&](int x1, float2 v) {
            int ix = -1;
            if (x1 < n / 2) ix = x1 + n / 2;
            else if (x1 >= M - n / 2) ix = x1 - (M - n / 2);
            if (ix >= 0) {
                const float d = dy * __ldg(&deax[ix]);
                st_r(oA, ix, v.x * d);
                if (hasB) st_r(oB, ix, v.y * d);
            }
        });
}

template <int M, class TC>
static int launch_cols_t(const tcp_ctx* c, cudaStream_t st) {
    constexpr int W = cols_w(M), WP = cols_wp(M);
    const size_t smem = (size_t)WP * cols_stride(M) * sizeof(cpair);
    if constexpr (sizeof(TC) == sizeof(__half2)) {
        const size_t smem_pf = smem + (size_t)M * W * sizeof(__half2);
        if (c->grid_strip == W && smem_pf <= 227 * 1024 && smem > 64 * 1024) {      // long lines, one CTA per SM
            auto kpf = ifft_cols_pf_kernel<M>;
            TCP_SMEM(kpf, (int)smem_pf);
            const int nunits = (M / W) * c->npair;
            kpf<<<nunits < c->nsm ? nunits : c->nsm, WP * M / 16, smem_pf, st>>>((const __half2*)c->grid, (__half2*)c->pass1, c->tw, nunits);
            TCP_CUDA_CHECK(cudaGetLastError());
            return TCP_OK;
        }
    }
    auto kern = ifft_cols_kernel<M, TC>;
    TCP_SMEM(kern, (int)smem);
    dim3 grid(M / W, c->npair);
    kern<<<grid, WP * M / 16, smem, st>>>((const TC*)c->grid, (TC*)c->pass1, c->tw, c->grid_strip);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

template <int M, class TC, class TO>
static int launch_rows_t(const tcp_ctx* c, void* out, cudaStream_t st) {
    constexpr int TG = M / 16;
    constexpr int ROWS = (TG >= 128) ? 1 : 128 / TG;
    const size_t smem = (size_t)ROWS * padded_len(M) * sizeof(float2);
    auto kern = ifft_rows_kernel<M, ROWS, TC, TO>;
    TCP_SMEM(kern, (int)smem);
    dim3 grid((M / 2) / ROWS, c->npair);
    kern<<<grid, ROWS * TG, smem, st>>>((const TC*)c->pass1, (TO*)out, c->tw, c->deax, c->deay, c->nz);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

template <int M>
static int cols_m(const tcp_ctx* c, cudaStream_t st) {
    return c->half_store ? launch_cols_t<M, __half2>(c, st) : launch_cols_t<M, float2>(c, st);
}
template <int M>
static int rows_m(const tcp_ctx* c, void* out, cudaStream_t st) {
    if (!c->half_store) return launch_rows_t<M, float2, float>(c, out, st);
    return c->half_out ? launch_rows_t<M, __half2, __half>(c, out, st) : launch_rows_t<M, __half2, float>(c, out, st);
}

int cols_strip_width(int M) { return cols_w(M); }

int launch_ifft_cols(const tcp_ctx* c, cudaStream_t st) {
    switch (c->M) {
        case 128: return cols_m<128>(c, st);
        case 256: return cols_m<256>(c, st);
        case 512: return cols_m<512>(c, st);
        case 1024: return cols_m<1024>(c, st);
        case 2048: return cols_m<2048>(c, st);
        case 4096: return cols_m<4096>(c, st);
        case 8192: return cols_m<8192>(c, st);
    }
    return set_error(TCP_EUNSUPPORTED, "unsupported M=%d", c->M);
}

int launch_ifft_rows(const tcp_ctx* c, void* out, cudaStream_t st) {
    switch (c->M) {
        case 128: return rows_m<128>(c, out, st);
        case 256: return rows_m<256>(c, out, st);
        case 512: return rows_m<512>(c, out, st);
        case 1024: return rows_m<1024>(c, out, st);
        case 2048: return rows_m<2048>(c, out, st);
        case 4096: return rows_m<4096>(c, out, st);
        case 8192: return rows_m<8192>(c, out, st);
    }
    return set_error(TCP_EUNSUPPORTED, "unsupported M=%d", c->M);
}

}  // namespace tcpk
