// k_tcfft.cu -- row pass of the inverse 2D transform (S6 pass 2 + S7) for fp16 storage at M = 4096
// (config C4) as DFT-as-GEMM on the tensor cores (tcfft.cuh): same input, output and layout as
// ifft_rows_kernel (k_ifft2.cu).  Opt-in through TCP_OPT_TCFFT: it is parity-green but measured slower
// than the Stockham kernel (profiles/r1_tcfft.md).  (PAPER.md:61, :173, :300.)
// CTAs are persistent (the 32 KB matrix is loaded once per CTA); every group of 128 threads walks lines.
#include "tcfft.cuh"
#include "tcp_internal.h"

namespace tcpk {

using namespace tcfft;

constexpr int TC_M = 4096, TC_N = 2048;

__device__ __forceinline__ void st_out8(__half* p, const float* v) {
    *reinterpret_cast<uint4*>(p) = make_uint4(pack_half2(v[0], v[1]), pack_half2(v[2], v[3]), pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
}
__device__ __forceinline__ void st_out8(float* p, const float* v) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}

// ---------------------------------------------------------------------------------------
// pass 2 of the inverse 2D transform: line = row iy of pass1[pair] (4096 half2 along l1).
// IFFT by the swap identity: D rows c = 0 hold Im (slice 2 pair + 1), c = 1 hold Re (slice 2 pair).
// Kept outputs x1 in [-n/2, n/2) are natural indices [0, 1024) and [3072, 4096): rows k2 < 16 and
// k2 >= 48, i.e. lane quarters 0 and 3 only; ix = (x1 + n/2) mod M.
template <int NG, class TO>
__global__ void __launch_bounds__(128 * NG, 1) ifft_rows_tc_kernel(const __half2* __restrict__ pass1, TO* __restrict__ out,
                                                                   const uint4* __restrict__ amat,
                                                                   const float* __restrict__ deax, const float* __restrict__ deay,
                                                                   int nz, int npair) {
    extern __shared__ __align__(128) unsigned char smem[];
    using C = Cta<1, NG>;
    Group<1> g = C::setup(smem, amat);
    const Twid tw = make_twid(g);
    const int grp = threadIdx.x >> 7;
    const int nlines = npair * TC_N, step = gridDim.x * NG;
    int ln = blockIdx.x * NG + grp;
    LineRegs pf;
    // pass-1 array: [pair][M/4][n iy][4 l1] (k_ifft2.cu)
    auto line_base = [&](int l) { return pass1 + (size_t)(l / TC_N) * TC_N * TC_M + (size_t)(l % TC_N) * 4; };
    if (ln < nlines) fetch_line_strip4(g, line_base(ln), (size_t)TC_N * 4, pf);
    for (; ln < nlines; ln += step) {
        const int pair = ln / TC_N, iy = ln % TC_N;
        put_line_c<1, true>(g, 0, pf);
        if (ln + step < nlines) fetch_line_strip4(g, line_base(ln + step), (size_t)TC_N * 4, pf);
        stage_mma<1, false>(g, 0xffu);
        twiddle_step(g, tw);
        stage_mma<1, true>(g, 0xffu);
        if (g.q == 0 || g.q == 3) {
            const int k2 = 16 * g.q + g.j;
            const int ix0 = (64 * k2 + TC_N / 2) & (TC_M - 1);
            const int z = 2 * pair + (g.c ? 0 : 1);
            if (z < nz) {
                const float dy = __ldg(&deay[iy]);
                TO* dst = out + ((size_t)z * TC_N + iy) * TC_N + ix0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    uint32_t r[32];
                    ld_d(g, 0, h, r);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float4 da = __ldg(reinterpret_cast<const float4*>(deax + ix0 + 32 * h + 8 * e));
                        const float4 db = __ldg(reinterpret_cast<const float4*>(deax + ix0 + 32 * h + 8 * e) + 1);
                        const float dx[8] = {da.x, da.y, da.z, da.w, db.x, db.y, db.z, db.w};
                        float v[8];
#pragma unroll
                        for (int u = 0; u < 8; ++u) v[u] = __uint_as_float(r[8 * e + u]) * (dy * dx[u]);
                        st_out8(dst + 32 * h + 8 * e, v);
                    }
                }
            }
        }
    }
    C::teardown(g);
}

template <int NG, class TO>
static int launch_ifft_rows_tc_t(const tcp_ctx* c, void* out, cudaStream_t st) {
    using C = Cta<1, NG>;
    auto kern = ifft_rows_tc_kernel<NG, TO>;
    TCP_SMEM(kern, C::total);
    const int nlines = c->npair * TC_N;
    int ctas = c->nsm;
    if (ctas * NG > nlines) ctas = (nlines + NG - 1) / NG;
    kern<<<ctas, C::threads, C::total, st>>>((const __half2*)c->pass1, (TO*)out, (const uint4*)c->tc_amat, c->deax,
                                              c->deay, c->nz, c->npair);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_ifft_rows_tc(const tcp_ctx* c, void* out, cudaStream_t st) {
    if (c->half_out) return launch_ifft_rows_tc_t<4, __half>(c, out, st);
    return launch_ifft_rows_tc_t<4, float>(c, out, st);
}

}  // namespace tcpk
