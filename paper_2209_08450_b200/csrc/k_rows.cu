// k_rows.cu -- S3 + S4 for one detector row of a slice pair, entirely in shared memory:
//   a = [pA + i pB, 0]  -> FFT_M -> * H/M -> IFFT_M -> crop to [0,n), zero-pad -> FFT_M
//   -> * S C e^{+2 pi i k c / M}  -> spectrum G[pair][j][k]
// Two adjacent slices ride one complex transform (slice 2p -> real, 2p+1 -> imaginary):
// H is real and even and the Nyquist bin is zeroed, so the packing survives the filter.
// HBM sees one read of the two sinogram rows and one write of the spectrum row.
#include "fft.cuh"
#include "tcp_internal.h"

namespace tcpk {

// RAW: the two rows come straight from the uint16 projections raw[nproj][nz][n] with fdtab[nz][n] = (1 / max(flat - dark,
// eps_d), dark) of this call (trig_kernel): S1+S2 run in the
// loader with the arithmetic of normalize_half_kernel (same half value bit for bit, rounded to the storage type before
// use), so the sinogram never goes to HBM and back (TCP_OPT_FUSE_NORMALIZE; fp16 storage only).
template <int M, int ROWS, bool PAD_EDGE, bool RAW, class TS, class TC>
__global__ void __launch_bounds__(ROWS* M / 16) rows_kernel(const TS* __restrict__ sino, TC* __restrict__ spec,
                                                            const float2* __restrict__ tw,
                                                            const float* __restrict__ hfilt,
                                                            const float2* __restrict__ ptab, int nproj, int nz, int try_mode,
                                                            const float* __restrict__ wq, const uint16_t* __restrict__ raw,
                                                            const float2* __restrict__ fdtab) {
    constexpr bool pad_edge = PAD_EDGE;
    constexpr int n = M / 2;
    constexpr int TG = M / 16;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / TG;       // row group inside the CTA
    const int tid = threadIdx.x % TG;
    float2* s = smem + (size_t)g * padded_len(M);
    int j = blockIdx.x * ROWS + g;
    const bool live = j < nproj;
    if (!live) j = nproj - 1;             // keep the group in the barriers; its stores are masked
    const int pair = blockIdx.y;
    // try mode (tcp_recon_try): every pair transforms slice 0 alone and carries the phases of two candidate
    // centres in its own table ptab[pair][M] = S C (e^{2 pi i k c1/M} + i e^{2 pi i k c2/M})
    const int zA = try_mode ? 0 : 2 * pair, zB = try_mode ? nz : 2 * pair + 1;
    const TS* pA = sino + ((size_t)zA * nproj + j) * n;
    const TS* pB = sino + ((size_t)(zB < nz ? zB : zA) * nproj + j) * n;
    const bool hasB = zB < nz;
    if (try_mode) ptab += (size_t)pair * M;
    const float wj = wq ? __ldg(&wq[j]) : 1.f;      // TCP_OPT_ANGLE_WEIGHTS: everything after S2 is linear in the projection

    const int zBs = hasB ? zB : zA;
    auto neglog_raw = [&](int z, int i) {
        const float2 fd = __ldg(&fdtab[(size_t)z * n + i]);
        const float p = -0.69314718055994531f * fast_lg2(fmaxf((u16f(__ldg(&raw[((size_t)j * nz + z) * n + i])) - fd.y) * fd.x, 1e-6f));
        return __half2float(__float2half_rn(p));
    };
    auto load_padded = [&](int i) {
        // padding samples: zeros, or (TCP_OPT_PAD = TCP_PAD_EDGE) the nearest edge of the periodic row
        if (i >= n) {
            if (!pad_edge) return make_float2(0.f, 0.f);
            i = (i < n + n / 2) ? n - 1 : 0;
        }
        if constexpr (RAW) return make_float2(neglog_raw(zA, i) * wj, hasB ? neglog_raw(zBs, i) * wj : 0.f);
        else return make_float2(ld_r(pA, i) * wj, hasB ? ld_r(pB, i) * wj : 0.f);
    };
    TC* out = spec + ((size_t)pair * nproj + j) * M;
    // the three transforms hand their lines over in registers (fft_chain_slot: same elements, permuted slots):
    // no shared-memory round trip and no barrier at the two boundaries; results are bit-identical
    float2 keep[16];
    // FFT #1: zero-padded load, filter on the way out
    fft_line<M, false>(s, tid, tw, load_padded, [&](int k, float2 v, int slot) {
        const float h = __ldg(&hfilt[k]);
        keep[fft_chain_slot<M>(slot)] = make_float2(v.x * h, v.y * h);
    });
    // FFT #2 (inverse): crop to the detector on the way out
    fft_line<M, true>(s, tid, tw, [&](int, int slot) { return keep[slot]; },
                      [&](int i, float2 v, int slot) { keep[fft_chain_slot<M>(slot)] = (i < n) ? v : make_float2(0.f, 0.f); });
    // FFT #3: spectrum, centre phase and scale on store
    fft_line<M, false>(s, tid, tw, [&](int, int slot) { return keep[slot]; }, [&](int k, float2 v) {
        if (live) st_c(out, k, cmul(v, __ldg(&ptab[k])));
    });
}

// S3 + S4 fused without the crop (TCP_OPT_FILTER_FUSED; SURVEY 8(c) Q6's second reading, an option): one
// transform, G = FFT_M(padded row) x (H x S C e^{+2 pi i k c/M}); the table carries the whole product.
template <int M, int ROWS, bool PAD_EDGE, class TS, class TC>
__global__ void __launch_bounds__(ROWS* M / 16) rows_fused_kernel(const TS* __restrict__ sino, TC* __restrict__ spec,
                                                                  const float2* __restrict__ tw,
                                                                  const float2* __restrict__ ftab, int nproj, int nz,
                                                                  const float* __restrict__ wq) {
    constexpr int n = M / 2;
    constexpr int TG = M / 16;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / TG;
    const int tid = threadIdx.x % TG;
    float2* s = smem + (size_t)g * padded_len(M);
    int j = blockIdx.x * ROWS + g;
    const bool live = j < nproj;
    if (!live) j = nproj - 1;
    const int pair = blockIdx.y;
    const int zA = 2 * pair, zB = 2 * pair + 1;
    const bool hasB = zB < nz;
    const TS* pA = sino + ((size_t)zA * nproj + j) * n;
    const TS* pB = sino + ((size_t)(hasB ? zB : zA) * nproj + j) * n;
    TC* out = spec + ((size_t)pair * nproj + j) * M;
    const float wj = wq ? __ldg(&wq[j]) : 1.f;
    fft_line<M, false>(
        s, tid, tw,
        [&](int i) {
            if (i >= n) {
                if (!PAD_EDGE) return make_float2(0.f, 0.f);
                i = (i < n + n / 2) ? n - 1 : 0;
            }
            return make_float2(ld_r(pA, i) * wj, hasB ? ld_r(pB, i) * wj : 0.f);
        },
        [&](int k, float2 v) {
            if (live) st_c(out, k, cmul(v, __ldg(&ftab[k])));
        });
}

// S3 alone, for the line-summation operator (k_line.cu): the same two transforms, the cropped filtered
// rows written back over the two sinogram rows they came from (each CTA reads its rows completely before
// the first pass ends and writes them in the last pass of the inverse transform).
template <int M, int ROWS, class TS>
__global__ void __launch_bounds__(ROWS* M / 16) filter_kernel(TS* __restrict__ sino, const float2* __restrict__ tw,
                                                              const float* __restrict__ hfilt, int nproj, int nz, int pad_edge,
                                                              const float* __restrict__ wq) {
    constexpr int n = M / 2;
    constexpr int TG = M / 16;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / TG;
    const int tid = threadIdx.x % TG;
    float2* s = smem + (size_t)g * padded_len(M);
    int j = blockIdx.x * ROWS + g;
    const bool live = j < nproj;
    if (!live) j = nproj - 1;
    const int pair = blockIdx.y;
    const int zA = 2 * pair, zB = 2 * pair + 1;
    const bool hasB = zB < nz;
    TS* pA = sino + ((size_t)zA * nproj + j) * n;
    TS* pB = sino + ((size_t)(hasB ? zB : zA) * nproj + j) * n;
    const float wj = wq ? __ldg(&wq[j]) : 1.f;
    float2 keep[16];
    fft_line<M, false>(
        s, tid, tw,
        [&](int i) {
            // padding samples: zeros, or (TCP_OPT_PAD = TCP_PAD_EDGE) the nearest edge of the periodic row
            if (i >= n) {
                if (!pad_edge) return make_float2(0.f, 0.f);
                i = (i < n + n / 2) ? n - 1 : 0;
            }
            return make_float2(ld_r(pA, i) * wj, hasB ? ld_r(pB, i) * wj : 0.f);
        },
        [&](int k, float2 v, int slot) {
            const float h = __ldg(&hfilt[k]);
            keep[fft_chain_slot<M>(slot)] = make_float2(v.x * h, v.y * h);      // handed over in registers (fft.cuh)
        });
    fft_line<M, true>(
        s, tid, tw, [&](int, int slot) { return keep[slot]; },
        [&](int i, float2 v) {
            if (live && i < n) {
                st_r(pA, i, v.x);
                if (hasB) st_r(pB, i, v.y);
            }
        });
}

template <int M, class TS>
static int launch_filter_t(const tcp_ctx* c, cudaStream_t st) {
    constexpr int TG = M / 16;
    constexpr int ROWS = (TG >= 128) ? 1 : 128 / TG;
    const size_t smem = (size_t)ROWS * padded_len(M) * sizeof(float2);
    auto kern = filter_kernel<M, ROWS, TS>;
    TCP_SMEM(kern, (int)smem);
    dim3 grid((c->nproj + ROWS - 1) / ROWS, c->npair);
    kern<<<grid, ROWS * TG, smem, st>>>((TS*)c->sino, c->tw, c->hfilt, c->nproj, c->nz, c->pad, c->angle_weights ? c->wq : nullptr);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

template <int M>
static int launch_filter_m(const tcp_ctx* c, cudaStream_t st) {
    return c->half_store ? launch_filter_t<M, __half>(c, st) : launch_filter_t<M, float>(c, st);
}

int launch_filter(const tcp_ctx* c, cudaStream_t st) {
    switch (c->M) {
        case 128: return launch_filter_m<128>(c, st);
        case 256: return launch_filter_m<256>(c, st);
        case 512: return launch_filter_m<512>(c, st);
        case 1024: return launch_filter_m<1024>(c, st);
        case 2048: return launch_filter_m<2048>(c, st);
        case 4096: return launch_filter_m<4096>(c, st);
        case 8192: return launch_filter_m<8192>(c, st);
    }
    return set_error(TCP_EUNSUPPORTED, "unsupported M=%d", c->M);
}

template <int M, class TS, class TC>
static int launch_rows_t(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw, const float* flat, const float* dark) {
    constexpr int TG = M / 16;
    constexpr int ROWS = (TG >= 128) ? 1 : 128 / TG;
    const size_t smem = (size_t)ROWS * padded_len(M) * sizeof(float2);
    if (c->filter_fused && !c->try_ptab) {
        auto kf = c->pad ? rows_fused_kernel<M, ROWS, true, TS, TC> : rows_fused_kernel<M, ROWS, false, TS, TC>;
        TCP_SMEM(kf, (int)smem);
        kf<<<dim3((c->nproj + ROWS - 1) / ROWS, c->npair), ROWS * TG, smem, st>>>((const TS*)c->sino, (TC*)c->spec, c->tw, c->ftab, c->nproj,
                                                                                   c->nz, c->angle_weights ? c->wq : nullptr);
        TCP_CUDA_CHECK(cudaGetLastError());
        return TCP_OK;
    }
    auto kern = c->pad ? rows_kernel<M, ROWS, true, false, TS, TC> : rows_kernel<M, ROWS, false, false, TS, TC>;
    if constexpr (std::is_same_v<TS, __half>) {
        if (raw) kern = c->pad ? rows_kernel<M, ROWS, true, true, TS, TC> : rows_kernel<M, ROWS, false, true, TS, TC>;
    }
    TCP_SMEM(kern, (int)smem);
    dim3 grid((c->nproj + ROWS - 1) / ROWS, c->npair);
    kern<<<grid, ROWS * TG, smem, st>>>((const TS*)c->sino, (TC*)c->spec, c->tw, c->hfilt, c->try_ptab ? c->try_ptab : c->ptab, c->nproj, c->nz,
                                       c->try_ptab ? 1 : 0, c->angle_weights ? c->wq : nullptr, raw, c->fdtab);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

template <int M>
static int launch_rows_m(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw, const float* flat, const float* dark) {
    return c->half_store ? launch_rows_t<M, __half, __half2>(c, st, raw, flat, dark) : launch_rows_t<M, float, float2>(c, st, nullptr, nullptr, nullptr);
}

// S1+S2 can ride the loader of rows_kernel: fp16 storage (the fused value is the stored half, bit for bit), the default
// chain (not the uncropped-filter option, not the try mode), the caller's rows as wide as the transform's
bool rows_fuses_normalize(const tcp_ctx* c) {
    return c->fuse_norm && c->half_store && c->algorithm == TCP_ALG_FOURIER && !c->filter_fused && !c->try_ptab && c->ndet == c->n &&
           !(c->zinger_dif > 0.0) && !(c->ring_alpha > 0.0);       // pre-processing works on the sinogram workspace
}

int launch_rows(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw, const float* flat, const float* dark) {
    if (raw && !rows_fuses_normalize(c)) return set_error(TCP_EINVAL, "fused S1+S2 not available on this context");
    switch (c->M) {
        case 128: return launch_rows_m<128>(c, st, raw, flat, dark);
        case 256: return launch_rows_m<256>(c, st, raw, flat, dark);
        case 512: return launch_rows_m<512>(c, st, raw, flat, dark);
        case 1024: return launch_rows_m<1024>(c, st, raw, flat, dark);
        case 2048: return launch_rows_m<2048>(c, st, raw, flat, dark);
        case 4096: return launch_rows_m<4096>(c, st, raw, flat, dark);
        case 8192: return launch_rows_m<8192>(c, st, raw, flat, dark);
    }
    return set_error(TCP_EUNSUPPORTED, "unsupported M=%d", c->M);
}

}  // namespace tcpk
