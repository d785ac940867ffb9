// tcp_internal.h -- context layout and kernel launchers shared by the .cu files of libtcp.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/tcp.h"

struct tcp_ctx {
    int n, M, nproj, nz, npair, dtype, filter, m;
    int kernel;           // gridding kernel family: 0 Gaussian, 1 Kaiser-Bessel (tcp_create_ex code 16 + m)
    float* kbtab;         // Kaiser-Bessel: phi over u = 1 - (d/m)^2, KB_NTAB + 1 samples (NULL for the Gaussian)
    float center;         // rotation centre in the padded row (caller's centre + pad_l)
    int ndet, pad_l;      // tcp_create_det: caller's detector width / image side, air samples left of it (ndet == n, 0 otherwise)
    void* out_pad;        // [nz][n][n] in the output dtype when ndet != n (the central ndet x ndet pixels are then copied out)
    bool half_store;      // intermediates in half / half2 (TCP_F16, TCP_F16_OUT32)
    bool half_out;        // out in half (TCP_F16)
    double scale;         // power-of-two scale S of SPECTRUM / GRID / PASS1 (1 in fp32)
    int grid_impl;
    int filter_fused;     // TCP_OPT_FILTER_FUSED: S3 + S4 as one transform, no crop (FourierRec only)
    float2* ftab;         // [M] H[k] x ptab[k]: the fused path's table
    int pad;              // TCP_PAD_ZERO | TCP_PAD_EDGE: padding samples of the filter stage S3
    int algorithm;        // TCP_ALG_FOURIER (gridding, default) | TCP_ALG_LINE (direct line summation)
    int grid_strip;       // 0: grid rows are contiguous; W > 0: strip-major [pair][M/W][M l2][W l1] (tcgen05 gridding)
    int device, nsm;      // CUDA device and its SM count
    int tcfft;            // TCP_TCFFT_* mask of transforms whose butterflies run on the tensor cores (k_mmafft.cu)
    int tcfft_ok;         // the mask this context supports (fp16 storage, M = 4096)
    int mf_ok;            // = tcfft_ok, set by mmafft_setup
    uint32_t* mf_atab;    // mmafft.cuh: butterfly-matrix fragments [variant][lane][16]
    // workspaces (device)
    void* sino;           // [nz][nproj][n]      float | half
    void* spec;           // [npair][nproj][M]   float2 | half2   (S * G of stage S4, FFT order)
    void* grid;           // [npair][M][M]       float2 | half2   (row = l2, FFT order)
    void* pass1;          // [npair][M/W][n][W]  float2 | half2   (strip of W = cols_strip_width(M) columns l1, row = iy)
    double2* trig;        // [nproj] (cos, sin) of theta, fp64
    float4* trigf;        // [nproj] (cos hi, cos lo, sin hi, sin lo): float-float split of trig
    float* wq;            // [nproj] quadrature weight of every projection relative to pi/nproj (trig_kernel, every call)
    float2* fdtab;        // [nz][n] (1 / max(flat - dark, eps_d), dark) of the call, written by trig_kernel for the fused S1+S2 loader
    double zinger_dif;    // TCP_PARAM_ZINGER_DIF (0: off) and TCP_PARAM_RING_ALPHA (0: off): pre-processing between S2 and S3 (k_pre.cu)
    double ring_alpha;
    double* pre_buf;      // ring removal: [nz][n] angle means + [nz][5][n] solver work, allocated when the option is first set
    int fuse_norm;        // TCP_OPT_FUSE_NORMALIZE: S1+S2 in the loader of rows_kernel where that applies (fp16 storage)
    int angle_weights;    // TCP_OPT_ANGLE_WEIGHTS: the row kernels scale projection j by wq[j] (unequally spaced angles)
    // tables (device), built in fp64 on the host at create
    float2* tw;           // [M] e^{-2 pi i t / M}
    float* hfilt;         // [M] H[k] / M
    float2* ptab;         // [M] S * C * e^{+2 pi i k c / M}, k signed; 0 at k = M/2
    float2* try_ptab;     // tcp_recon_try: [npair][M] two-centre phase tables (NULL outside a try call's context copy)
    float2* try_buf;      // its device storage, [ceil(nz/2)][M], allocated on first use
    float* deax;          // [n] 1 / (S * Phi(x))
    float* deay;          // [n] 1 / Phi(y)
    int* tile_order;      // gather gridding: tiles sorted by decreasing work
    int ntiles;
    // tile gridding (k_grid_tile.cu): work items, split-tile reduce list, partial tiles, per-call plan
    int4* g_items;
    int4* g_red;
    float2* g_partial;
    int2* g_plan;
    // weight cache of the tcgen05 gridding (k_grid_mma.cu): per-step records, built on the device when theta changes
    int* w_state; int* w_count; int* w_off; uint4* w_rec; unsigned* w_samp; int w_cap, w_enable;
    int grid_dirty;          // 1: the grid workspace must be zeroed before the next tile / tensor-core gridding (they never write the empty corner tiles)
    volatile int* w_hflag;   // pinned, mapped: the last wc_decide_kernel's verdict (1: the cache must be rebuilt) as the host may see it, late
    float* w_theta;       // [nproj] the angles the cached weights were built for (compared element by element on every call)
    int* g_counter;       // [64] next-item counters of the persistent gridding CTAs, zeroed by the plan kernel
    int g_nitems, g_nred;
    size_t bytes;
    // per-kernel profiling (TCP_OPT_PROFILE): ring of event sets, TCP_NSTAGES + 1 events per call
    bool profile;
    cudaEvent_t* pev;
    int pcalls;           // calls recorded since the last collect
    // chunk pipeline (lazily created by tcp_recon_volume_host)
    struct Pipe* pipe;
};

// The tensor-core transforms of the inverse 2D transform (k_mmafft.cu) take their input lines straight into their
// swizzled shared-memory layout with one bulk copy, so their producers store rows pre-permuted: the gridding writes
// row l2 of a grid strip at position swz<4>(l2), the column pass writes column l1 of a row pair at swz<2>(l1).
static inline bool ifft2_on_mma(const tcp_ctx* c) {
    return (c->tcfft & (TCP_TCFFT_COLS | TCP_TCFFT_IROWS)) == (TCP_TCFFT_COLS | TCP_TCFFT_IROWS) && c->grid_strip == 4;
}

namespace tcpk {

int set_error(int code, const char* fmt, ...);
#define TCP_CUDA_CHECK(expr)                                                                   \
    do {                                                                                       \
        cudaError_t e__ = (expr);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return tcpk::set_error(TCP_ECUDA, "%s failed: %s (%s:%d)", #expr,                  \
                                   cudaGetErrorString(e__), __FILE__, __LINE__);               \
    } while (0)

// Opt a kernel into `bytes` of dynamic shared memory ONCE per (device, kernel): cudaFuncSetAttribute is a host API
// call, so the launchers memoise it instead of repeating it on every launch of every chunk.
int ensure_smem(const void* kern, int bytes);
#define TCP_SMEM(kern, bytes)                                                     \
    do {                                                                          \
        int rc__ = tcpk::ensure_smem((const void*)(kern), (int)(bytes));          \
        if (rc__ != TCP_OK) return rc__;                                          \
    } while (0)

// kernel launchers: each enqueues on `st` and returns TCP_OK or an error code
// flat != NULL: also fill c->fdtab from the call's flat / dark (fused S1+S2 loader of rows_kernel)
int launch_trig(const tcp_ctx* c, const float* theta, cudaStream_t st, const float* flat = nullptr, const float* dark = nullptr);
int launch_normalize(const tcp_ctx* c, const uint16_t* raw, const float* flat, const float* dark,
                     cudaStream_t st);
// raw != NULL: S1+S2 fused into the loader (rows_fuses_normalize(c) must hold); else the sinogram workspace is read
int launch_rows(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw = nullptr, const float* flat = nullptr,
                const float* dark = nullptr);
bool rows_fuses_normalize(const tcp_ctx* c);
int launch_filter(const tcp_ctx* c, cudaStream_t st);
int launch_pre(const tcp_ctx* c, cudaStream_t st);          // zinger / ring removal on the sinogram workspace
int launch_line_bp(const tcp_ctx* c, void* out, cudaStream_t st);
int launch_grid_scatter(const tcp_ctx* c, cudaStream_t st);
int launch_grid_gather(const tcp_ctx* c, const float* theta, cudaStream_t st);
int launch_grid_tile(const tcp_ctx* c, const float* theta, cudaStream_t st);
int launch_grid_mma_main(const tcp_ctx* c, const float* theta, cudaStream_t st);
int grid_mma_cache_setup(tcp_ctx* c);
void grid_mma_cache_free(tcp_ctx* c);
int grid_tile_setup(tcp_ctx* c);
void grid_tile_free(tcp_ctx* c);
int launch_ifft_cols(const tcp_ctx* c, cudaStream_t st);
int cols_strip_width(int M);
int launch_ifft_rows(const tcp_ctx* c, void* out, cudaStream_t st);
int mmafft_setup(tcp_ctx* c);
void mmafft_free(tcp_ctx* c);
int launch_rows_mma(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw);
int launch_cols_mma(const tcp_ctx* c, cudaStream_t st);
int launch_irows_mma(const tcp_ctx* c, void* out, cudaStream_t st);
int launch_fft_lines(const tcp_ctx* c, const void* in, void* out, int batch, int inverse, cudaStream_t st);
int launch_crop_out(const tcp_ctx* c, int nslices, void* out, cudaStream_t st);
int launch_mean_frames(const uint16_t* frames, int nframes, int nz, int n, float* mean, cudaStream_t st);
int setup_kernel_attributes(const tcp_ctx* c);
void pipe_destroy(tcp_ctx* c);

// storage <-> fp32 helpers
__device__ __forceinline__ float2 ld_c(const float2* p, size_t i) { return p[i]; }
__device__ __forceinline__ float2 ld_c(const __half2* p, size_t i) { return __half22float2(p[i]); }
__device__ __forceinline__ void st_c(float2* p, size_t i, float2 v) { p[i] = v; }
// fp32 -> half with saturation to +-65504 (cvt.rn.satfinite): a hot or dead detector pixel must not turn into inf and then,
// through the transforms, into a slice pair of NaN
__device__ __forceinline__ __half2 f2h2_sat(float2 v) {
    unsigned r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(v.y), "f"(v.x));
    return *reinterpret_cast<__half2*>(&r);
}
__device__ __forceinline__ __half f2h_sat(float v) {
    unsigned short r;
    asm("cvt.rn.satfinite.f16.f32 %0, %1;" : "=h"(r) : "f"(v));
    return *reinterpret_cast<__half*>(&r);
}
__device__ __forceinline__ void st_c(__half2* p, size_t i, float2 v) { p[i] = f2h2_sat(v); }
__device__ __forceinline__ float ld_r(const float* p, size_t i) { return p[i]; }
__device__ __forceinline__ float ld_r(const __half* p, size_t i) { return __half2float(p[i]); }
__device__ __forceinline__ void st_r(float* p, size_t i, float v) { p[i] = v; }
__device__ __forceinline__ void st_r(__half* p, size_t i, float v) { p[i] = f2h_sat(v); }

// S1+S2 for fp16 storage (normalize_half_kernel and the fused loader of rows_kernel share these, so both give the
// same half value bit for bit): hardware approximations (~2^-22) under a rounding to 2^-11
__device__ __forceinline__ float fast_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// uint16 -> float without the conversion pipe: 0x4B000000 | u is 2^23 + u exactly
__device__ __forceinline__ float u16f(unsigned u) { return __uint_as_float(0x4B000000u | u) - 8388608.f; }

}  // namespace tcpk
