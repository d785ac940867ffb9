// tcp_api.cu -- the C ABI of include/tcp.h: context, tables (built in fp64 on the host),
// validation, error reporting and the per-chunk launch sequence S1..S7.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <vector>

#include "grid_common.cuh"
#include "tcp_internal.h"

namespace tcpk {

static thread_local char g_err[512] = "";

int set_error(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// (device, kernel) -> largest dynamic shared-memory size set so far
int ensure_smem(const void* kern, int bytes) {
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, int> done;
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(mu);
    int& have = done[std::make_pair(dev, kern)];
    if (have >= bytes && have > 0) return TCP_OK;
    if (bytes > 48 * 1024 || have > 0) TCP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    have = bytes > 0 ? bytes : 1;
    return TCP_OK;
}

static const int kProfileRing = 512;
static const double kPi = 3.14159265358979323846264338327950288;

// H[k]/M: band-limited ramp (h[0] = 1/4, h[i] = -1/(pi^2 i^2) for odd i) transformed as a real
// cosine series, times the window; Nyquist bin zeroed (reading Q4).
static void build_filter(int M, int filter, std::vector<float>& out) {
    out.resize(M);
    std::vector<double> coef;   // 2 h[i] for odd i in (0, M/2)
    for (int i = 1; i < M / 2; i += 2) coef.push_back(-2.0 / (kPi * kPi * (double)i * (double)i));
    for (int k = 0; k <= M / 2; ++k) {
        double r = 0.25;
        // sum small terms first for accuracy
        for (int t = (int)coef.size() - 1; t >= 0; --t) {
            long long ki = ((long long)k * (2 * t + 1)) % M;
            r += coef[t] * cos(2.0 * kPi * (double)ki / (double)M);
        }
        double w = 1.0;
        if (filter == TCP_FILTER_SHEPP) {
            double a = kPi * (double)k / (double)M;
            w = (k == 0) ? 1.0 : sin(a) / a;
        } else if (filter == TCP_FILTER_PARZEN) {
            double u = (double)k / (double)(M / 2);
            w = (u <= 0.5) ? 1.0 - 6.0 * u * u * (1.0 - u) : 2.0 * (1.0 - u) * (1.0 - u) * (1.0 - u);
        } else if (filter == TCP_FILTER_COSINE || filter == TCP_FILTER_HANN || filter == TCP_FILTER_HAMMING) {
            const double u = (double)k / (double)(M / 2);       // "or other filter": textbook apodisation windows
            w = filter == TCP_FILTER_COSINE ? cos(0.5 * kPi * u) : filter == TCP_FILTER_HANN ? 0.5 * (1.0 + cos(kPi * u)) : 0.54 + 0.46 * cos(kPi * u);
        }
        double h = (k == M / 2) ? 0.0 : r * w / (double)M;
        out[k] = (float)h;
        if (k > 0 && k < M / 2) out[M - k] = (float)h;
    }
}

template <class T>
static int upload(T** dptr, const std::vector<T>& h, size_t* bytes) {
    TCP_CUDA_CHECK(cudaMalloc((void**)dptr, h.size() * sizeof(T)));
    TCP_CUDA_CHECK(cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    *bytes += h.size() * sizeof(T);
    return TCP_OK;
}

static int dev_alloc(void** p, size_t nbytes, size_t* bytes) {
    cudaError_t e = cudaMalloc(p, nbytes);
    if (e != cudaSuccess) {
        *p = nullptr;
        return set_error(e == cudaErrorMemoryAllocation ? TCP_ENOMEM : TCP_ECUDA, "cudaMalloc(%zu) failed: %s", nbytes,
                         cudaGetErrorString(e));
    }
    *bytes += nbytes;
    return TCP_OK;
}

static int build_context(tcp_ctx* c) {
    const int n = c->n, M = c->M, m = c->m;
    const size_t rb = c->half_store ? 2 : 4, cb = 2 * rb;
    int rc;
    if ((rc = dev_alloc(&c->sino, (size_t)c->nz * c->nproj * n * rb, &c->bytes))) return rc;
    if ((rc = dev_alloc(&c->spec, (size_t)c->npair * c->nproj * M * cb, &c->bytes))) return rc;
    if ((rc = dev_alloc(&c->grid, (size_t)c->npair * M * M * cb, &c->bytes))) return rc;
    if ((rc = dev_alloc(&c->pass1, (size_t)c->npair * n * M * cb, &c->bytes))) return rc;
    if ((rc = dev_alloc((void**)&c->trig, (size_t)c->nproj * sizeof(double2), &c->bytes))) return rc;
    if ((rc = dev_alloc((void**)&c->trigf, (size_t)c->nproj * sizeof(float4), &c->bytes))) return rc;
    if ((rc = dev_alloc((void**)&c->wq, (size_t)c->nproj * sizeof(float), &c->bytes))) return rc;
    if (c->half_store && (rc = dev_alloc((void**)&c->fdtab, (size_t)c->nz * n * sizeof(float2), &c->bytes))) return rc;

    std::vector<float2> tw(M);
    for (int t = 0; t < M; ++t) {
        double a = -2.0 * kPi * (double)t / (double)M;
        tw[t] = make_float2((float)cos(a), (float)sin(a));
    }
    if ((rc = upload(&c->tw, tw, &c->bytes))) return rc;

    std::vector<float> hf;
    build_filter(M, c->filter, hf);
    if ((rc = upload(&c->hfilt, hf, &c->bytes))) return rc;

    const double C = kPi / ((double)c->nproj * (double)M);
    std::vector<float2> pt(M);
    for (int k = 0; k < M; ++k) {
        int ks = (k < M / 2) ? k : k - M;
        double fr = fmod((double)ks * (double)c->center, (double)M) / (double)M;
        double a = 2.0 * kPi * fr;
        pt[k] = make_float2((float)(c->scale * C * cos(a)), (float)(c->scale * C * sin(a)));
    }
    pt[M / 2] = make_float2(0.f, 0.f);
    if ((rc = upload(&c->ptab, pt, &c->bytes))) return rc;
    {   // fused path: (H[k]/M) M x ptab[k]
        std::vector<float2> ft(M);
        for (int k = 0; k < M; ++k) {
            const double h = (double)hf[k] * (double)M;
            ft[k] = make_float2((float)(h * (double)pt[k].x), (float)(h * (double)pt[k].y));
        }
        if ((rc = upload(&c->ftab, ft, &c->bytes))) return rc;
    }

    const double alpha = kPi / (sqrt(2.0) * (double)m);
    // Kaiser-Bessel window (tcp_create_ex kernel code 16 + m; reading Q21): beta = pi sqrt(2.25 m^2 - 0.8),
    // phi(t) = I0(beta sqrt(1 - (t/m)^2)) / I0(beta), Phi(x) = (2m / I0(beta)) sinh(z) / z with z^2 = beta^2 - (2 pi m x / M)^2
    const double beta = kPi * sqrt(2.25 * (double)m * (double)m - 0.8);
    auto i0 = [](double z) {
        const double q = 0.25 * z * z;
        double term = 1.0, sum = 1.0;
        for (int k = 1; k < 200 && term > 1e-18 * sum; ++k) { term *= q / ((double)k * (double)k); sum += term; }
        return sum;
    };
    if (c->kernel == 1) {
        std::vector<float> kb(tcpk::KB_NTAB + 1);
        for (int i = 0; i <= tcpk::KB_NTAB; ++i) kb[i] = (float)(i0(beta * sqrt((double)i / (double)tcpk::KB_NTAB)) / i0(beta));
        if ((rc = upload(&c->kbtab, kb, &c->bytes))) return rc;
    }
    std::vector<float> dx(n), dy(n);
    for (int i = 0; i < n; ++i) {
        double x = (double)(i - n / 2);
        double phi = sqrt(kPi / alpha) * exp(-kPi * kPi * x * x / (alpha * (double)M * (double)M));
        if (c->kernel == 1) {
            const double a = 2.0 * kPi * (double)m * x / (double)M, z = sqrt(beta * beta - a * a);     // |x| <= n/2: a <= pi m / 2 < beta
            phi = 2.0 * (double)m * sinh(z) / (z * i0(beta));
        }
        dy[i] = (float)(1.0 / phi);
        dx[i] = (float)(1.0 / (phi * c->scale));
    }
    if ((rc = upload(&c->deax, dx, &c->bytes))) return rc;
    if ((rc = upload(&c->deay, dy, &c->bytes))) return rc;

    if ((rc = mmafft_setup(c))) return rc;
    c->tcfft_ok = c->mf_ok;
    c->tcfft = c->tcfft_ok;      // default: every transform that can runs its butterflies on the tensor cores

    // gather tiles, heaviest (closest to DC) first: sample density falls as 1/radius
    const int T = 16, tx = M / T;
    std::vector<std::pair<long long, int>> key;
    auto mind = [&](int t) {
        long long best = 1LL << 60;
        for (int q = 0; q < T; ++q) {
            int L = t * T + q, l = (L < n) ? L : L - M;
            best = std::min<long long>(best, llabs((long long)l));
        }
        return best;
    };
    for (int ty = 0; ty < tx; ++ty)
        for (int txi = 0; txi < tx; ++txi) {
            long long a = mind(txi), b = mind(ty);
            key.push_back({a * a + b * b, ty * tx + txi});
        }
    std::sort(key.begin(), key.end());
    std::vector<int> order;
    for (auto& kv : key) order.push_back(kv.second);
    c->ntiles = (int)order.size();
    if ((rc = upload(&c->tile_order, order, &c->bytes))) return rc;
    return grid_tile_setup(c);
}

// which transforms take the tensor-core butterflies (TCP_OPT_TCFFT; k_mmafft.cu): the row kernel unless the uncropped
// filter option is on; the two passes of S6 together (they share the row-pair layout of the pass-1 array) when the
// grid is strip-major with strips of 4 columns, i.e. written by the tensor-core gridding
static bool rows_on_mma(const tcp_ctx* c) { return (c->tcfft & TCP_TCFFT_ROWS) && !(c->filter_fused && !c->try_ptab); }

// tcp_recon_try: candidate centres of up to kMax / 2 pairs by value (a negative entry = no slice B in the last pair)
struct TryCentres {
    static constexpr int kMax = 256;
    float c[kMax];
};

__global__ void try_ptab_kernel(float2* __restrict__ ptab, TryCentres tc, int M, double SC) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x, p = blockIdx.y;
    if (k >= M) return;
    const int ks = (k < M / 2) ? k : k - M;
    double re = 0.0, im = 0.0;
    for (int h = 0; h < 2; ++h) {
        const float ce = tc.c[2 * p + h];
        if (ce < 0.f) continue;
        const double fr = fmod((double)ks * (double)ce, (double)M) / (double)M;
        double sn, cs;
        sincospi(2.0 * fr, &sn, &cs);
        if (h == 0) { re += SC * cs; im += SC * sn; }    // slice A: real part
        else { re -= SC * sn; im += SC * cs; }           // slice B: times i
    }
    ptab[(size_t)p * M + k] = (k == M / 2) ? make_float2(0.f, 0.f) : make_float2((float)re, (float)im);
}

}  // namespace tcpk

using namespace tcpk;

extern "C" {

const char* tcp_last_error(void) { return g_err; }

// n: the power of two the transforms run on; ndet <= n: the caller's detector width (tcp_create_det), embedded at pad_l
static tcp_ctx* create_impl(int n, int ndet, int pad_l, int nproj, int nz_chunk, float center, int dtype, int filter, int m) {
    g_err[0] = 0;
    if (m == 0) m = TCP_KERNEL_KB + 2;    // the default: Kaiser-Bessel, half-width 2 (tcp.h)
    const int kernel = m >> 4;            // kernel code: half-width (Gaussian) or 16 + half-width (Kaiser-Bessel)
    m &= 15;
    if (kernel > 1 || (kernel == 1 && m != 2 && m != 3)) { set_error(TCP_EINVAL, "kernel code %d: Kaiser-Bessel half-width must be 2 or 3", m | (kernel << 4)); return nullptr; }
    if (n < 64 || n > 4096 || (n & (n - 1)) != 0) {
        set_error(TCP_EINVAL, "n=%d must be a power of two in [64, 4096]", n);
        return nullptr;
    }
    if (nproj < 1 || nz_chunk < 1) { set_error(TCP_EINVAL, "nproj=%d and nz_chunk=%d must be >= 1", nproj, nz_chunk); return nullptr; }
    if (!(center >= 0.f && center <= (float)(ndet - 1))) { set_error(TCP_EINVAL, "center=%g outside [0, n-1]", (double)center); return nullptr; }
    center += (float)pad_l;
    if (dtype < TCP_F32 || dtype > TCP_F16_OUT32) { set_error(TCP_EINVAL, "unknown dtype %d", dtype); return nullptr; }
    if (filter < TCP_FILTER_RAMP || filter > TCP_FILTER_HAMMING) { set_error(TCP_EINVAL, "unknown filter %d", filter); return nullptr; }
    if (kernel == 0 && m != 3 && m != 4) { set_error(TCP_EINVAL, "kernel half-width m=%d must be 3 or 4", m); return nullptr; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        set_error(TCP_ECUDA, "no usable CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    tcp_ctx* c = (tcp_ctx*)calloc(1, sizeof(tcp_ctx));
    if (!c) { set_error(TCP_ENOMEM, "out of host memory"); return nullptr; }
    c->grid_dirty = 1;            // the griddings that skip the empty corner tiles zero the grid on their first call
    c->n = n; c->M = 2 * n; c->nproj = nproj; c->nz = nz_chunk; c->npair = (nz_chunk + 1) / 2;
    c->dtype = dtype; c->filter = filter; c->m = m; c->kernel = kernel; c->center = center;
    c->ndet = ndet; c->pad_l = pad_l;
    c->fuse_norm = 1;
    c->half_store = dtype != TCP_F32;
    c->half_out = dtype == TCP_F16;
    // fp16 storage: S = 2^13 puts |f| Phi^2 S <= 65504 for |f| < 1.9 per pixel while keeping
    // noise-level spectrum samples above the half subnormal range
    c->scale = c->half_store ? 8192.0 : 1.0;
    c->grid_impl = c->half_store ? TCP_GRID_MMA : TCP_GRID_TILE;
    c->grid_strip = (c->grid_impl == TCP_GRID_MMA) ? cols_strip_width(c->M) : 0;
    cudaGetDevice(&c->device);
    cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, c->device);
    int rc_pad = TCP_OK;
    if (ndet != n) rc_pad = dev_alloc(&c->out_pad, (size_t)nz_chunk * n * n * (c->half_out ? 2 : 4), &c->bytes);
    if (rc_pad != TCP_OK || build_context(c) != TCP_OK || setup_kernel_attributes(c) != TCP_OK) {
        char keep[512];
        strncpy(keep, g_err, sizeof(keep));
        tcp_destroy(c);
        strncpy(g_err, keep, sizeof(g_err));
        return nullptr;
    }
    return c;
}

tcp_ctx* tcp_create_ex(int n, int nproj, int nz_chunk, float center, int dtype, int filter, int m) {
    return create_impl(n, n, 0, nproj, nz_chunk, center, dtype, filter, m);
}

tcp_ctx* tcp_create_det(int ndet, int nproj, int nz_chunk, float center, int dtype, int filter, int m) {
    if (ndet < 8 || ndet > 4096) {
        g_err[0] = 0;
        set_error(TCP_EINVAL, "ndet=%d must be in [8, 4096]", ndet);
        return nullptr;
    }
    int n = 64;
    while (n < ndet) n *= 2;
    return create_impl(n, ndet, (n - ndet + 1) / 2, nproj, nz_chunk, center, dtype, filter, m);
}

int tcp_padded_n(const tcp_ctx* c) { return c ? c->n : 0; }

tcp_ctx* tcp_create(int n, int nproj, int nz_chunk, float center, int dtype, int filter) {
    return tcp_create_ex(n, nproj, nz_chunk, center, dtype, filter, 0);
}

void tcp_destroy(tcp_ctx* c) {
    if (!c) return;
    pipe_destroy(c);
    if (c->pev) {
        for (int i = 0; i < kProfileRing * (TCP_NSTAGES + 1); ++i) cudaEventDestroy(c->pev[i]);
        free(c->pev);
    }
    cudaFree(c->sino); cudaFree(c->spec); cudaFree(c->grid); cudaFree(c->pass1); cudaFree(c->trig); cudaFree(c->trigf); cudaFree(c->wq); cudaFree(c->fdtab);
    cudaFree(c->tw); cudaFree(c->hfilt); cudaFree(c->ptab); cudaFree(c->ftab); cudaFree(c->deax); cudaFree(c->deay);
    cudaFree(c->tile_order);
    cudaFree(c->kbtab);
    cudaFree(c->pre_buf);
    cudaFree(c->try_buf);
    cudaFree(c->out_pad);
    mmafft_free(c);
    grid_tile_free(c);
    free(c);
}

int tcp_normalize(tcp_ctx* c, const uint16_t* raw, const float* flat, const float* dark, tcp_stream_t stream) {
    if (!c || !raw || !flat || !dark) return set_error(TCP_EINVAL, "NULL argument");
    return launch_normalize(c, raw, flat, dark, (cudaStream_t)stream);
}

// The tile and tensor-core griddings have no work item for the tiles no sample can reach (grid_tile_setup): those cells are
// zeroed here, once per context and again after a tcp_set_option that may change the layout or the writer of the grid.
static int clean_grid(tcp_ctx* c, cudaStream_t st) {
    if (!c->grid_dirty) return TCP_OK;
    TCP_CUDA_CHECK(cudaMemsetAsync(c->grid, 0, (size_t)c->npair * c->M * c->M * (c->half_store ? sizeof(__half2) : sizeof(float2)), st));
    c->grid_dirty = 0;
    return TCP_OK;
}

int tcp_recon(tcp_ctx* c, const uint16_t* raw, const float* flat, const float* dark, const float* theta, void* out,
              tcp_stream_t stream) {
    if (!c || !raw || !flat || !dark || !theta || !out) return set_error(TCP_EINVAL, "NULL argument");
    // the kernels move rows with 16-byte loads, stores and bulk copies (tcp.h: alignment of the device arrays)
    if (c->ndet == c->n && (((uintptr_t)raw | (uintptr_t)flat | (uintptr_t)dark | (uintptr_t)out) & 15))
        return set_error(TCP_EINVAL, "raw_u16, flat, dark and out must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    void* const user_out = out;
    if (c->out_pad) out = c->out_pad;         // tcp_create_det: reconstruct at n, then cut the ndet x ndet image out
    cudaEvent_t* ev = nullptr;
    if (c->profile) {
        if (c->pcalls >= kProfileRing) return set_error(TCP_EINVAL, "profile ring full: call tcp_profile_collect");
        ev = c->pev + (size_t)c->pcalls * (TCP_NSTAGES + 1);
        c->pcalls++;
    }
#define TCP_MARK(i) do { if (ev) TCP_CUDA_CHECK(cudaEventRecord(ev[i], st)); } while (0)
    TCP_MARK(0);
    const bool fused_s12 = rows_fuses_normalize(c);       // S1+S2 in the loader of rows_kernel: no sinogram round trip
    if ((rc = fused_s12 ? launch_trig(c, theta, st, flat, dark) : launch_trig(c, theta, st))) return rc;
    TCP_MARK(1);
    if (!fused_s12 && (rc = launch_normalize(c, raw, flat, dark, st))) return rc;
    if ((c->zinger_dif > 0.0 || c->ring_alpha > 0.0) && (rc = launch_pre(c, st))) return rc;
    TCP_MARK(2);
    if (c->algorithm == TCP_ALG_LINE) {       // LineRec: filter (timed as "rows"), backprojection (timed as "grid")
        if ((rc = launch_filter(c, st))) return rc;
        TCP_MARK(3);
        if ((rc = launch_line_bp(c, out, st))) return rc;
        if (c->out_pad && (rc = launch_crop_out(c, c->nz, user_out, st))) return rc;
        TCP_MARK(4);
        TCP_MARK(5);
        TCP_MARK(6);
        return TCP_OK;
    }
    if (rows_on_mma(c)) rc = launch_rows_mma(c, st, fused_s12 ? raw : nullptr);
    else rc = fused_s12 ? launch_rows(c, st, raw, flat, dark) : launch_rows(c, st);
    if (rc) return rc;
    TCP_MARK(3);
    if (c->grid_impl == TCP_GRID_SCATTER_ATOMIC) rc = launch_grid_scatter(c, st);
    else if (c->grid_impl == TCP_GRID_GATHER) rc = launch_grid_gather(c, theta, st);
    else {
        if ((rc = clean_grid(c, st))) return rc;
        rc = launch_grid_tile(c, theta, st);
    }
    if (rc) return rc;
    TCP_MARK(4);
    if ((rc = ifft2_on_mma(c) ? launch_cols_mma(c, st) : launch_ifft_cols(c, st))) return rc;
    TCP_MARK(5);
    if ((rc = ifft2_on_mma(c) ? launch_irows_mma(c, out, st) : launch_ifft_rows(c, out, st))) return rc;
    if (c->out_pad && (rc = launch_crop_out(c, c->nz, user_out, st))) return rc;
    TCP_MARK(6);
#undef TCP_MARK
    return TCP_OK;
}

int tcp_recon_try(tcp_ctx* c, const uint16_t* raw, const float* flat, const float* dark, const float* theta,
                  const float* centers, int ncenter, void* out, tcp_stream_t stream) {
    if (!c || !raw || !flat || !dark || !theta || !centers || !out) return set_error(TCP_EINVAL, "NULL argument");
    if (c->algorithm != TCP_ALG_FOURIER) return set_error(TCP_EUNSUPPORTED, "tcp_recon_try is FourierRec only");
    if (c->ndet == c->n && (((uintptr_t)raw | (uintptr_t)flat | (uintptr_t)dark | (uintptr_t)out) & 15))
        return set_error(TCP_EINVAL, "raw_u16, flat, dark and out must be 16-byte aligned");
    if (ncenter < 1 || ncenter > c->nz) return set_error(TCP_EINVAL, "ncenter=%d outside [1, nz_chunk=%d]", ncenter, c->nz);
    for (int i = 0; i < ncenter; ++i)
        if (!(centers[i] >= 0.f && centers[i] <= (float)(c->ndet - 1)))
            return set_error(TCP_EINVAL, "centers[%d]=%g outside [0, n-1]", i, (double)centers[i]);
    cudaStream_t st = (cudaStream_t)stream;
    const int M = c->M, npair = (ncenter + 1) / 2;
    if (!c->try_buf) {
        int rc = dev_alloc((void**)&c->try_buf, (size_t)c->npair * M * sizeof(float2), &c->bytes);
        if (rc) return rc;
    }
    // ptab[pair][k] = S C (e^{+2 pi i k c1/M} + i e^{+2 pi i k c2/M}), k signed, 0 at k = M/2 (build_context's table twice),
    // built on the device in fp64; the centres travel by value as kernel arguments (no pageable copy, no hidden sync)
    for (int p0 = 0; p0 < npair; p0 += TryCentres::kMax / 2) {
        TryCentres tc;
        const int np = std::min(npair - p0, TryCentres::kMax / 2);
        for (int i = 0; i < 2 * np; ++i) tc.c[i] = (2 * p0 + i < ncenter) ? centers[2 * p0 + i] + (float)c->pad_l : -1.f;
        try_ptab_kernel<<<dim3((M + 255) / 256, np), 256, 0, st>>>(c->try_buf + (size_t)p0 * M, tc, M, c->scale * kPi / ((double)c->nproj * (double)M));
        TCP_CUDA_CHECK(cudaGetLastError());
    }
    int rc;
    tcp_ctx one = *c;                 // the single input slice
    one.nz = 1; one.npair = 1;
    if ((rc = launch_trig(c, theta, st))) return rc;
    if ((rc = launch_normalize(&one, raw, flat, dark, st))) return rc;
    if ((c->zinger_dif > 0.0 || c->ring_alpha > 0.0) && (rc = launch_pre(&one, st))) return rc;
    tcp_ctx t = *c;                   // ncenter output "slices"
    t.nz = ncenter; t.npair = npair; t.try_ptab = c->try_buf;
    if ((rc = rows_on_mma(&t) ? launch_rows_mma(&t, st, nullptr) : launch_rows(&t, st))) return rc;
    if (c->grid_impl == TCP_GRID_SCATTER_ATOMIC) rc = launch_grid_scatter(&t, st);
    else if (c->grid_impl == TCP_GRID_GATHER) rc = launch_grid_gather(&t, theta, st);
    else {
        if ((rc = clean_grid(c, st))) return rc;        // all npair planes of the context's grid
        rc = launch_grid_tile(&t, theta, st);
    }
    if (rc) return rc;
    if ((rc = ifft2_on_mma(&t) ? launch_cols_mma(&t, st) : launch_ifft_cols(&t, st))) return rc;
    if ((rc = ifft2_on_mma(&t) ? launch_irows_mma(&t, c->out_pad ? c->out_pad : out, st) : launch_ifft_rows(&t, c->out_pad ? c->out_pad : out, st))) return rc;
    return c->out_pad ? launch_crop_out(c, ncenter, out, st) : TCP_OK;
}

int tcp_profile_collect(tcp_ctx* c, double* ms_sum, int* ncalls) {
    if (!c || !ms_sum || !ncalls) return set_error(TCP_EINVAL, "NULL argument");
    for (int s = 0; s < TCP_NSTAGES; ++s) ms_sum[s] = 0.0;
    *ncalls = c->pcalls;
    for (int k = 0; k < c->pcalls; ++k) {
        cudaEvent_t* ev = c->pev + (size_t)k * (TCP_NSTAGES + 1);
        TCP_CUDA_CHECK(cudaEventSynchronize(ev[TCP_NSTAGES]));
        for (int s = 0; s < TCP_NSTAGES; ++s) {
            float ms = 0.f;
            TCP_CUDA_CHECK(cudaEventElapsedTime(&ms, ev[s], ev[s + 1]));
            ms_sum[s] += (double)ms;
        }
    }
    c->pcalls = 0;
    return TCP_OK;
}

int tcp_launches_per_recon(const tcp_ctx* c) {
    if (!c) return 0;
    const int crop = (c->out_pad ? 1 : 0) - (rows_fuses_normalize(c) ? 1 : 0) + (c->zinger_dif > 0.0 ? 1 : 0) + (c->ring_alpha > 0.0 ? 3 : 0);   // tcp_create_det: + the cut-out copy; fused S1+S2: - normalise
    if (c->algorithm == TCP_ALG_LINE) return 4 + crop;                   // trig, normalise, filter, backprojection
    if (c->grid_impl == TCP_GRID_MMA)       // + plan, cache decide (+ cached kernel) (+ reduce); NOT counted: count, scan, fill of a call that may have to rebuild the cache
        return 8 + (c->w_cap > 0 ? 1 : 0) + (c->g_nred ? 1 : 0) + crop;
    if (c->grid_impl == TCP_GRID_TILE) return 7 + (c->g_nred ? 1 : 0) + crop;   // + plan (+ reduce)
    return 6 + crop;                                                     // (scatter adds a memset, not a kernel)
}

int tcp_mean_frames_u16(const uint16_t* frames, int nframes, int nz, int n, float* mean, tcp_stream_t stream) {
    if (!frames || !mean || nframes < 1 || nz < 1 || n < 1) return set_error(TCP_EINVAL, "bad argument");
    return launch_mean_frames(frames, nframes, nz, n, mean, (cudaStream_t)stream);
}

int tcp_workspace(tcp_ctx* c, int which, void** ptr, size_t* bytes) {
    if (!c || !ptr || !bytes) return set_error(TCP_EINVAL, "NULL argument");
    const size_t rb = c->half_store ? 2 : 4, cb = 2 * rb;
    switch (which) {
        case TCP_WS_SINOGRAM: *ptr = c->sino; *bytes = (size_t)c->nz * c->nproj * c->n * rb; return TCP_OK;
        case TCP_WS_SPECTRUM: *ptr = c->spec; *bytes = (size_t)c->npair * c->nproj * c->M * cb; return TCP_OK;
        case TCP_WS_GRID: *ptr = c->grid; *bytes = (size_t)c->npair * c->M * c->M * cb; return TCP_OK;
        case TCP_WS_PASS1: *ptr = c->pass1; *bytes = (size_t)c->npair * c->n * c->M * cb; return TCP_OK;
        case TCP_WS_TRIG: *ptr = c->trig; *bytes = (size_t)c->nproj * sizeof(double2); return TCP_OK;
    }
    return set_error(TCP_EINVAL, "unknown workspace %d", which);
}

int tcp_read_workspace(tcp_ctx* c, int which, void* dst, size_t dst_bytes, tcp_stream_t stream) {
    void* src = nullptr;
    size_t nb = 0;
    int rc = tcp_workspace(c, which, &src, &nb);
    if (rc) return rc;
    if (!dst || dst_bytes < nb) return set_error(TCP_EINVAL, "dst too small: %zu < %zu", dst_bytes, nb);
    TCP_CUDA_CHECK(cudaMemcpyAsync(dst, src, nb, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return TCP_OK;
}

double tcp_scale(const tcp_ctx* c) { return c ? c->scale : 0.0; }
int tcp_pass1_layout(const tcp_ctx* c) { return c && ifft2_on_mma(c) ? 1 : 0; }
int tcp_grid_swizzled(const tcp_ctx* c) { return c && ifft2_on_mma(c) ? 1 : 0; }
int tcp_fft_lines(tcp_ctx* c, const void* in_half2, void* out_float2, int batch, int inverse, tcp_stream_t stream) {
    if (!c || !in_half2 || !out_float2 || batch < 1) return set_error(TCP_EINVAL, "bad argument");
    if (!c->mf_ok) return set_error(TCP_EUNSUPPORTED, "tensor-core transforms need fp16 storage and M = 4096");
    return launch_fft_lines(c, in_half2, out_float2, batch, inverse, (cudaStream_t)stream);
}
int tcp_grid_strip(const tcp_ctx* c) { return c ? c->grid_strip : 0; }
size_t tcp_workspace_bytes(const tcp_ctx* c) { return c ? c->bytes : 0; }

int tcp_set_param(tcp_ctx* c, int param, double value) {
    if (!c) return set_error(TCP_EINVAL, "NULL context");
    if (!(value >= 0.0) || !(value - value == 0.0)) return set_error(TCP_EINVAL, "parameter value %g must be finite and >= 0", value);
    if (value > 0.0 && c->ndet != c->n) return set_error(TCP_EUNSUPPORTED, "pre-processing needs a power-of-two detector width");
    if (param == TCP_PARAM_ZINGER_DIF) { c->zinger_dif = value; return TCP_OK; }
    if (param == TCP_PARAM_RING_ALPHA) {
        if (value > 0.0 && !c->pre_buf) {
            int rc = dev_alloc((void**)&c->pre_buf, (size_t)c->nz * c->n * 6 * sizeof(double), &c->bytes);
            if (rc) return rc;
        }
        c->ring_alpha = value;
        return TCP_OK;
    }
    return set_error(TCP_EINVAL, "unknown parameter %d", param);
}

int tcp_set_option(tcp_ctx* c, int option, int value) {
    if (!c) return set_error(TCP_EINVAL, "NULL context");
    // these two change the grid's layout or its writer: the corner tiles that are never written must be zeroed again
    if (option == TCP_OPT_GRID_IMPL || option == TCP_OPT_TCFFT) c->grid_dirty = 1;
    if (option == TCP_OPT_GRID_IMPL) {
        if (value < TCP_GRID_GATHER || value > TCP_GRID_MMA) return set_error(TCP_EINVAL, "bad grid impl %d", value);
        if ((c->kernel == 1 || c->m == 2) && value != TCP_GRID_TILE && value != TCP_GRID_MMA)
            return set_error(TCP_EUNSUPPORTED, "the Kaiser-Bessel kernel is built into the tile and tensor-core griddings only");
        if (value == TCP_GRID_SCATTER_ATOMIC && c->half_store) return set_error(TCP_EUNSUPPORTED, "scatter gridding supports TCP_F32 only");
        if (value == TCP_GRID_MMA && !c->half_store) return set_error(TCP_EUNSUPPORTED, "tensor-core gridding needs fp16 storage");
        c->grid_impl = value;
        c->grid_strip = (value == TCP_GRID_MMA) ? cols_strip_width(c->M) : 0;
        return TCP_OK;
    }
    if (option == TCP_OPT_WEIGHT_CACHE) {
        c->w_enable = value != 0;
        return TCP_OK;
    }
    if (option == TCP_OPT_FUSE_NORMALIZE) {
        c->fuse_norm = value != 0;
        return TCP_OK;
    }
    if (option == TCP_OPT_ANGLE_WEIGHTS) {
        c->angle_weights = value != 0;
        return TCP_OK;
    }
    if (option == TCP_OPT_FILTER_FUSED) {
        c->filter_fused = value != 0;
        return TCP_OK;
    }
    if (option == TCP_OPT_PAD) {
        if (value != TCP_PAD_ZERO && value != TCP_PAD_EDGE) return set_error(TCP_EINVAL, "unknown padding %d", value);
        // tcp_create_det rows carry air (p = 0) around the detector inside the power-of-two row, so replicating the
        // ROW's edge samples would pad with zeros and silently bring the truncation artefacts back: refuse instead
        if (value == TCP_PAD_EDGE && c->ndet != c->n)
            return set_error(TCP_EUNSUPPORTED, "TCP_PAD_EDGE needs a power-of-two detector width (tcp_create_det pads the row with air)");
        c->pad = value;
        return TCP_OK;
    }
    if (option == TCP_OPT_ALGORITHM) {
        if (value != TCP_ALG_FOURIER && value != TCP_ALG_LINE) return set_error(TCP_EINVAL, "unknown algorithm %d", value);
        c->algorithm = value;
        return TCP_OK;
    }
    if (option == TCP_OPT_TCFFT) {
        if (value & ~c->tcfft_ok) return set_error(TCP_EUNSUPPORTED, "tensor-core transforms %d not available here (mask %d)", value, c->tcfft_ok);
        if (((value & TCP_TCFFT_COLS) != 0) != ((value & TCP_TCFFT_IROWS) != 0))
            return set_error(TCP_EINVAL, "the two passes of the inverse 2D transform switch together (mask 6)");
        c->tcfft = value;
        return TCP_OK;
    }
    if (option == TCP_OPT_PROFILE) {
        if (value && !c->pev) {
            c->pev = (cudaEvent_t*)calloc((size_t)kProfileRing * (TCP_NSTAGES + 1), sizeof(cudaEvent_t));
            if (!c->pev) return set_error(TCP_ENOMEM, "out of host memory");
            for (int i = 0; i < kProfileRing * (TCP_NSTAGES + 1); ++i) TCP_CUDA_CHECK(cudaEventCreate(&c->pev[i]));
        }
        c->profile = value != 0;
        c->pcalls = 0;
        return TCP_OK;
    }
    return set_error(TCP_EINVAL, "unknown option %d", option);
}

}  // extern "C"
