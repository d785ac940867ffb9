// k_pre.cu -- optional pre-processing of the sinogram between S2 and S3 ("zinger artifacts reduction
// (Rivers, 1998)", ring removal "with an analytical formula by V. Titarenko"; readings Q22, Q23):
//   zingers: p'[j][i] = med if med - p[j][i] > dif, med = median of the 3 x 3 (projection, pixel) neighbourhood of the
//            ORIGINAL sinogram with clamped indices (an isolated bright detector hit is an isolated low sample of p);
//   rings:   p'[j][i] = p[j][i] - r[i], (A + alpha I) r = A pbar, A = D2^T D2 (second differences), pbar = mean over the
//            projections: the closed-form Tikhonov estimate of a per-pixel offset that is the same in every projection.
// Both work on the context's sinogram workspace [nz][nproj][n] (float or half); tcp_recon then skips the fused S1+S2
// loader.  The ring system is solved in fp64 (one thread per slice, O(n), banded LDL^T): its result is a small correction,
// and fp64 keeps it exact at the level of the fp32 gate whatever alpha is.
#include <math.h>

#include <algorithm>
#include <map>
#include <mutex>

#include "tcp_internal.h"

namespace tcpk {

__device__ __forceinline__ void cswap(float& a, float& b) {
    const float lo = fminf(a, b), hi = fmaxf(a, b);
    a = lo;
    b = hi;
}
// median of 9 by the 19-exchange selection network
__device__ __forceinline__ float median9(float (&v)[9]) {
    cswap(v[1], v[2]); cswap(v[4], v[5]); cswap(v[7], v[8]);
    cswap(v[0], v[1]); cswap(v[3], v[4]); cswap(v[6], v[7]);
    cswap(v[1], v[2]); cswap(v[4], v[5]); cswap(v[7], v[8]);
    cswap(v[0], v[3]); cswap(v[5], v[8]); cswap(v[4], v[7]);
    cswap(v[3], v[6]); cswap(v[1], v[4]); cswap(v[2], v[5]);
    cswap(v[4], v[7]); cswap(v[4], v[2]); cswap(v[6], v[4]);
    cswap(v[4], v[2]);
    return v[4];
}

template <class TS>
__global__ void __launch_bounds__(256) zinger_kernel(const TS* __restrict__ sino, TS* __restrict__ out, int nz, int nproj, int n,
                                                     float dif) {
    const size_t total = (size_t)nz * nproj * n;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(v % n);
        const size_t row = v / n;
        const int j = (int)(row % nproj);
        const TS* s = sino + (row - j) * n;             // slice base
        float w[9];
        int t = 0;
#pragma unroll
        for (int dj = -1; dj <= 1; ++dj)
#pragma unroll
            for (int di = -1; di <= 1; ++di) {
                const int jj = min(max(j + dj, 0), nproj - 1), ii = min(max(i + di, 0), n - 1);
                w[t++] = ld_r(s, (size_t)jj * n + ii);
            }
        const float x = w[4];
        const float med = median9(w);
        st_r(out, v, (med - x > dif) ? med : x);
    }
}

// pbar[z][i] = mean over j of sino[z][j][i], in fp64
template <class TS>
__global__ void __launch_bounds__(256) ring_mean_kernel(const TS* __restrict__ sino, double* __restrict__ pbar, int nz, int nproj, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, z = blockIdx.y;
    if (i >= n) return;
    const TS* s = sino + (size_t)z * nproj * n + i;
    double acc = 0.0;
    for (int j = 0; j < nproj; ++j) acc += (double)ld_r(s, (size_t)j * n);
    pbar[(size_t)z * n + i] = acc / (double)nproj;
}

// one thread per slice: (A + alpha I) r = A pbar by banded LDL^T; work[z][5][n] doubles: d, l1, l2, y, r
__global__ void ring_solve_kernel(const double* __restrict__ pbar, double* __restrict__ work, int nz, int n, double alpha) {
    const int z = blockIdx.x * blockDim.x + threadIdx.x;
    if (z >= nz) return;
    const double* pb = pbar + (size_t)z * n;
    double* d = work + (size_t)z * 5 * n;
    double *l1 = d + n, *l2 = d + 2 * n, *y = d + 3 * n, *r = d + 4 * n;
    auto D2 = [&](int i) { return (i >= 0 && i + 2 < n) ? pb[i] - 2.0 * pb[i + 1] + pb[i + 2] : 0.0; };
    for (int i = 0; i < n; ++i) {
        // row i of A = D2^T D2: second-difference rows i-2, i-1, i touch column i with coefficients 1, -2, 1
        const double a0 = ((i + 2 < n) ? 1.0 : 0.0) + ((i >= 1 && i + 1 < n) ? 4.0 : 0.0) + ((i >= 2) ? 1.0 : 0.0) + alpha;
        const double a1 = ((i + 2 < n) ? -2.0 : 0.0) + ((i >= 1 && i + 1 < n) ? -2.0 : 0.0);       // A[i][i+1]
        const double a2 = (i + 2 < n) ? 1.0 : 0.0;                                                    // A[i][i+2]
        double di = a0;
        if (i >= 1) di -= l1[i - 1] * l1[i - 1] * d[i - 1];
        if (i >= 2) di -= l2[i - 2] * l2[i - 2] * d[i - 2];
        d[i] = di;
        if (i + 1 < n) {
            double v = a1;
            if (i >= 1) v -= l1[i - 1] * l2[i - 1] * d[i - 1];
            l1[i] = v / di;
        }
        if (i + 2 < n) l2[i] = a2 / di;
        double rhs = D2(i) - 2.0 * D2(i - 1) + D2(i - 2);             // (D2^T D2 pbar)[i]
        if (i >= 1) rhs -= l1[i - 1] * y[i - 1];
        if (i >= 2) rhs -= l2[i - 2] * y[i - 2];
        y[i] = rhs;
    }
    for (int i = n - 1; i >= 0; --i) {
        double v = y[i] / d[i];
        if (i + 1 < n) v -= l1[i] * r[i + 1];
        if (i + 2 < n) v -= l2[i] * r[i + 2];
        r[i] = v;
    }
}

template <class TS>
__global__ void __launch_bounds__(256) ring_sub_kernel(TS* __restrict__ sino, const double* __restrict__ work, int nz, int nproj, int n) {
    const size_t total = (size_t)nz * nproj * n;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(v % n);
        const int z = (int)(v / ((size_t)nproj * n));
        const double r = work[((size_t)z * 5 + 4) * n + i];
        st_r(sino, v, (float)((double)ld_r(sino, v) - r));
    }
}

template <class TS>
static int launch_pre_t(const tcp_ctx* c, cudaStream_t st) {
    const size_t total = (size_t)c->nz * c->nproj * c->n;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)c->nsm * 16);
    if (c->zinger_dif > 0.0) {
        // out of place (every median is taken on the original samples): the spectrum workspace is free at this point
        zinger_kernel<TS><<<blocks, 256, 0, st>>>((const TS*)c->sino, (TS*)c->spec, c->nz, c->nproj, c->n, (float)c->zinger_dif);
        TCP_CUDA_CHECK(cudaGetLastError());
        TCP_CUDA_CHECK(cudaMemcpyAsync(c->sino, c->spec, total * sizeof(TS), cudaMemcpyDeviceToDevice, st));
    }
    if (c->ring_alpha > 0.0) {
        double* pbar = c->pre_buf;
        double* work = c->pre_buf + (size_t)c->nz * c->n;
        ring_mean_kernel<TS><<<dim3((c->n + 255) / 256, c->nz), 256, 0, st>>>((const TS*)c->sino, pbar, c->nz, c->nproj, c->n);
        ring_solve_kernel<<<(c->nz + 31) / 32, 32, 0, st>>>(pbar, work, c->nz, c->n, c->ring_alpha);
        ring_sub_kernel<TS><<<blocks, 256, 0, st>>>((TS*)c->sino, work, c->nz, c->nproj, c->n);
        TCP_CUDA_CHECK(cudaGetLastError());
    }
    return TCP_OK;
}

int launch_pre(const tcp_ctx* c, cudaStream_t st) {
    return c->half_store ? launch_pre_t<__half>(c, st) : launch_pre_t<float>(c, st);
}

}  // namespace tcpk

// ------------------------------------------------------------------------------------------------ allocation-free ring removal
// tcp_ring_remove_static (tcp.h): the ring-removal step above for callers that may not allocate (CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc).  The same three kernels run on the caller's arrays; the scratch that
// tcp_set_param(TCP_PARAM_RING_ALPHA) would cudaMalloc per context (angle means [nz][n] + solver work [nz][5][n], fp64)
// lives in ONE file-scope device array of fixed size instead: 6 * TCP_RING_STATIC_MAX doubles = 3 MiB, held by every GPU
// that loads the library until the process exits, shared by every call (calls that overlap on the GPU race on it).
// Nothing in it has to start at zero: ring_mean_kernel writes every mean, and ring_solve_kernel writes d, l1, l2, y, r at
// index i before it reads them at i - 1, i - 2 (factorisation) or i + 1, i + 2 (back substitution); the last call's
// contents are never read.
namespace tcpk {

static __device__ __align__(256) double g_ring_static[6 * (size_t)TCP_RING_STATIC_MAX];

// out-of-place form of ring_sub_kernel (in == out allowed: one read and one write of the same element per thread)
template <class TS>
__global__ void __launch_bounds__(256) ring_sub_io_kernel(const TS* in, TS* out, const double* __restrict__ work, int nz, int nproj, int n) {
    const size_t total = (size_t)nz * nproj * n;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(v % n);
        const int z = (int)(v / ((size_t)nproj * n));
        const double r = work[((size_t)z * 5 + 4) * n + i];
        st_r(out, v, (float)((double)ld_r(in, v) - r));
    }
}

// In host code `g_ring_static` is the host-side stand-in of the symbol, not a device address: the device address is asked
// for once per device, with that device current, and cached.
struct RingStaticDev {
    double* scratch;
    int nsm;
};
static std::mutex g_ring_static_mu;
static std::map<int, RingStaticDev> g_ring_static_dev;

static int ring_static_setup(RingStaticDev* out) {
    int dev = -1;
    TCP_CUDA_CHECK(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_ring_static_mu);
    auto it = g_ring_static_dev.find(dev);
    if (it == g_ring_static_dev.end()) {
        RingStaticDev d{nullptr, 0};
        TCP_CUDA_CHECK(cudaGetSymbolAddress((void**)&d.scratch, g_ring_static));
        if (!d.scratch) return set_error(TCP_ECUDA, "tcp_ring_remove_static: cudaGetSymbolAddress returned a null address on device %d", dev);
        TCP_CUDA_CHECK(cudaDeviceGetAttribute(&d.nsm, cudaDevAttrMultiProcessorCount, dev));
        it = g_ring_static_dev.emplace(dev, d).first;
    }
    *out = it->second;
    return TCP_OK;
}

template <class TS>
static int ring_static_launch(const RingStaticDev& d, const void* in, void* out, int nz, int nproj, int n, double alpha, cudaStream_t st) {
    const size_t total = (size_t)nz * nproj * n;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)d.nsm * 16);
    double* pbar = d.scratch;
    double* work = d.scratch + (size_t)nz * n;
    ring_mean_kernel<TS><<<dim3((n + 255) / 256, nz), 256, 0, st>>>((const TS*)in, pbar, nz, nproj, n);
    ring_solve_kernel<<<(nz + 31) / 32, 32, 0, st>>>(pbar, work, nz, n, alpha);
    ring_sub_io_kernel<TS><<<blocks, 256, 0, st>>>((const TS*)in, (TS*)out, work, nz, nproj, n);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

}  // namespace tcpk

extern "C" int tcp_ring_static_setup(void) {
    tcpk::RingStaticDev d;
    return tcpk::ring_static_setup(&d);
}

extern "C" int tcp_ring_remove_static(const void* sino_in, void* sino_out, int nz, int nproj, int n, int dtype, double alpha,
                                      tcp_stream_t stream) {
    using namespace tcpk;
    if (!sino_in || !sino_out) return set_error(TCP_EINVAL, "tcp_ring_remove_static: NULL sinogram pointer");
    if (dtype != TCP_F32 && dtype != TCP_F16) return set_error(TCP_EINVAL, "tcp_ring_remove_static: dtype %d is neither TCP_F32 nor TCP_F16", dtype);
    if (nz < 1 || nproj < 1 || n < 3) return set_error(TCP_EINVAL, "tcp_ring_remove_static: need nz >= 1, nproj >= 1, n >= 3 (got %d, %d, %d)", nz, nproj, n);
    if (!(alpha > 0.0) || !isfinite(alpha)) return set_error(TCP_EINVAL, "tcp_ring_remove_static: alpha must be positive and finite");
    if ((long long)nz * n > (long long)TCP_RING_STATIC_MAX)
        return set_error(TCP_EINVAL, "tcp_ring_remove_static: nz * n = %lld exceeds TCP_RING_STATIC_MAX = %d (the fixed scratch array); "
                         "split the slices over several calls or use tcp_set_param(TCP_PARAM_RING_ALPHA)", (long long)nz * n, (int)TCP_RING_STATIC_MAX);
    if (nz > 65535) return set_error(TCP_EINVAL, "tcp_ring_remove_static: nz = %d exceeds 65535", nz);
    RingStaticDev d;
    int rc = ring_static_setup(&d);
    if (rc != TCP_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    return dtype == TCP_F16 ? ring_static_launch<__half>(d, sino_in, sino_out, nz, nproj, n, alpha, st)
                            : ring_static_launch<float>(d, sino_in, sino_out, nz, nproj, n, alpha, st);
}
