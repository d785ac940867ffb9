// pipeline.cu -- the chunk pipeline of PAPER.md:71-83 (Fig. 1): while chunk N is copied host ->
// device, chunk N-1 is reconstructed and chunk N-2 is copied device -> host, on three CUDA
// streams.  The paper allocates 2 pinned + 2 device buffers per direction and synchronises all
// streams after every chunk; here the host never blocks inside the loop: buffer reuse is ordered
// by events, so the three engines (H2D copy, SMs, D2H copy) run back to back, with nbuf = 2 or 3
// device buffer sets (B200 has the memory for deeper buffering).
#include <stdlib.h>

#include "tcp_internal.h"

struct Pipe {
    int nbuf;
    cudaStream_t s_h2d, s_comp, s_d2h;
    uint16_t* raw[3];
    float* flat[3];
    float* dark[3];
    void* out[3];
    float* theta;
    cudaEvent_t ev_h2d[3], ev_comp[3], ev_d2h[3], ev_start, ev_stop;
};

namespace tcpk {

// Called once from tcp_create: the device must offer the opt-in shared memory the context's transforms need (one padded
// line of M complex values per row transform, cols_wp(M) lines + staging for the column pass: up to 227 KB); the
// per-kernel opt-in itself is memoised at first launch (ensure_smem), not repeated per launch.
int setup_kernel_attributes(const tcp_ctx* c) {
    int optin = 0;
    TCP_CUDA_CHECK(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
    const int line = (c->M + c->M / 16) * 8;
    if (optin < 2 * line || optin < 200 * 1024)
        return set_error(TCP_EUNSUPPORTED, "device offers %d B of opt-in shared memory per block; sm_100a (227 KB) is required", optin);
    return TCP_OK;
}

void pipe_destroy(tcp_ctx* c) {
    Pipe* p = c->pipe;
    if (!p) return;
    for (int b = 0; b < p->nbuf; ++b) {
        cudaFree(p->raw[b]); cudaFree(p->flat[b]); cudaFree(p->dark[b]); cudaFree(p->out[b]);
        if (p->ev_h2d[b]) cudaEventDestroy(p->ev_h2d[b]);
        if (p->ev_comp[b]) cudaEventDestroy(p->ev_comp[b]);
        if (p->ev_d2h[b]) cudaEventDestroy(p->ev_d2h[b]);
    }
    cudaFree(p->theta);
    if (p->ev_start) cudaEventDestroy(p->ev_start);
    if (p->ev_stop) cudaEventDestroy(p->ev_stop);
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_comp) cudaStreamDestroy(p->s_comp);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    free(p);
    c->pipe = nullptr;
}

static int pipe_fill(tcp_ctx* c, Pipe* p, int nbuf);

// The pipe is published in the context only when every stream, buffer and event exists: a failed allocation leaves
// c->pipe NULL (and frees what was made), so the next call starts over instead of running on NULL handles.
static int pipe_create(tcp_ctx* c, int nbuf) {
    if (c->pipe && c->pipe->nbuf == nbuf) return TCP_OK;
    pipe_destroy(c);
    Pipe* p = (Pipe*)calloc(1, sizeof(Pipe));
    if (!p) return set_error(TCP_ENOMEM, "out of host memory");
    p->nbuf = nbuf;
    const int rc = pipe_fill(c, p, nbuf);
    c->pipe = p;
    if (rc != TCP_OK) pipe_destroy(c);        // cudaFree / destroy of a zero handle is a no-op or a harmless error
    cudaGetLastError();
    return rc;
}

static int pipe_fill(tcp_ctx* c, Pipe* p, int nbuf) {
    const size_t ob = c->half_out ? 2 : 4;
    const int n = c->ndet;                    // width of the caller's rows and side of the caller's images
    TCP_CUDA_CHECK(cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
    TCP_CUDA_CHECK(cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking));
    TCP_CUDA_CHECK(cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
    TCP_CUDA_CHECK(cudaEventCreate(&p->ev_start));
    TCP_CUDA_CHECK(cudaEventCreate(&p->ev_stop));
    TCP_CUDA_CHECK(cudaMalloc((void**)&p->theta, (size_t)c->nproj * sizeof(float)));
    for (int b = 0; b < nbuf; ++b) {
        TCP_CUDA_CHECK(cudaMalloc((void**)&p->raw[b], (size_t)c->nproj * c->nz * n * 2));
        TCP_CUDA_CHECK(cudaMalloc((void**)&p->flat[b], (size_t)c->nz * n * 4));
        TCP_CUDA_CHECK(cudaMalloc((void**)&p->dark[b], (size_t)c->nz * n * 4));
        TCP_CUDA_CHECK(cudaMalloc(&p->out[b], (size_t)c->nz * n * n * ob));
        // (buffers start zeroed: nothing reads rows a call did not write, this only keeps debugging dumps clean)
        TCP_CUDA_CHECK(cudaMemset(p->raw[b], 0, (size_t)c->nproj * c->nz * n * 2));
        TCP_CUDA_CHECK(cudaMemset(p->flat[b], 0, (size_t)c->nz * n * 4));
        TCP_CUDA_CHECK(cudaMemset(p->dark[b], 0, (size_t)c->nz * n * 4));
        TCP_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_h2d[b], cudaEventDisableTiming));
        TCP_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_comp[b], cudaEventDisableTiming));
        TCP_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_d2h[b], cudaEventDisableTiming));
    }
    TCP_CUDA_CHECK(cudaDeviceSynchronize());
    return TCP_OK;
}

}  // namespace tcpk

using namespace tcpk;

// Contiguous slice range of rank `rank` of `world` (one process per GPU on a subset of the
// slices, no exchange between them): ranges differ by at most one slice and tile [0, nz_total) in rank order.
extern "C" int tcp_slice_range(int nz_total, int rank, int world, int* z0, int* z1) {
    if (nz_total < 0 || world < 1 || rank < 0 || rank >= world || !z0 || !z1) return set_error(TCP_EINVAL, "bad slice-range argument");
    const long long q = nz_total / world, r = nz_total % world;
    *z0 = (int)(q * rank + (rank < r ? rank : r));
    *z1 = *z0 + (int)q + (rank < r ? 1 : 0);
    return TCP_OK;
}

// HOST logic: the angles tcp_recon accepts (the projection window of a grid region is an index range of theta)
extern "C" int tcp_check_angles(const float* theta_host, int nproj) {
    if (!theta_host || nproj < 1) return set_error(TCP_EINVAL, "bad angle array");
    for (int j = 0; j < nproj; ++j) {
        if (!(theta_host[j] == theta_host[j]) || !(theta_host[j] - theta_host[j] == 0.f)) return set_error(TCP_EINVAL, "theta[%d] is not finite", j);
        if (j > 0 && !(theta_host[j] > theta_host[j - 1]))
            return set_error(TCP_EINVAL, "theta must be strictly increasing: theta[%d]=%g <= theta[%d]=%g", j, (double)theta_host[j], j - 1, (double)theta_host[j - 1]);
    }
    if (!((double)theta_host[nproj - 1] - (double)theta_host[0] < 3.14159265358979323846))
        return set_error(TCP_EINVAL, "theta spans %g >= pi: fold a full turn onto [0, pi) first", (double)theta_host[nproj - 1] - (double)theta_host[0]);
    return TCP_OK;
}

extern "C" int tcp_recon_volume_host(tcp_ctx* c, const uint16_t* raw_host, const float* flat_host,
                                     const float* dark_host, const float* theta_host, void* out_host, int nz_total,
                                     int nbuf, float* ms_out) {
    return tcp_recon_volume_host_rows(c, raw_host, flat_host, dark_host, theta_host, out_host, nz_total, 0, nz_total, nbuf, ms_out);
}

extern "C" int tcp_recon_volume_host_rows(tcp_ctx* c, const uint16_t* raw_host, const float* flat_host,
                                          const float* dark_host, const float* theta_host, void* out_host, int nz_stack,
                                          int z_begin, int z_end, int nbuf, float* ms_out) {
    if (!c || !raw_host || !flat_host || !dark_host || !theta_host || !out_host)
        return set_error(TCP_EINVAL, "NULL argument");
    int rc0;
    if (nz_stack < 1) return set_error(TCP_EINVAL, "nz_total=%d must be >= 1", nz_stack);
    if ((rc0 = tcp_check_angles(theta_host, c->nproj))) return rc0;
    if (z_begin < 0 || z_end > nz_stack || z_begin >= z_end)
        return set_error(TCP_EINVAL, "rows [%d, %d) must be a non-empty range inside [0, %d)", z_begin, z_end, nz_stack);
    if (nbuf != 2 && nbuf != 3) return set_error(TCP_EINVAL, "nbuf=%d must be 2 or 3", nbuf);
    int rc;
    if ((rc = pipe_create(c, nbuf))) return rc;
    Pipe* p = c->pipe;
    const int n = c->ndet, nz = c->nz;
    const size_t ob = c->half_out ? 2 : 4;
    const int nz_total = z_end - z_begin;                  // slices of this call; the arrays hold nz_stack
    const int nchunks = (nz_total + nz - 1) / nz;

    // An error inside the loop must not return while copies on the caller's pinned buffers are in flight (the caller
    // may free or reuse them): the loop runs in a lambda and every exit path drains the three streams first.
    auto enqueue = [&]() -> int {
    TCP_CUDA_CHECK(cudaEventRecord(p->ev_start, p->s_h2d));
    TCP_CUDA_CHECK(cudaMemcpyAsync(p->theta, theta_host, (size_t)c->nproj * 4, cudaMemcpyHostToDevice, p->s_h2d));
    for (int ch = 0; ch < nchunks; ++ch) {
        const int b = ch % nbuf;
        const int z0 = z_begin + ch * nz;
        const int nzc = (z_end - z0 < nz) ? z_end - z0 : nz;
        // H2D: raw[b] is free once the compute of chunk ch - nbuf has finished
        if (ch >= nbuf) TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_h2d, p->ev_comp[b], 0));
        // strided gather of rows z0..z0+nzc of every projection: one 2D copy.  A partial last chunk is laid out and
        // reconstructed as a chunk of nzc slices (device array [nproj][nzc][n]): its result does not depend on what
        // an earlier chunk left in the buffers, and an odd last slice is paired with zeros
        TCP_CUDA_CHECK(cudaMemcpy2DAsync(p->raw[b], (size_t)nzc * n * 2, raw_host + (size_t)z0 * n,
                                         (size_t)nz_stack * n * 2, (size_t)nzc * n * 2, c->nproj,
                                         cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaMemcpyAsync(p->flat[b], flat_host + (size_t)z0 * n, (size_t)nzc * n * 4,
                                       cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaMemcpyAsync(p->dark[b], dark_host + (size_t)z0 * n, (size_t)nzc * n * 4,
                                       cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_h2d[b], p->s_h2d));
        // compute: needs the inputs, and out[b] drained by the D2H of chunk ch - nbuf
        TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_comp, p->ev_h2d[b], 0));
        if (ch >= nbuf) TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_comp, p->ev_d2h[b], 0));
        if (nzc == nz) {
            rc = tcp_recon(c, p->raw[b], p->flat[b], p->dark[b], p->theta, p->out[b], p->s_comp);
        } else {
            tcp_ctx part = *c;                 // same workspaces and tables, fewer slices (as tcp_recon_try does)
            part.nz = nzc;
            part.npair = (nzc + 1) / 2;
            part.profile = false;
            rc = tcp_recon(&part, p->raw[b], p->flat[b], p->dark[b], p->theta, p->out[b], p->s_comp);
        }
        if (rc) return rc;
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_comp[b], p->s_comp));
        // D2H
        TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_d2h, p->ev_comp[b], 0));
        TCP_CUDA_CHECK(cudaMemcpyAsync((char*)out_host + (size_t)z0 * n * n * ob, p->out[b], (size_t)nzc * n * n * ob,
                                       cudaMemcpyDeviceToHost, p->s_d2h));
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_d2h[b], p->s_d2h));
    }
    TCP_CUDA_CHECK(cudaEventRecord(p->ev_stop, p->s_d2h));
    return TCP_OK;
    };
    rc = enqueue();
    const cudaError_t e1 = cudaStreamSynchronize(p->s_d2h), e2 = cudaStreamSynchronize(p->s_comp), e3 = cudaStreamSynchronize(p->s_h2d);
    if (rc) return rc;
    TCP_CUDA_CHECK(e1);
    TCP_CUDA_CHECK(e2);
    TCP_CUDA_CHECK(e3);
    if (ms_out) TCP_CUDA_CHECK(cudaEventElapsedTime(ms_out, p->ev_start, p->ev_stop));
    return TCP_OK;
}
