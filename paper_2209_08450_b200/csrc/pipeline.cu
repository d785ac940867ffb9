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

int setup_kernel_attributes(const tcp_ctx*) { return TCP_OK; }

void pipe_destroy(tcp_ctx* c) {
    Pipe* p = c->pipe;
    if (!p) return;
    for (int b = 0; b < p->nbuf; ++b) {
        cudaFree(p->raw[b]); cudaFree(p->flat[b]); cudaFree(p->dark[b]); cudaFree(p->out[b]);
        cudaEventDestroy(p->ev_h2d[b]); cudaEventDestroy(p->ev_comp[b]); cudaEventDestroy(p->ev_d2h[b]);
    }
    cudaFree(p->theta);
    cudaEventDestroy(p->ev_start); cudaEventDestroy(p->ev_stop);
    cudaStreamDestroy(p->s_h2d); cudaStreamDestroy(p->s_comp); cudaStreamDestroy(p->s_d2h);
    free(p);
    c->pipe = nullptr;
}

static int pipe_create(tcp_ctx* c, int nbuf) {
    if (c->pipe && c->pipe->nbuf == nbuf) return TCP_OK;
    pipe_destroy(c);
    Pipe* p = (Pipe*)calloc(1, sizeof(Pipe));
    if (!p) return set_error(TCP_ENOMEM, "out of host memory");
    c->pipe = p;
    p->nbuf = nbuf;
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
        // a partial last chunk leaves rows unwritten: keep them finite
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

extern "C" int tcp_recon_volume_host(tcp_ctx* c, const uint16_t* raw_host, const float* flat_host,
                                     const float* dark_host, const float* theta_host, void* out_host, int nz_total,
                                     int nbuf, float* ms_out) {
    if (!c || !raw_host || !flat_host || !dark_host || !theta_host || !out_host)
        return set_error(TCP_EINVAL, "NULL argument");
    if (nz_total < 1) return set_error(TCP_EINVAL, "nz_total=%d must be >= 1", nz_total);
    if (nbuf != 2 && nbuf != 3) return set_error(TCP_EINVAL, "nbuf=%d must be 2 or 3", nbuf);
    int rc;
    if ((rc = pipe_create(c, nbuf))) return rc;
    Pipe* p = c->pipe;
    const int n = c->ndet, nz = c->nz;
    const size_t ob = c->half_out ? 2 : 4;
    const int nchunks = (nz_total + nz - 1) / nz;

    TCP_CUDA_CHECK(cudaEventRecord(p->ev_start, p->s_h2d));
    TCP_CUDA_CHECK(cudaMemcpyAsync(p->theta, theta_host, (size_t)c->nproj * 4, cudaMemcpyHostToDevice, p->s_h2d));
    for (int ch = 0; ch < nchunks; ++ch) {
        const int b = ch % nbuf;
        const int z0 = ch * nz;
        const int nzc = (nz_total - z0 < nz) ? nz_total - z0 : nz;
        // H2D: raw[b] is free once the compute of chunk ch - nbuf has finished
        if (ch >= nbuf) TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_h2d, p->ev_comp[b], 0));
        // strided gather of rows z0..z0+nzc of every projection: one 2D copy
        TCP_CUDA_CHECK(cudaMemcpy2DAsync(p->raw[b], (size_t)nz * n * 2, raw_host + (size_t)z0 * n,
                                         (size_t)nz_total * n * 2, (size_t)nzc * n * 2, c->nproj,
                                         cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaMemcpyAsync(p->flat[b], flat_host + (size_t)z0 * n, (size_t)nzc * n * 4,
                                       cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaMemcpyAsync(p->dark[b], dark_host + (size_t)z0 * n, (size_t)nzc * n * 4,
                                       cudaMemcpyHostToDevice, p->s_h2d));
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_h2d[b], p->s_h2d));
        // compute: needs the inputs, and out[b] drained by the D2H of chunk ch - nbuf
        TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_comp, p->ev_h2d[b], 0));
        if (ch >= nbuf) TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_comp, p->ev_d2h[b], 0));
        if ((rc = tcp_recon(c, p->raw[b], p->flat[b], p->dark[b], p->theta, p->out[b], p->s_comp))) return rc;
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_comp[b], p->s_comp));
        // D2H
        TCP_CUDA_CHECK(cudaStreamWaitEvent(p->s_d2h, p->ev_comp[b], 0));
        TCP_CUDA_CHECK(cudaMemcpyAsync((char*)out_host + (size_t)z0 * n * n * ob, p->out[b], (size_t)nzc * n * n * ob,
                                       cudaMemcpyDeviceToHost, p->s_d2h));
        TCP_CUDA_CHECK(cudaEventRecord(p->ev_d2h[b], p->s_d2h));
    }
    TCP_CUDA_CHECK(cudaEventRecord(p->ev_stop, p->s_d2h));
    TCP_CUDA_CHECK(cudaStreamSynchronize(p->s_d2h));
    TCP_CUDA_CHECK(cudaStreamSynchronize(p->s_comp));
    TCP_CUDA_CHECK(cudaStreamSynchronize(p->s_h2d));
    if (ms_out) TCP_CUDA_CHECK(cudaEventElapsedTime(ms_out, p->ev_start, p->ev_stop));
    return TCP_OK;
}
