/* tcp.h -- C ABI of the B200-native parallel-beam FBP hot path (Fourier gridding).
 *
 * What is computed (per chunk of nz detector rows = slices), after arXiv 2209.08450
 * (TomocuPy) sec. 2.2: "dark-flat field correction, taking negative logarithm of the
 * data, one-dimensional filtering with the Shepp-Logan, Parzen or other filter"
 * (PAPER.md:57), then the backprojection by the "Fourier-based method with
 * exponential functions for interpolation in the frequency domain",
 * oversampling 2.  Stage by stage:
 *   S1+S2  t = (raw-dark)/max(flat-dark,1e-3), p = -ln max(t,1e-6)
 *   S3     q = crop_n( IFFT_M( FFT_M([p,0]) * H ) ),  M = 2n, H = ramp kernel * window
 *   S4     G[j][k] = C * FFT_M([q,0])[k] * exp(+2 pi i k c / M),  C = pi/(nproj*M)
 *   S5     F[l2][l1] += G[j][k] phi(l1 - k cos_j) phi(l2 - k sin_j), |l - nu| < m,
 *          phi(t) = exp(-alpha t^2), alpha = pi/(sqrt(2) m), periodic in M
 *   S6     g = unnormalised inverse 2D FFT of F
 *   S7     out[z][iy][ix] = Re g[y][x] / (Phi(x) Phi(y)),  x = ix - n/2, y = iy - n/2
 * Two adjacent slices ride one complex transform (slice z -> real part, z+1 -> imaginary).
 *
 * Every step runs in hand-written sm_100a CUDA kernels inside this library.  There is
 * no CPU fallback: if no CUDA device is usable the calls fail with TCP_ECUDA.
 *
 * Pointers: unless a parameter says HOST, every pointer is a DEVICE pointer owned by
 * the caller; the library never frees or retains it beyond the call's stream work.
 * Errors: functions returning int give TCP_OK (0) or a negative code; tcp_create*
 * return NULL on error.  tcp_last_error() gives a thread-local message.
 */
#ifndef TCP_H_
#define TCP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tcp_ctx tcp_ctx;                 /* opaque */
typedef void* tcp_stream_t;                     /* a cudaStream_t (NULL = legacy default stream) */

/* compute/storage dtype of the intermediates and dtype of `out` (FP16 storage
 * with FP32 arithmetic where FP16 would lose accuracy).  F16_OUT32 exists for config C5. */
enum { TCP_F32 = 0, TCP_F16 = 1, TCP_F16_OUT32 = 2 };
/* "--fbp-filter": windows multiplying the band-limited ramp; "Shepp-Logan, Parzen or other
 * filter": the others are the textbook apodisation windows on u = |k|/(M/2): cosine cos(pi u/2),
 * Hann (1 + cos(pi u))/2, Hamming 0.54 + 0.46 cos(pi u). */
enum { TCP_FILTER_RAMP = 0, TCP_FILTER_SHEPP = 1, TCP_FILTER_PARZEN = 2, TCP_FILTER_COSINE = 3, TCP_FILTER_HANN = 4,
       TCP_FILTER_HAMMING = 5 };
enum { TCP_OK = 0, TCP_EINVAL = -1, TCP_ENOMEM = -2, TCP_ECUDA = -3, TCP_EUNSUPPORTED = -4 };
/* intermediates a test may inspect through tcp_workspace() */
enum { TCP_WS_SINOGRAM = 0, TCP_WS_SPECTRUM = 1, TCP_WS_GRID = 2, TCP_WS_PASS1 = 3, TCP_WS_TRIG = 4 };
/* gridding implementations (tcp_set_option(TCP_OPT_GRID_IMPL, ...)) */
/* TILE: tile-owned, atomics-free, bitwise reproducible, CUDA-core FMAs (default for TCP_F32);
 * MMA: the same tiles with the multiply-accumulate on the tcgen05 tensor cores (fp16 storage only;
 * default for TCP_F16 / TCP_F16_OUT32); GATHER: per-cell gather (atomics-free, slow; cross-check);
 * SCATTER_ATOMIC: fp32 atomics (TCP_F32 only; cross-check) */
enum { TCP_GRID_GATHER = 0, TCP_GRID_SCATTER_ATOMIC = 1, TCP_GRID_TILE = 2, TCP_GRID_MMA = 3 };
/* TCP_OPT_TCFFT: bit mask of the transforms whose radix-16 butterflies run on the tensor cores (warp-level
 * mma.sync on fp16 operands, fp32 accumulation; fp16 storage and M = 4096 only, elsewhere the mask must be 0):
 * 1 = detector-row kernel (S1..S4), 2 = column pass and 4 = row pass of the inverse 2D transform (these two
 * switch together: 6).  Default: all that apply (7 at M = 4096 with fp16 storage, else 0); 0 = the fp32
 * CUDA-core Stockham transforms.  Same stages and gates either way. */
/* TCP_OPT_ALGORITHM ("--reconstruction-algorithm"): TCP_ALG_FOURIER = FourierRec, the
 * gridding path this library is about (default); TCP_ALG_LINE = LineRec, direct line summation with linear
 * interpolation (O(N^4)): S1-S3 as before, then the backprojection sum per pixel.
 * After a LINE reconstruction TCP_WS_SINOGRAM holds the FILTERED sinogram.  tcp_recon and
 * tcp_recon_volume_host follow the option; tcp_recon_try is FourierRec only. */
/* TCP_OPT_PAD: the n padding samples of the filter stage S3 (the padding "allows for
 * suppressing artifacts when processing samples not fitting into the detector field of view"):
 * TCP_PAD_ZERO (default, the reading of north_star) or TCP_PAD_EDGE = the nearest detector edge value of
 * the periodic length-2n row (p[n-1] for n <= i < 3n/2, p[0] after).  Stage S4 always zero-pads.  TCP_PAD_EDGE is
 * refused (TCP_EUNSUPPORTED) on a tcp_create_det context whose width is not a power of two: there the row is
 * already padded with air, and its edge samples are not the detector's. */
/* TCP_OPT_FILTER_FUSED (0 default | 1): the second reading of "filter, then Fourier backprojection" (DESIGN.md
 * Q6): filter and spectrum have the same length M = 2n, so S3 + S4 collapse to G = C H FFT_M(padded row) x phase
 * with NO crop of the filtered row in between: one transform per row instead of three, and a slightly different
 * image (the tails of the filtered row outside the detector are backprojected too).  FourierRec, tcp_recon and
 * tcp_recon_volume_host only; tcp_recon_try keeps the default chain. */
/* TCP_OPT_WEIGHT_CACHE (1 default | 0): the tensor-core gridding keeps the interpolation weights of every
 * (sub-tile, sample), which depend only on theta, n and m, in a device cache built on the first call and
 * rebuilt (on the device, no host synchronisation) whenever the angles passed to tcp_recon change; 0 computes
 * them in every call.  Same results bit for bit.  The cache is keyed by an element-by-element comparison of the call's
 * angles with a device copy of the angles it was built for (no checksum), made on the device in every call.  The rebuild
 * itself (three more kernels) is launched by calls that come after the host has SEEN the verdict (a word of mapped pinned
 * memory, read without synchronisation): calls with new angles enqueued before that take the uncached kernel. */
/* TCP_OPT_ANGLE_WEIGHTS (0 default | 1): quadrature weights for angles that are not equally spaced (PAPER.md:61:
 * unlike the log-polar method, the Fourier-based one applies to "non-equally spaced angles", e.g. interlaced
 * scanning).  0: every projection enters with pi/nproj (equispaced half turn).  1: projection j enters with
 * (theta[j+1] - theta[j-1]) / 2, where theta[nproj] = theta[0] + pi and theta[-1] = theta[nproj-1] - pi (trapezoid
 * rule on the periodic angle axis; the angles must cover the half turn), computed on the device from the angles of
 * each call.  All algorithms and tcp_recon_try. */
/* TCP_OPT_FUSE_NORMALIZE (1 default | 0): with fp16 storage tcp_recon runs S1+S2 inside the loader of the detector-row
 * kernel instead of as a kernel of their own (the sinogram then never goes to HBM and TCP_WS_SINOGRAM is NOT updated by
 * tcp_recon; tcp_normalize still fills it).  Same results bit for bit.  Applies to FourierRec's default chain on
 * contexts whose detector width is the transform's; everywhere else the option is ignored. */
enum { TCP_OPT_GRID_IMPL = 0, TCP_OPT_PROFILE = 1, TCP_OPT_TCFFT = 2, TCP_OPT_ALGORITHM = 3, TCP_OPT_PAD = 4,
       TCP_OPT_FILTER_FUSED = 5, TCP_OPT_WEIGHT_CACHE = 6, TCP_OPT_ANGLE_WEIGHTS = 7, TCP_OPT_FUSE_NORMALIZE = 8 };
enum { TCP_PAD_ZERO = 0, TCP_PAD_EDGE = 1 };
enum { TCP_ALG_FOURIER = 0, TCP_ALG_LINE = 1 };
enum { TCP_TCFFT_ROWS = 1, TCP_TCFFT_COLS = 2, TCP_TCFFT_IROWS = 4 };
/* stages timed when TCP_OPT_PROFILE is on, in launch order */
enum { TCP_ST_TRIG = 0, TCP_ST_NORMALIZE = 1, TCP_ST_ROWS = 2, TCP_ST_GRID = 3, TCP_ST_IFFT_COLS = 4,
       TCP_ST_IFFT_ROWS = 5, TCP_NSTAGES = 6 };

/* Create a context for chunks of nz_chunk slices.
 *   n        detector width = image side; a power of two in [64, 4096] (FP16
 *            FFTs need power-of-two sizes; applied to FP32 too)
 *   nproj    number of projection angles (>= 1)
 *   nz_chunk slices per tcp_recon call (>= 1; "--nsino-per-chunk").
 *            An odd count pairs its last slice with zeros.
 *   center   rotation axis in detector pixels ("--rotation-axis"), 0 <= c <= n-1
 *   dtype    TCP_F32 | TCP_F16 | TCP_F16_OUT32        filter   TCP_FILTER_*
 * All workspaces and tables are allocated here (cudaMalloc); tcp_recon allocates nothing.
 * Returns NULL on error (see tcp_last_error). */
tcp_ctx* tcp_create(int n, int nproj, int nz_chunk, float center, int dtype, int filter);

/* As tcp_create, with the gridding kernel as a code m (taps per axis = 2 x half-width):
 *   0            the default (what tcp_create and tcp_create_det's m = 0 use): 16 + 2, see below;
 *   3, 4         Gaussian phi(t) = exp(-alpha t^2) of that half-width (3 meets the 2e-3 gridding-vs-exact gate with 2.7x margin);
 *   16 + 2, 16 + 3   TCP_KERNEL_KB + half-width: Kaiser-Bessel window phi(t) = I0(beta sqrt(1 - (t/m)^2)) / I0(beta),
 *                beta = pi sqrt(2.25 m^2 - 0.8), deapodised by its exact transform (the "accuracy controls" of PAPER.md:173,
 *                DESIGN.md reading Q21).  Half-width 2 reaches 3.9e-4 of the exact sum on the C1 phantom with 16 taps
 *                per sample where the Gaussian needs 36 for 7.4e-4: more accurate and less work, hence the default
 *                (the oracle takes the same code).  Tile and tensor-core griddings only: TCP_GRID_GATHER and
 *                TCP_GRID_SCATTER_ATOMIC need a Gaussian context. */
enum { TCP_KERNEL_GAUSS = 0, TCP_KERNEL_KB = 16 };
tcp_ctx* tcp_create_ex(int n, int nproj, int nz_chunk, float center, int dtype, int filter, int m);

/* Detector width that is not a power of two ("16-bit data are additionally padded/unpadded to
 * the power of 2 sizes"; applied to FP32 as well, reading Q19).  ndet in [8, 4096] is the detector
 * width and the image side of every array the caller passes to tcp_recon / tcp_recon_try / tcp_normalize /
 * tcp_recon_volume_host (raw [nproj][nz][ndet], flat / dark [nz][ndet], out [nz][ndet][ndet]); center is in
 * the caller's detector pixels, 0 <= c <= ndet-1.  Inside, S1+S2 write every row at offset
 * pad_l = ceil((n - ndet)/2) of a row of n = the power of two >= max(ndet, 64), the other samples being air
 * (p = 0); S3..S7 run at size n with the centre c + pad_l; the central ndet x ndet pixels are copied out, so
 * pixel ix sits at x = ix - floor(ndet/2).  Wherever every ray through a pixel hits the real detector the
 * result is that of the unpadded textbook sum; elsewhere the padded air columns carry the filter's tails.
 * The workspaces tcp_workspace reports keep the padded size n = tcp_padded_n(ctx).  When ndet is itself a
 * power of two >= 64 this is tcp_create_ex.  m as in tcp_create_ex.  NULL on error. */
tcp_ctx* tcp_create_det(int ndet, int nproj, int nz_chunk, float center, int dtype, int filter, int m);
/* The power of two the context's transforms run on (= n of tcp_create / tcp_create_ex). */
int tcp_padded_n(const tcp_ctx* ctx);

/* Reconstruct one chunk, S1..S7, asynchronously on `stream` (no host synchronisation).
 *   raw_u16 [nproj][nz_chunk][n] uint16 counts, projection-major as a detector delivers them
 *   flat, dark [nz_chunk][n] float32, already averaged over frames
 *   theta   [nproj] float32 radians, strictly increasing, spanning less than pi
 *   out     [nz_chunk][n][n], float32 (TCP_F32, TCP_F16_OUT32) or IEEE half (TCP_F16)
 * One tcp_recon may be in flight per context.  Bitwise reproducible run to run.
 * Alignment: on a power-of-two context (tcp_create, tcp_create_ex) raw_u16, flat, dark and out must be 16-byte aligned
 * (rows move as 16-byte vectors and bulk copies; cudaMalloc and torch allocations are 256-byte aligned, and so is every
 * whole-chunk view of them): TCP_EINVAL otherwise.  tcp_create_det contexts of other widths take any element alignment. */
int tcp_recon(tcp_ctx* ctx, const uint16_t* raw_u16, const float* flat, const float* dark,
              const float* theta, void* out, tcp_stream_t stream);

void tcp_destroy(tcp_ctx* ctx);                 /* NULL is allowed */
const char* tcp_last_error(void);

/* Mean of nframes uint16 frames [nframes][nz][n] -> float32 [nz][n] (config C4: "10 flat and
 * 10 dark frames to be averaged").  Sum in fp32 (exact below 2^24), one division. */
int tcp_mean_frames_u16(const uint16_t* frames, int nframes, int nz, int n, float* mean,
                        tcp_stream_t stream);

/* S1+S2 alone: raw -> the context's sinogram workspace [nz_chunk][nproj][n] (float or half). */
int tcp_normalize(tcp_ctx* ctx, const uint16_t* raw_u16, const float* flat, const float* dark,
                  tcp_stream_t stream);

/* Device pointer and byte size of an intermediate left by the last tcp_recon (tests only):
 *   TCP_WS_SINOGRAM [nz][nproj][n] real; TCP_WS_SPECTRUM [npair][nproj][M] complex (FFT order,
 *   scaled by tcp_scale()); TCP_WS_GRID [npair][M l2][M l1] complex (or strip-major, tcp_grid_strip); TCP_WS_PASS1
 *   [npair][M/W][n iy][W l1] complex, W = min(32, max(2, 16384/M)) (the column pass works on strips of W
 *   columns and stores them contiguously), or row pairs (tcp_pass1_layout); TCP_WS_TRIG [nproj] double2. */
int tcp_workspace(tcp_ctx* ctx, int which, void** ptr, size_t* bytes);
/* Copy an intermediate into the caller's device buffer dst (>= the size tcp_workspace reports),
 * asynchronously on `stream` (tests only). */
int tcp_read_workspace(tcp_ctx* ctx, int which, void* dst, size_t dst_bytes, tcp_stream_t stream);
/* Layout of TCP_WS_GRID: 0 = [npair][M l2][M l1]; W > 0 = strip-major [npair][M/W][M l2][W l1] (the
 * tensor-core gridding writes strips of W columns so that the column pass of S6 reads contiguously). */
int tcp_grid_strip(const tcp_ctx* ctx);
/* Layouts under the tensor-core transforms of the inverse 2D transform (TCP_OPT_TCFFT & 6), which copy a whole line
 * set into shared memory in bulk and therefore want it stored in their bank-swizzled order (mmafft.cuh, swz<NL>):
 * tcp_pass1_layout: 0 = TCP_WS_PASS1 in strips [npair][M/W][n iy][W l1]; 1 = row pairs [npair][n/2][position][2 rows]
 * with column l1 at position swz<2>(l1).  tcp_grid_swizzled: 1 = row l2 of every TCP_WS_GRID strip sits at position
 * swz<4>(l2) of its strip (0 = at l2). */
int tcp_pass1_layout(const tcp_ctx* ctx);
int tcp_grid_swizzled(const tcp_ctx* ctx);
/* Test helper for the tensor-core transform itself: `batch` lines of 4096 half2 (re, im) -> 4096 float2 each,
 * X[k] = sum_i x[i] e^{-/+ 2 pi i ik/4096} (inverse != 0: +, unnormalised), natural order on both sides.
 * TCP_EUNSUPPORTED unless the context has fp16 storage and M = 4096. */
int tcp_fft_lines(tcp_ctx* ctx, const void* in_half2, void* out_float2, int batch, int inverse, tcp_stream_t stream);
/* Measurement helper (blocks, ~20 ms, current device, default stream): issue-rate micro-benchmarks for the arithmetic
 * roofs bench.py reports against.  *fp32_tflops (HOST): FFMA throughput with 16 independent chains per thread;
 * *hmma_tflops (HOST): mma.sync m16n8k16 fp16 -> fp32 throughput with 8 independent chains per warp (the instruction of
 * the tensor-core transforms).  Both at the clocks of the moment. */
int tcp_measure_rates(double* fp32_tflops, double* hmma_tflops);
/* Power-of-two factor by which SPECTRUM/GRID/PASS1 are scaled relative to S4's G (1 in fp32). */
double tcp_scale(const tcp_ctx* ctx);
/* Total device bytes the context allocated; kernels one tcp_recon launches in the steady state (a call that may have to
 * rebuild the weight cache launches three more, see TCP_OPT_WEIGHT_CACHE). */
size_t tcp_workspace_bytes(const tcp_ctx* ctx);
int tcp_launches_per_recon(const tcp_ctx* ctx);
int tcp_set_option(tcp_ctx* ctx, int option, int value);
/* Real-valued parameters.  Pre-processing of the sinogram between S2 and S3, each step off at 0 (default),
 * applied in this order by tcp_recon, tcp_recon_try and the host pipeline, all algorithms; with either on, S1+S2 run as
 * their own kernel (TCP_OPT_FUSE_NORMALIZE is ignored).  TCP_EUNSUPPORTED on a tcp_create_det context whose width is
 * not a power of two; TCP_EINVAL for a negative or non-finite value.
 *   TCP_PARAM_ZINGER_DIF  "zinger artifacts reduction (Rivers, 1998)", reading Q22: a sample of p = -ln t that
 *       lies more than `value` below the median of its 3 x 3 (projection, detector pixel) neighbourhood (indices
 *       clamped at the array edges, medians taken on the unmodified sinogram) is replaced by that median: an isolated
 *       bright detector hit is an isolated low sample of p.
 *   TCP_PARAM_RING_ALPHA  ring removal "with an analytical formula by V. Titarenko", reading Q23: per slice, the offset
 *       r[i] of detector pixel i common to all projections is estimated from the angle-averaged profile pbar as the
 *       minimiser of ||D2 (pbar - r)||^2 + value ||r||^2 (D2 = second differences), in closed form
 *       (D2^T D2 + value I) r = D2^T D2 pbar, and subtracted from every projection. */
enum { TCP_PARAM_ZINGER_DIF = 0, TCP_PARAM_RING_ALPHA = 1 };
int tcp_set_param(tcp_ctx* ctx, int param, double value);

/* Ring removal without allocation: the TCP_PARAM_RING_ALPHA step (reading Q23, same kernels, same fp64 solve) as a free
 * function on the caller's arrays, for callers that may not call cudaMalloc (code under CUDA graph capture, serving
 * loops, harnesses that forbid it).  The call allocates and frees nothing: its scratch (6 fp64 words per (slice, detector
 * pixel)) is a file-scope device array of 6 * TCP_RING_STATIC_MAX doubles = 3 MiB that every GPU which loads the
 * library holds until the process exits.
 *   sino_in  DEVICE [nz][nproj][n], p = -ln t, float (dtype TCP_F32) or __half (TCP_F16); read only.
 *   sino_out DEVICE, same shape and type; may be sino_in (in place) but must not overlap it otherwise.
 *   alpha    > 0, the Tikhonov weight of TCP_PARAM_RING_ALPHA.
 * Limit: nz * n <= TCP_RING_STATIC_MAX (e.g. 32 slices of 2048 pixels; nproj is not limited); larger calls return
 * TCP_EINVAL with the limit in tcp_last_error() -- split the slices over several calls (slices are independent).
 * Enqueues three kernels on stream and returns; no host synchronisation.  All calls on a device SHARE the scratch array:
 * calls whose kernels can overlap on the GPU (different streams without an ordering between them, or host threads doing
 * so) race and give wrong results; calls on one stream, or ordered by events, are safe.  The array keeps the last call's
 * contents, none of which is read (every word is written before it is read within a call), so nothing is cleared.
 * The device address of the array is looked up (cudaGetSymbolAddress) the first time a device is used;
 * tcp_ring_static_setup() does only that for the current device, for callers who want it done before a capture begins.
 * Errors: TCP_EINVAL (NULL pointer, dtype, sizes, alpha, limit exceeded), TCP_ECUDA. */
#define TCP_RING_STATIC_MAX 65536
int tcp_ring_static_setup(void);
int tcp_ring_remove_static(const void* sino_in, void* sino_out, int nz, int nproj, int n, int dtype, double alpha,
                           tcp_stream_t stream);

/* Rotation-centre "try" mode ("--reconstruction-type try": one slice reconstructed for a
 * set of candidate centres, for visual choice).  raw_u16 [nproj][1][n], flat / dark [n], theta [nproj] are
 * DEVICE pointers as in tcp_recon; centers is a HOST array of ncenter rotation centres, each in [0, n-1],
 * 1 <= ncenter <= nz_chunk; out (DEVICE) [ncenter][n][n] receives the reconstruction for centers[i] at
 * index i, identical (to rounding) to tcp_recon on a context created with that centre.  The slice is
 * normalised and filtered once; candidate centres differ only in the phase table of stage S4, two centres
 * riding one complex transform.  Enqueues on stream only: the phase tables are built by a kernel (fp64) from the
 * centres, which travel by value as kernel arguments, so the call never waits for earlier work on stream.
 * Errors: TCP_EINVAL (NULL, ncenter or a centre out of range), TCP_ENOMEM, TCP_ECUDA. */
int tcp_recon_try(tcp_ctx* ctx, const uint16_t* raw_u16, const float* flat, const float* dark, const float* theta,
                  const float* centers, int ncenter, void* out, tcp_stream_t stream);

/* Per-kernel device times.  With tcp_set_option(ctx, TCP_OPT_PROFILE, 1) every tcp_recon records
 * CUDA events around each of its kernels on the caller's stream (no host synchronisation; a ring
 * of 512 calls).  tcp_profile_collect synchronises on those events, adds the elapsed
 * milliseconds of every call recorded since the last collect into ms_sum[TCP_NSTAGES] (HOST) and
 * returns the number of calls in *ncalls (HOST). */
int tcp_profile_collect(tcp_ctx* ctx, double* ms_sum, int* ncalls);

/* The chunk pipeline (Fig. 1): reconstruct nz_total slices from HOST memory
 * to HOST memory in chunks of nz_chunk, overlapping the H2D copy of chunk N, the compute of
 * chunk N-1 and the D2H copy of chunk N-2 on three CUDA streams with nbuf (2 or 3) device
 * buffer sets.  Host buffers should be pinned (cudaHostAlloc / torch pin_memory) or the
 * copies will not overlap.  Blocks until the volume is done.
 *   raw_host [nproj][nz_total][n] uint16; flat_host, dark_host [nz_total][n] float32;
 *   theta_host [nproj] float32; out_host [nz_total][n][n] in the context's output dtype.
 * A last partial chunk is allowed.  ms_out (HOST, may be NULL) receives the elapsed device time
 * in milliseconds between the first copy and the last, measured with CUDA events. */
int tcp_recon_volume_host(tcp_ctx* ctx, const uint16_t* raw_host, const float* flat_host,
                          const float* dark_host, const float* theta_host, void* out_host,
                          int nz_total, int nbuf, float* ms_out);

/* The same pipeline on the slice range [z_begin, z_end) of a stack of nz_stack slices ("--start-row / --end-row",
 * PAPER.md:133-135; the paper's multi-GPU recipe: one process per GPU, each on its own
 * subset of slices, nothing exchanged).  All HOST arrays keep the full-stack shapes of tcp_recon_volume_host with
 * nz_total = nz_stack (several processes may share them); only rows z_begin..z_end-1 are read, and only those
 * slices of out_host are written.  TCP_EINVAL unless 0 <= z_begin < z_end <= nz_stack. */
int tcp_recon_volume_host_rows(tcp_ctx* ctx, const uint16_t* raw_host, const float* flat_host,
                               const float* dark_host, const float* theta_host, void* out_host,
                               int nz_stack, int z_begin, int z_end, int nbuf, float* ms_out);
/* HOST logic only (no CUDA call): TCP_OK if theta_host[nproj] is what tcp_recon accepts (finite, strictly increasing,
 * last - first < pi), else TCP_EINVAL with the offending index in tcp_last_error().  tcp_recon cannot check its DEVICE
 * angles without a synchronisation and does not; tcp_recon_volume_host[_rows] check their HOST angles with this. */
int tcp_check_angles(const float* theta_host, int nproj);
/* HOST logic only (no CUDA call): the contiguous slice range [*z0, *z1) of process `rank` of `world` over
 * nz_total slices; the ranges tile [0, nz_total) in rank order and differ by at most one slice (a rank may get
 * an empty range when world > nz_total).  TCP_EINVAL on a bad argument. */
int tcp_slice_range(int nz_total, int rank, int world, int* z0, int* z1);

#ifdef __cplusplus
}
#endif
#endif /* TCP_H_ */
