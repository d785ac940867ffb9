// k_mmafft.cu -- the three transform kernels of the fp16 path at M = 4096 with their radix-16 butterflies on the
// tensor cores (mmafft.cuh): S1+S2+S3+S4 per detector row (rows_mma_kernel), and the two passes of the inverse 2D
// transform S6 with S7 fused (cols_mma_kernel, irows_mma_kernel).  Same stages, tables and layouts at the HBM
// boundaries as k_rows.cu / k_ifft2.cu except the pass-1 array, which holds ROW PAIRS here:
//   pass1[pair][iy / 2][l1][iy % 2]   (half2)
// so that the column pass stores 32 contiguous bytes per thread (4 columns x 2 rows) and the row pass, which
// transforms rows iy and iy + 1 in one CTA, loads both with one 8-byte access per element.
#include <math.h>

#include <algorithm>
#include <vector>

#include "mmafft.cuh"
#include "umma.cuh"
#include "tcp_internal.h"

namespace tcpk {

using namespace mf;

static const double kPiM = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------------ tables (host, fp64)
static int inmap(int variant, int q) {                   // input digit held in K slot q' (mmafft.cuh "MMA mapping")
    if (variant == AV_NAT) return q;
    const int c = q & 3, i = q >> 2;                     // pass 3 loads digits (2c, 2c+1) and (8+2c, 9+2c) as 8-byte pairs
    return (i & 1) + 2 * c + 8 * (i >> 1);
}
static int outmap(int variant, int t, int r) {           // output digit of tile t, row r (re) and r + 8 (im)
    if (variant == AV_LOC) return t == 0 ? (r < 4 ? r : r + 8) : r + 4;
    return r + 8 * t;
}
static void build_atab(std::vector<uint32_t>& tab) {
    tab.assign(ATAB_WORDS, 0u);
    auto h16 = [](double v) { return (uint32_t)__half_as_ushort(__float2half_rn((float)v)); };
    for (int v = 0; v < AV_COUNT; ++v)
        for (int lane = 0; lane < 32; ++lane) {
            const int g = lane >> 2, c = lane & 3;
            for (int t = 0; t < 2; ++t)
                for (int s = 0; s < 2; ++s)
                    for (int r = 0; r < 4; ++r) {
                        const int row = g + 8 * (r & 1);                    // tile row
                        const int q = 8 * s + c + 4 * (r >> 1);             // K slot: columns 2q (re), 2q + 1 (im)
                        const int o = outmap(v, t, row & 7), j = inmap(v, q);
                        const double a = 2.0 * kPiM * (double)((o * j) & 15) / 16.0;
                        const double fr = GAMMA * cos(a), fi = -GAMMA * sin(a);   // W_16^(o j) = fr + i fi
                        // re row: (fr, -fi) . (x_re, x_im); im row: (fi, fr)
                        const double e0 = row < 8 ? fr : fi, e1 = row < 8 ? -fi : fr;
                        tab[((size_t)v * 32 + lane) * 16 + t * 8 + s * 4 + r] = h16(e0) | (h16(e1) << 16);
                    }
        }
}

int mmafft_setup(tcp_ctx* c) {
    c->mf_ok = 0;
    if (!c->half_store || c->M != N) return TCP_OK;
    std::vector<uint32_t> tab;
    build_atab(tab);
    TCP_CUDA_CHECK(cudaMalloc((void**)&c->mf_atab, tab.size() * sizeof(uint32_t)));
    TCP_CUDA_CHECK(cudaMemcpy(c->mf_atab, tab.data(), tab.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    c->bytes += tab.size() * sizeof(uint32_t);
    c->mf_ok = TCP_TCFFT_ROWS | TCP_TCFFT_COLS | TCP_TCFFT_IROWS;
    return TCP_OK;
}
void mmafft_free(tcp_ctx* c) { cudaFree(c->mf_atab); }

// The filtered row rides fp16 operands between the transforms: Q = H P is stored as 2^12 (H / M) P (typical
// magnitude 1) and the factor is undone in the phase table.
constexpr float kRowScale = 4096.f;

// ------------------------------------------------------------------------------------------------ detector rows
// negate the imaginary output rows (registers 1, 3) of tile 0: the transform then returns the conjugate of its result
__device__ __forceinline__ void conj_tile0(AFrag& f) {
#pragma unroll
    for (int s = 0; s < 2; ++s) { f.a[0][s][1] ^= 0x80008000u; f.a[0][s][3] ^= 0x80008000u; }
}
template <bool PAD_EDGE, bool RAW>
__global__ void __launch_bounds__(NT, 2) rows_mma_kernel(const __half* __restrict__ sino, __half2* __restrict__ spec,
                                                          const float2* __restrict__ tw, const uint32_t* __restrict__ atab,
                                                          const float* __restrict__ hfilt, const float2* __restrict__ ptab, int nproj,
                                                          int nz, int try_mode, const float* __restrict__ wq,
                                                          const uint16_t* __restrict__ raw, const float2* __restrict__ fdtab, int npair_try) {
    constexpr int n = N / 2;
    extern __shared__ __align__(16) uint32_t L[];
    float2* T1TAB = reinterpret_cast<float2*>(L + 1 * N);               // pass-1 twiddle table behind the lines
    // per-thread copies of the tables the epilogues and the loader need, [slot][thread] (conflict free, and a shared-memory
    // wavefront moves 128 bytes where the L1 path of a global load moves a 32-byte sector per cycle)
    float2* HT = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(T1TAB) + T1_BYTES);   // 2^12 H/M at (k0, k0 + 1) of the 8 output pairs
    float4* PT = reinterpret_cast<float4*>(HT + 8 * NT);                // phase table / 2^12 at the same indices
    float4* FD = PT + 8 * NT;                                           // RAW: (1/(flat-dark), dark) of the thread's 8 pixels, slices A and B
    // RAW: the two detector rows of the NEXT projection arrive by bulk asynchronous copies (2 x 4 KB) while this one is
    // transformed; loaded with __ldg at the top of the loop they cost a DRAM latency per unit with nothing to hide it
    // (profiles/r2_kernels.md: 11 % of the warp samples wait on that load)
    uint16_t* RB = reinterpret_cast<uint16_t*>(FD + 8 * NT);            // [2][n]
    uint64_t* rbar = reinterpret_cast<uint64_t*>(RB + 2 * n);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, c = lane & 3;
    // persistent CTAs: the npair x nproj units (pair-major) are cut into gridDim.x contiguous runs of equal length, so a CTA
    // works through consecutive projections of ONE slice pair (two when its run crosses a pair boundary): what depends on the
    // thread and the pair only -- the flat/dark table, in try mode the phase table -- is set up when the pair changes, the
    // butterfly fragments, twiddles and the filter table once.  (A fixed pair per CTA left 8 of the 296 CTA slots idle.)
    const int npair_grid = npair_try;                                  // slice pairs of the call
    const long long nunit = (long long)npair_grid * nproj;
    const int u0 = (int)((long long)blockIdx.x * nunit / gridDim.x), u1 = (int)(((long long)blockIdx.x + 1) * nunit / gridDim.x);
    auto slices_of = [&](int p, int& a, int& bs, bool& hb) {
        a = try_mode ? 0 : 2 * p;
        const int b = try_mode ? nz : 2 * p + 1;
        hb = b < nz;
        bs = hb ? b : a;
    };
    auto fetch_raw = [&](int u) {                                       // thread 0 only
        const int p = u / nproj, j = u - p * nproj;
        int a, bs;
        bool hb;
        slices_of(p, a, bs, hb);
        mbar_expect_tx(rbar, 2 * n * 2);
        bulk_g2s(RB, raw + ((size_t)j * nz + a) * n, n * 2, rbar);
        bulk_g2s(RB + n, raw + ((size_t)j * nz + bs) * n, n * 2, rbar);
    };
    if constexpr (RAW) {
        if (tid == 0) {
            mbar_init(rbar, 1);
            fence_mbar_init();
        }
        __syncthreads();
        if (tid == 0 && u0 < u1) fetch_raw(u0);
    }
    uint32_t rphase = 0;
    const int kbase = pass3_index<false>(0, 0, warp, g, c);
#pragma unroll
    for (int sl = 0; sl < 8; ++sl) {
        const int k0 = kbase + 2048 * (sl & 1) + 64 * (sl >> 1);
        const float2 h = __ldg(reinterpret_cast<const float2*>(hfilt + k0));
        HT[sl * NT + tid] = make_float2(h.x * kRowScale, h.y * kRowScale);
    }
    // the per-thread tables are written and read by the same thread only: no barrier around a change of pair
    auto setup_pair = [&](int p, int zA, int zBs, bool first) {
        if (first || try_mode) {
            const float2* pt = try_mode ? ptab + (size_t)p * N : ptab;
#pragma unroll
            for (int sl = 0; sl < 8; ++sl) {
                const int k0 = kbase + 2048 * (sl & 1) + 64 * (sl >> 1);
                const float4 v = __ldg(reinterpret_cast<const float4*>(pt + k0));
                const float s = 1.f / kRowScale;
                PT[sl * NT + tid] = make_float4(v.x * s, v.y * s, v.z * s, v.w * s);
            }
        }
        if constexpr (RAW) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                FD[q * NT + tid] = __ldg(reinterpret_cast<const float4*>(fdtab + (size_t)zA * n + tid * 8) + q);
                FD[(4 + q) * NT + tid] = __ldg(reinterpret_cast<const float4*>(fdtab + (size_t)zBs * n + tid * 8) + q);
            }
        }
    };
    AFrag An, Al;
    load_afrag(An, atab, AV_NAT, lane);
    load_afrag(Al, atab, AV_LO, lane);
    Twid T;
    load_twid(T, T1TAB, tw, warp, g, c, (float)(1.0 / GAMMA), (float)(1.0 / (GAMMA * GAMMA)));
    __syncwarp();
    Offs<1> O;
    make_offs<1>(O, warp, g, c);
    auto no_in = [](int) { return 0u; };
    auto slot_of = [&](int k0) { return 2 * (((k0 - kbase) >> 6) & 3) + ((k0 - kbase) >> 11); };   // folds to a constant per call site
    int pair = -1, zA = 0, zBs = 0;
    bool hasB = false;
#pragma unroll 1
    for (int u = u0; u < u1; ++u) {
    const int up = u / nproj, j = u - up * nproj;
    if (up != pair) {
        const bool first = pair < 0;
        pair = up;
        slices_of(pair, zA, zBs, hasB);
        setup_pair(pair, zA, zBs, first);
    }
    const float wj = wq ? __ldg(&wq[j]) : 1.f;

    // ---- stage the two rows as half2 (pA, pB): 8 detector pixels per thread, 128-bit loads
    {
        const int i0 = tid * 8;
        float a[8], b[8];
        if constexpr (RAW) {
            mbar_wait(rbar, rphase);
            rphase ^= 1;
            const uint4 ra = *reinterpret_cast<const uint4*>(RB + i0);
            const uint4 rb = *reinterpret_cast<const uint4*>(RB + n + i0);
            const unsigned ua[4] = {ra.x, ra.y, ra.z, ra.w}, ub[4] = {rb.x, rb.y, rb.z, rb.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 da = FD[q * NT + tid], db = FD[(4 + q) * NT + tid];      // (rcp, dark) of pixels 2q, 2q + 1
                // S1+S2 with the arithmetic of normalize_half_kernel (tcp_internal.h), rounded to the storage type
                a[2 * q] = -0.69314718055994531f * fast_lg2(fmaxf((u16f(ua[q] & 0xffffu) - da.y) * da.x, 1e-6f));
                a[2 * q + 1] = -0.69314718055994531f * fast_lg2(fmaxf((u16f(ua[q] >> 16) - da.w) * da.z, 1e-6f));
                b[2 * q] = -0.69314718055994531f * fast_lg2(fmaxf((u16f(ub[q] & 0xffffu) - db.y) * db.x, 1e-6f));
                b[2 * q + 1] = -0.69314718055994531f * fast_lg2(fmaxf((u16f(ub[q] >> 16) - db.w) * db.z, 1e-6f));
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) { a[q] = __half2float(__float2half_rn(a[q])); b[q] = __half2float(__float2half_rn(b[q])); }
        } else {
            const uint4 ha = __ldg(reinterpret_cast<const uint4*>(sino + ((size_t)zA * nproj + j) * n + i0));
            const uint4 hb = __ldg(reinterpret_cast<const uint4*>(sino + ((size_t)zBs * nproj + j) * n + i0));
            const unsigned ua[4] = {ha.x, ha.y, ha.z, ha.w}, ub[4] = {hb.x, hb.y, hb.z, hb.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float2 fa = __half22float2(*reinterpret_cast<const __half2*>(&ua[q])), fb = __half22float2(*reinterpret_cast<const __half2*>(&ub[q]));
                a[2 * q] = fa.x; a[2 * q + 1] = fa.y; b[2 * q] = fb.x; b[2 * q + 1] = fb.y;
            }
        }
        uint32_t w[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) w[q] = pack_h2(a[q] * wj, hasB ? b[q] * wj : 0.f);
        uint4* dst = reinterpret_cast<uint4*>(&L[swz<1>(i0)]);
        dst[0] = make_uint4(w[0], w[1], w[2], w[3]);
        dst[1] = make_uint4(w[4], w[5], w[6], w[7]);
    }
    __syncthreads();
    if constexpr (RAW) {                  // every thread has read the raw rows: the next projection's may land
        if (tid == 0 && u + 1 < u1) {
            fence_proxy_async();
            fetch_raw(u + 1);
        }
    }
    if constexpr (PAD_EDGE) {     // padding samples of the filter stage: the nearest edge of the periodic row
        const uint32_t last = L[swz<1>(n - 1)], first = L[swz<1>(0)];
        const uint32_t v = tid < NT / 2 ? last : first;
        uint4* dst = reinterpret_cast<uint4*>(&L[swz<1>(n + tid * 8)]);
        dst[0] = make_uint4(v, v, v, v);
        dst[1] = make_uint4(v, v, v, v);
        __syncthreads();
    }

    // ---- transform 1: spectrum of the padded row, times 2^12 H / M
    pass1<1, false, !PAD_EDGE, true>(L, An, T, O, warp, g, c, no_in);
    __syncthreads();
    pass2<1, false>(L, An, T, O);
    __syncthreads();
    // the epilogue stores conj(Q): the inverse transform below is conj(FFT(conj(Q))), i.e. a FORWARD transform whose
    // pass-3 fragments have their imaginary rows negated (4 sign flips instead of 64 to turn both fragment sets around)
    pass3<1, false, false, true>(L, Al, O, warp, g, c, [&](int k0, const float2(&y0)[1], const float2(&y1)[1]) {
        const float2 h = HT[slot_of(k0) * NT + tid];
        const float h0 = h.x, h1 = h.y;
        *reinterpret_cast<uint2*>(&L[swz<1>(k0)]) = make_uint2(pack_h2(y0[0].x * h0, y0[0].y * -h0), pack_h2(y1[0].x * h1, y1[0].y * -h1));
    });
    __syncthreads();
    // ---- transform 2 (inverse, see above): the filtered row, cropped to the detector (only tile 0 = samples below n is computed)
    pass1<1, false, false, true>(L, An, T, O, warp, g, c, no_in);
    __syncthreads();
    pass2<1, false>(L, An, T, O);
    __syncthreads();
    conj_tile0(Al);
    pass3<1, true, false, true>(L, Al, O, warp, g, c, [&](int k0, const float2(&y0)[1], const float2(&y1)[1]) {
        *reinterpret_cast<uint2*>(&L[swz<1>(k0)]) = make_uint2(pack_h2(y0[0].x, y0[0].y), pack_h2(y1[0].x, y1[0].y));
    });
    conj_tile0(Al);
    __syncthreads();
    // ---- transform 3: spectrum of the zero-padded filtered row, centre phase and scale on store
    pass1<1, false, true, true>(L, An, T, O, warp, g, c, no_in);
    __syncthreads();
    pass2<1, false>(L, An, T, O);
    __syncthreads();
    __half2* out = spec + ((size_t)pair * nproj + j) * N;
    pass3<1, false, false, false>(L, Al, O, warp, g, c, [&](int k0, const float2(&y0)[1], const float2(&y1)[1]) {
        const float4 p = PT[slot_of(k0) * NT + tid];
        const float2 v0 = make_float2(y0[0].x * p.x - y0[0].y * p.y, y0[0].x * p.y + y0[0].y * p.x);
        const float2 v1 = make_float2(y1[0].x * p.z - y1[0].y * p.w, y1[0].x * p.w + y1[0].y * p.z);
        *reinterpret_cast<uint2*>(out + k0) = make_uint2(pack_h2(v0.x, v0.y), pack_h2(v1.x, v1.y));
    });
    __syncthreads();                      // the line is free for the next unit's rows
    }
}

// ------------------------------------------------------------------------------------------------ column pass of S6
// One unit = one strip of 4 adjacent columns of the strip-major grid [pair][M/4][M l2][4 l1], whose rows the gridding
// kernel stores at position swz<4>(l2) (tcp_internal.h: ifft2_on_mma): the 64 KB block is exactly the team's 4
// interleaved lines, and ONE bulk asynchronous copy (TMA) brings it in.  Persistent CTAs; while one CTA of an SM waits for
// its copy the others transform.  Only the central n outputs are computed in the last pass (tile 0 of the AV_LOC fragments).
// Output: pass1[pair][iy / 2][swz<2>(l1)][iy % 2] -- the row pass loads its lines the same way.  A thread holds 32
// contiguous bytes (4 columns x 2 rows); lane pairs swap halves so that every 16-byte store instruction fills whole sectors.
__device__ __forceinline__ void st_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.global.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
// Samples lie within radius n of DC and reach at most 4 cells further, so in a strip of columns |x| >= xmin only the rows
// |l2| < h = sqrt((n + 8)^2 - xmin^2) can be non-zero (a fifth of the grid is corners that the gridding never writes): the
// rows [0, h) and [M - h, M) come from the grid, the rows between from this block of zeros, which stays in L2.  Row positions
// are swizzled within aligned groups of 8 (swz<4>), so h is rounded up to a multiple of 8.
__device__ __align__(128) uint4 g_zero_rows[N];
__global__ void __launch_bounds__(NT, 2) cols_mma_kernel(const uint4* __restrict__ grid, uint2* __restrict__ p1arr,
                                                          const float2* __restrict__ tw, const uint32_t* __restrict__ atab, int nunits) {
    constexpr int n = N / 2;
    extern __shared__ __align__(128) uint32_t L[];
    float2* T1TAB = reinterpret_cast<float2*>(L + 4 * N);
    uint64_t* bar = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(T1TAB) + T1_BYTES);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, c = lane & 3;
    auto fetch_strip = [&](int unit) {                                    // thread 0 only: 64 KB in one, or in three copies
        const int l1 = 4 * (unit % (N / 4));
        const int xmin = l1 < n ? l1 : N - l1 - 3;                        // smallest |x| of the strip's four columns
        const int R = n + 8;
        int h = (int)sqrtf((float)(R * R - xmin * xmin)) + 2;
        h = (h + 7) & ~7;
        const uint4* src = grid + (size_t)unit * N;
        uint4* dst = reinterpret_cast<uint4*>(L);
        mbar_expect_tx(bar, 4 * N * 4);
        if (2 * h >= N) {
            bulk_g2s(dst, src, 4 * N * 4, bar);
        } else {
            bulk_g2s(dst, src, h * 16, bar);
            bulk_g2s(dst + h, g_zero_rows, (N - 2 * h) * 16, bar);
            bulk_g2s(dst + (N - h), src + (N - h), h * 16, bar);
        }
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0 && (int)blockIdx.x < nunits) fetch_strip(blockIdx.x);
    AFrag An, Ac;
    load_afrag(An, atab, AV_NAT, lane);
    flip_afrag(An);
    load_afrag(Ac, atab, AV_LOC, lane);
    flip_afrag(Ac);
    Twid T;
    load_twid(T, T1TAB, tw, warp, g, c, (float)(1.0 / GAMMA), (float)(1.0 / (GAMMA * GAMMA)));
    __syncwarp();
    Offs<4> O;
    make_offs<4>(O, warp, g, c);
    auto no_in = [](int) { return make_uint4(0u, 0u, 0u, 0u); };
    uint32_t phase = 0;
#pragma unroll 1
    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x) {       // unit = pair (N / 4) + strip: consecutive blocks of the grid
    const int strip = unit % (N / 4), pair = unit / (N / 4);
    mbar_wait(bar, phase);
    phase ^= 1;
    pass1<4, true, false, true>(L, An, T, O, warp, g, c, no_in);
    __syncthreads();
    pass2<4, true>(L, An, T, O);
    __syncthreads();
    // columns 4 strip + l sit at swz<2>(4 strip + l) = base + (l ^ x1) of their row pair
    const int sw = swz<2>(4 * strip), x1 = sw & 1;
    unsigned char* dst = reinterpret_cast<unsigned char*>(p1arr + (size_t)pair * (n / 2) * N + (sw & ~3));
    pass3<4, true, true, false>(L, Ac, O, warp, g, c, [&](int k0, const float2(&y0)[4], const float2(&y1)[4]) {
        const int iy0 = k0 < n / 2 ? k0 + n / 2 : k0 - (N - n / 2);       // even; rows iy0 and iy0 + 1 are one pair
        uint32_t w[8];                                                     // the thread's 32 bytes: [position][row]
#pragma unroll
        for (int l = 0; l < 4; ++l) {
            const int pos = l ^ x1;
            const uint32_t a = pack_h2(y0[l].x, y0[l].y), b = pack_h2(y1[l].x, y1[l].y);
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (q == pos) { w[2 * q] = a; w[2 * q + 1] = b; }
        }
        // lanes c and c ^ 1 hold the chunks of row pairs iy0 / 2 and iy0 / 2 +- 1: the even lane takes both first halves,
        // the odd lane both second halves, so that each of the two store instructions writes whole 32-byte sectors
        const bool odd = c & 1;
        uint32_t r[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) r[q] = __shfl_xor_sync(0xffffffffu, odd ? w[q] : w[4 + q], 1);
        unsigned char* mine = dst + (size_t)(iy0 >> 1) * (N * 8);
        unsigned char* other = odd ? mine - N * 8 : mine + N * 8;
        // two unconditional 16-byte stores per thread (addresses and values selected, no divergent branch: the compiler
        // splits a store whose address comes out of a merged branch into four 4-byte stores, 4 x the tag requests)
        st_v4(odd ? other + 16 : mine, odd ? r[0] : w[0], odd ? r[1] : w[1], odd ? r[2] : w[2], odd ? r[3] : w[3]);
        st_v4(odd ? mine + 16 : other, odd ? w[4] : r[0], odd ? w[5] : r[1], odd ? w[6] : r[2], odd ? w[7] : r[3]);
    });
    __syncthreads();                      // the lines are free for the next unit
    if (tid == 0 && unit + (int)gridDim.x < nunits) {
        fence_proxy_async();
        fetch_strip(unit + gridDim.x);
    }
    }
}

// ------------------------------------------------------------------------------------------------ row pass of S6 + S7
__device__ __forceinline__ void st_out2(__half* p, float a, float b) { *reinterpret_cast<uint32_t*>(p) = pack_h2(a, b); }
__device__ __forceinline__ void st_out2(float* p, float a, float b) { *reinterpret_cast<float2*>(p) = make_float2(a, b); }

// One unit = one row pair (iy, iy + 1) of one slice pair: a contiguous 32 KB block of the pass-1 array, columns already
// at their swizzled positions (cols_mma_kernel), brought in by one bulk asynchronous copy.
template <class TO>
__global__ void __launch_bounds__(NT, 2) irows_mma_kernel(const uint2* __restrict__ p1arr, TO* __restrict__ out,
                                                           const float2* __restrict__ tw, const uint32_t* __restrict__ atab,
                                                           const float* __restrict__ deax, const float* __restrict__ deay, int nz, int nunits) {
    constexpr int n = N / 2;
    extern __shared__ __align__(128) uint32_t L0[];                       // two line sets: the next unit arrives while this one is transformed
    float2* T1TAB = reinterpret_cast<float2*>(L0 + 2 * 2 * N);
    uint64_t* bar = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(T1TAB) + T1_BYTES);   // [2]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, c = lane & 3;
    auto fetch = [&](int unit, int b) {                                   // thread 0 only
        mbar_expect_tx(&bar[b], 2 * N * 4);
        bulk_g2s(L0 + b * 2 * N, p1arr + (size_t)unit * N, 2 * N * 4, &bar[b]);
    };
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0 && (int)blockIdx.x < nunits) fetch(blockIdx.x, 0);
    AFrag An, Ac;
    load_afrag(An, atab, AV_NAT, lane);
    flip_afrag(An);
    load_afrag(Ac, atab, AV_LOC, lane);
    flip_afrag(Ac);
    Twid T;
    load_twid(T, T1TAB, tw, warp, g, c, (float)(1.0 / GAMMA), (float)(1.0 / (GAMMA * GAMMA)));
    __syncwarp();
    Offs<2> O;
    make_offs<2>(O, warp, g, c);
    auto no_in = [](int) { return make_uint2(0u, 0u); };
    int it = 0;
#pragma unroll 1
    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++it) { // unit = pair (n / 2) + row pair rp: rows iy = 2 rp, 2 rp + 1
    const int rp = unit % (n / 2), pair = unit / (n / 2);
    const int b = it & 1;
    uint32_t* L = L0 + b * 2 * N;
    // the other line set was last read in pass 3 of the previous unit, which every thread left through the barrier below
    if (tid == 0 && unit + (int)gridDim.x < nunits) {
        fence_proxy_async();
        fetch(unit + gridDim.x, b ^ 1);
    }
    mbar_wait(&bar[b], (it >> 1) & 1);
    pass1<2, true, false, true>(L, An, T, O, warp, g, c, no_in);
    __syncthreads();
    pass2<2, true>(L, An, T, O);
    __syncthreads();
    const int zA = 2 * pair, zB = 2 * pair + 1;
    const bool hasB = zB < nz;
    const float dy0 = __ldg(&deay[2 * rp]), dy1 = __ldg(&deay[2 * rp + 1]);
    TO* oA = out + ((size_t)zA * n + 2 * rp) * n;
    TO* oB = out + ((size_t)zB * n + 2 * rp) * n;
    pass3<2, true, true, false>(L, Ac, O, warp, g, c, [&](int k0, const float2(&y0)[2], const float2(&y1)[2]) {
        const int ix = k0 < n / 2 ? k0 + n / 2 : k0 - (N - n / 2);
        const float2 dx = __ldg(reinterpret_cast<const float2*>(deax + ix));
#pragma unroll
        for (int l = 0; l < 2; ++l) {
            const float d0 = (l ? dy1 : dy0) * dx.x, d1 = (l ? dy1 : dy0) * dx.y;
            st_out2(oA + (size_t)l * n + ix, y0[l].x * d0, y1[l].x * d1);
            if (hasB) st_out2(oB + (size_t)l * n + ix, y0[l].y * d0, y1[l].y * d1);
        }
    });
    __syncthreads();                      // this line set is free
    }
}

// ------------------------------------------------------------------------------------------------ test helper
// batch lines of N half2 -> N float2, natural order both sides (tcp_fft_lines)
template <bool INV>
__global__ void __launch_bounds__(NT, 2) fft_lines_kernel(const uint32_t* __restrict__ in, float2* __restrict__ out,
                                                           const float2* __restrict__ tw, const uint32_t* __restrict__ atab) {
    extern __shared__ __align__(16) uint32_t L[];
    float2* T1TAB = reinterpret_cast<float2*>(L + 1 * N);               // pass-1 twiddle table behind the lines
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, c = lane & 3;
    const uint32_t* src = in + (size_t)blockIdx.x * N;
    float2* dst = out + (size_t)blockIdx.x * N;
    AFrag An, Al;
    load_afrag(An, atab, AV_NAT, lane);
    load_afrag(Al, atab, AV_LO, lane);
    if (INV) { flip_afrag(An); flip_afrag(Al); }
    Twid T;
    load_twid(T, T1TAB, tw, warp, g, c, (float)(1.0 / GAMMA), (float)(1.0 / (GAMMA * GAMMA)));
    __syncwarp();
    Offs<1> O;
    make_offs<1>(O, warp, g, c);
    pass1<1, INV, false, false>(L, An, T, O, warp, g, c, [&](int k) { return __ldg(src + k); });
    __syncthreads();
    pass2<1, INV>(L, An, T, O);
    __syncthreads();
    pass3<1, false, false, false>(L, Al, O, warp, g, c, [&](int k0, const float2(&y0)[1], const float2(&y1)[1]) {
        *reinterpret_cast<float4*>(dst + k0) = make_float4(y0[0].x, y0[0].y, y1[0].x, y1[0].y);
    });
}

// ------------------------------------------------------------------------------------------------ launchers
int launch_rows_mma(const tcp_ctx* c, cudaStream_t st, const uint16_t* raw) {
    const size_t smem = (size_t)N * 4 + T1_BYTES + 8 * NT * (8 + 16 + (raw ? 16 : 0)) + (raw ? 2 * (N / 2) * 2 + 16 : 0);
    auto kern = raw ? (c->pad ? rows_mma_kernel<true, true> : rows_mma_kernel<false, true>)
                    : (c->pad ? rows_mma_kernel<true, false> : rows_mma_kernel<false, false>);
    TCP_SMEM(kern, smem);
    // every CTA takes one contiguous run of the npair x nproj units
    const int nctas = (int)std::min<long long>((long long)c->npair * c->nproj, 2 * c->nsm);
    kern<<<nctas, NT, smem, st>>>((const __half*)c->sino, (__half2*)c->spec, c->tw, c->mf_atab, c->hfilt,
                                                c->try_ptab ? c->try_ptab : c->ptab, c->nproj, c->nz, c->try_ptab ? 1 : 0,
                                                c->angle_weights ? c->wq : nullptr, raw, c->fdtab, c->npair);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_cols_mma(const tcp_ctx* c, cudaStream_t st) {
    const size_t smem = (size_t)4 * N * 4 + T1_BYTES + 16;
    TCP_SMEM(cols_mma_kernel, smem);
    const int nunits = (N / 4) * c->npair;
    cols_mma_kernel<<<std::min(nunits, 2 * c->nsm), NT, smem, st>>>((const uint4*)c->grid, (uint2*)c->pass1, c->tw, c->mf_atab, nunits);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_irows_mma(const tcp_ctx* c, void* out, cudaStream_t st) {
    const size_t smem = (size_t)2 * 2 * N * 4 + T1_BYTES + 16;
    const int nunits = (N / 4) * c->npair;
    const int grid = std::min(nunits, 2 * c->nsm);
    if (c->half_out) {
        TCP_SMEM(irows_mma_kernel<__half>, smem);
        irows_mma_kernel<__half><<<grid, NT, smem, st>>>((const uint2*)c->pass1, (__half*)out, c->tw, c->mf_atab, c->deax, c->deay, c->nz, nunits);
    } else {
        TCP_SMEM(irows_mma_kernel<float>, smem);
        irows_mma_kernel<float><<<grid, NT, smem, st>>>((const uint2*)c->pass1, (float*)out, c->tw, c->mf_atab, c->deax, c->deay, c->nz, nunits);
    }
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

int launch_fft_lines(const tcp_ctx* c, const void* in, void* out, int batch, int inverse, cudaStream_t st) {
    const size_t smem = (size_t)N * 4 + T1_BYTES;
    if (inverse) {
        TCP_SMEM(fft_lines_kernel<true>, smem);
        fft_lines_kernel<true><<<batch, NT, smem, st>>>((const uint32_t*)in, (float2*)out, c->tw, c->mf_atab);
    } else {
        TCP_SMEM(fft_lines_kernel<false>, smem);
        fft_lines_kernel<false><<<batch, NT, smem, st>>>((const uint32_t*)in, (float2*)out, c->tw, c->mf_atab);
    }
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

}  // namespace tcpk
