// tcfft.cuh -- length-4096 complex DFT as two 64-point DFT-as-GEMM stages on the 5th-generation
// tensor cores (tcgen05, fp16 operands, fp32 accumulators in TMEM), for the fp16-storage path.
//
// north_star allows tensor cores for "a DFT-as-GEMM stage [that] measurably wins and is justified by
// ncu": the shared-memory Stockham transforms (fft.cuh) are bound by fp32 instruction issue (about 55
// thread instructions per point and transform, profiles/r1_bench.md), and here the butterflies leave
// the CUDA cores entirely; what stays on them is one twiddle multiply and one fp16 conversion per point
// and stage.
//
// Cooley-Tukey with N = 64 x 64, natural index i = 64 i1 + i2 in, k = 64 k2 + k1 out:
//   stage A   Y[k1][i2]  = sum_i1 W64^(k1 i1) x[64 i1 + i2]
//   twiddle   Y'[k1][i2] = Y[k1][i2] W4096^(k1 i2)
//   stage C   X[64 k2 + k1] = sum_i2 W64^(k2 i2) Y'[k1][i2]
// Both stages are D[128 x N] = A[128 x 128] B[128 x N] with the same constant real matrix
//   A[(k, c)][(i, c')] = [[cos, sin], [-sin, cos]](2 pi k i / 64)        (W = e^{-2 pi i/64}, forward)
// acting on planar data (K index kappa = 64 c' + i: real plane, then imaginary plane) and N = 64 NB
// columns (NB lines side by side).  Row rho = 32 q + 16 c + j of D holds (k = 16 q + j, c): the real and
// the imaginary part of one output sit 16 lanes apart in the same warp, because a warp can only read
// its own quarter of the TMEM lanes and the twiddle needs both (one SHFL per value).
//   stage A: B = x as [kappa][n = (line, i2)], n contiguous  -> MN-major operand, natural input order
//   stage C: B = Y' as [kappa = (c, i2)][n = (line, k1)], kappa contiguous -> K-major operand; thread
//            (row k1) of the twiddle step writes 16-byte runs of its own row
//   D of stage C: row (k2, c) holds the 64 consecutive natural-order outputs 64 k2 + k1 of every line.
// The inverse transform uses the same matrix on swapped planes: IFFT(x) = swap(FFT(swap(x))),
// swap(a + i b) = b + i a, which in planar storage is only a relabelling (template flag SWAP of the
// loaders; rows c = 0 then hold the imaginary and c = 1 the real part of the result).
//
// A group of 128 threads (4 warps = the 4 lane quarters) owns NB lines, one B buffer (16 KB per line,
// reused by both stages), one TMEM accumulator of 64 NB columns and one mbarrier.  Per stage: the
// threads write B, fence.proxy.async, group barrier, one thread issues the K steps and commits, all
// wait on the mbarrier, read D back with tcgen05.ld.
// Rounding: operands are fp16 (data rounded once per stage, matrix entries to 2^-12 relative), sums
// are fp32; measured against the 5e-3 gate in tests/test_gpu_parity.py.
#pragma once
#include <cuda_fp16.h>
#include <math.h>

#include <vector>

#include "umma.cuh"

namespace tcpk {
namespace tcfft {

constexpr int A_BYTES = 128 * 128 * 2;      // the DFT-64 matrix, K-major blocks [mb 16][kb 16][8 m][8 k] half
constexpr int A_LBO = 128, A_SBO = 16 * 128;

template <int NB>
struct Group {
    static constexpr int NT = 64 * NB;              // MMA N
    static constexpr int B_BYTES = 128 * NT * 2;    // one B operand: 128 kappa x NT columns, half
    static constexpr int B1_LBO = (NT / 8) * 128;   // MN-major [kb 16][nb NT/8][8 k][8 n]: k-block stride (n-block stride 128)
    static constexpr int B2_SBO = 16 * 128;         // K-major  [nb NT/8][kb 16][8 n][8 k]: n-block stride (k-block stride 128)
    uint32_t tmem;                                  // TMEM address of D (lane 0, first column)
    uint32_t a_addr, b_addr;                        // shared-memory addresses of A and of this group's B buffer
    unsigned char* bbuf;
    uint64_t* bar;
    uint32_t phase;                                 // parity of the next completion of bar
    int t, q, lane, j, c, barid;                    // thread in group, lane quarter, lane, row in half-quarter, re|im half
};

template <int NB>
__device__ __forceinline__ void group_sync(const Group<NB>& g) {
    asm volatile("bar.sync %0, 128;" ::"r"(g.barid) : "memory");
}

// All threads of the group have written B (generic proxy): publish it to the tensor core, run the K
// steps selected by kmask (bit s = kappa blocks 2s, 2s + 1; a zero block may be skipped) and wait for D.
template <int NB, bool KMAJOR>
__device__ __forceinline__ void stage_mma(Group<NB>& g, uint32_t kmask) {
    using G = Group<NB>;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    group_sync(g);
    if (g.t == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // D fp32, A/B fp16, A K-major, B K- or MN-major, N = NT, M = 128
        constexpr uint32_t IDESC = (1u << 4) | ((KMAJOR ? 0u : 1u) << 16) | ((uint32_t)(G::NT >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        uint32_t acc = 0;
#pragma unroll
        for (int s = 0; s < 8; ++s)
            if ((kmask >> s) & 1u) {
                const uint64_t da = umma_desc(g.a_addr + s * 256, A_LBO, A_SBO);
                const uint64_t db = KMAJOR ? umma_desc(g.b_addr + s * 256, 128, G::B2_SBO)
                                           : umma_desc(g.b_addr + s * 2 * G::B1_LBO, G::B1_LBO, 128);
                umma_f16(g.tmem, da, db, IDESC, acc);
                acc = 1;
            }
        umma_commit(g.bar);
    }
    mbar_wait(g.bar, g.phase);
    g.phase ^= 1u;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}

// this thread's row of D, columns [64 line + 32 h, +32)
template <int NB>
__device__ __forceinline__ void ld_d(const Group<NB>& g, int line, int h, uint32_t* r) {
    TmemLd<32>::run(g.tmem + ((uint32_t)(g.q * 32) << 16) + (uint32_t)(line * 64 + h * 32), r);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// 16-byte chunk (8 consecutive n) of row kappa of the MN-major operand
template <int NB>
__device__ __forceinline__ uint4* b1_chunk(const Group<NB>& g, int kappa, int line, int nb) {
    return reinterpret_cast<uint4*>(g.bbuf + (kappa >> 3) * Group<NB>::B1_LBO + (line * 8 + nb) * 128 + (kappa & 7) * 16);
}
// 16-byte chunk (8 consecutive kappa, block kb) of column n of the K-major operand
template <int NB>
__device__ __forceinline__ uint4* b2_chunk(const Group<NB>& g, int n, int kb) {
    return reinterpret_cast<uint4*>(g.bbuf + (n >> 3) * Group<NB>::B2_SBO + kb * 128 + (n & 7) * 16);
}

__device__ __forceinline__ uint32_t pack_half2(float a, float b) {
    const __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<const uint32_t*>(&h);
}

// between the stages: D = Y (row (k1, c), column (line, i2)) -> Y' = Y W4096^(k1 i2) -> B of stage C.
// (Yr + i Yi)(C - i S): the c = 0 lane holds Yr and wants Yr C + Yi S, the c = 1 lane holds Yi and wants
// Yi C - Yr S; the partner value comes by SHFL from 16 lanes away.  The twiddles are NOT read from a
// table: the kernels are bound by the shared-memory / TMEM / shuffle data path (profiles/), the FMA pipe
// idles, so each thread steps (C, +-S)(k1, i2) along i2 by complex multiplication with its own
// w1 = e^{2 pi i k1/4096} (sign of S folded in), restarted every 16 points from w16^m: chains of 16
// fp32 products, error ~1e-6, far below the fp16 operand rounding.
struct Twid { float c1, s1, c16, s16; };
template <int NB>
__device__ __forceinline__ Twid make_twid(const Group<NB>& g) {
    const int k1 = 16 * g.q + g.j;
    Twid t;
    sincospif((float)k1 * (1.f / 2048.f), &t.s1, &t.c1);
    sincospif((float)((16 * k1) & 4095) * (1.f / 2048.f), &t.s16, &t.c16);
    if (g.c) { t.s1 = -t.s1; t.s16 = -t.s16; }
    return t;
}
template <int NB>
__device__ __forceinline__ void twiddle_step(const Group<NB>& g, const Twid& tw) {
    const int k1 = 16 * g.q + g.j;
#pragma unroll 1
    for (int line = 0; line < NB; ++line) {
        float bc = 1.f, bs = 0.f;                   // w16^m, m = i2 / 16
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            uint32_t r[32];
            ld_d(g, line, h, r);
            uint32_t pk[16];
#pragma unroll
            for (int m = 0; m < 2; ++m) {
                float tc = bc, ts = bs;
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const int i = 16 * m + e;
                    const float own = __uint_as_float(r[i]);
                    const float oth = __uint_as_float(__shfl_xor_sync(0xffffffffu, r[i], 16));
                    const float o = fmaf(oth, ts, own * tc);
                    if (e & 1) pk[i >> 1] = pack_half2(__uint_as_float(pk[i >> 1]), o);
                    else pk[i >> 1] = __float_as_uint(o);
                    const float nc = fmaf(-ts, tw.s1, tc * tw.c1), ns = fmaf(tc, tw.s1, ts * tw.c1);
                    tc = nc; ts = ns;
                }
                const float nc = fmaf(-bs, tw.s16, bc * tw.c16), ns = fmaf(bc, tw.s16, bs * tw.c16);
                bc = nc; bs = ns;
            }
            const int n = line * 64 + k1;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch)
                *b2_chunk(g, n, g.c * 8 + h * 4 + ch) = make_uint4(pk[4 * ch], pk[4 * ch + 1], pk[4 * ch + 2], pk[4 * ch + 3]);
        }
    }
}

// natural-order complex line (4096 half2, 16-byte aligned) -> B of stage A, in two steps so that the
// global loads of the next line fly while the current one is transformed.  A lane takes 8 consecutive
// points (32 bytes); lanes 0-7 take 8 consecutive i1 (consecutive 16-byte chunks of one block: no bank
// conflicts), the lane's upper bits walk the n blocks so that 4 lanes consume a whole 128-byte line.
struct LineRegs { uint4 v[8]; };
template <int NB>
__device__ __forceinline__ void fetch_line_c(const Group<NB>& g, const __half2* __restrict__ src, LineRegs& r) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int combo = g.q * 4 + u, i1 = 8 * (combo >> 1) + (g.lane & 7), nb = 4 * (combo & 1) + (g.lane >> 3);
        const uint4* p = reinterpret_cast<const uint4*>(src + 64 * i1 + 8 * nb);
        // one 32-byte load: a lane's two 16-byte halves share a sector
        asm volatile("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(r.v[2 * u].x), "=r"(r.v[2 * u].y), "=r"(r.v[2 * u].z), "=r"(r.v[2 * u].w), "=r"(r.v[2 * u + 1].x),
                       "=r"(r.v[2 * u + 1].y), "=r"(r.v[2 * u + 1].z), "=r"(r.v[2 * u + 1].w)
                     : "l"(p));
    }
}
// the same line held strip-major with strips of 4 points: point l at base[(l / 4) * strip_stride + l % 4]
// (the pass-1 array of the inverse 2D transform): a lane's 8 points are two 16-byte pieces
template <int NB>
__device__ __forceinline__ void fetch_line_strip4(const Group<NB>& g, const __half2* __restrict__ base, size_t strip_stride, LineRegs& r) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int combo = g.q * 4 + u, i1 = 8 * (combo >> 1) + (g.lane & 7), nb = 4 * (combo & 1) + (g.lane >> 3);
        const __half2* p = base + (size_t)((64 * i1 + 8 * nb) >> 2) * strip_stride;
        r.v[2 * u] = __ldg(reinterpret_cast<const uint4*>(p));
        r.v[2 * u + 1] = __ldg(reinterpret_cast<const uint4*>(p + strip_stride));
    }
}
template <int NB, bool SWAP>
__device__ __forceinline__ void put_line_c(const Group<NB>& g, int line, const LineRegs& r) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int combo = g.q * 4 + u, i1 = 8 * (combo >> 1) + (g.lane & 7), nb = 4 * (combo & 1) + (g.lane >> 3);
        const uint4 v0 = r.v[2 * u], v1 = r.v[2 * u + 1];
        const uint4 re = make_uint4(__byte_perm(v0.x, v0.y, 0x5410), __byte_perm(v0.z, v0.w, 0x5410), __byte_perm(v1.x, v1.y, 0x5410),
                                    __byte_perm(v1.z, v1.w, 0x5410));
        const uint4 im = make_uint4(__byte_perm(v0.x, v0.y, 0x7632), __byte_perm(v0.z, v0.w, 0x7632), __byte_perm(v1.x, v1.y, 0x7632),
                                    __byte_perm(v1.z, v1.w, 0x7632));
        *b1_chunk(g, (SWAP ? 64 : 0) + i1, line, nb) = re;
        *b1_chunk(g, (SWAP ? 0 : 64) + i1, line, nb) = im;
    }
}
template <int NB, bool SWAP>
__device__ __forceinline__ void load_line_c(const Group<NB>& g, int line, const __half2* __restrict__ src) {
    LineRegs r;
    fetch_line_c(g, src, r);
    put_line_c<NB, SWAP>(g, line, r);
}

// CTA prologue: tables into shared memory, one mbarrier and one TMEM accumulator per group.
// Shared memory: [A 32 KB][NG x B][NG mbarriers][TMEM slot]; 128 NG threads.
template <int NB, int NG>
struct Cta {
    static constexpr int offA = 0, offB = A_BYTES, offBar = offB + NG * Group<NB>::B_BYTES;
    static constexpr int offSlot = offBar + 8 * NG, total = offSlot + 4 * NG + 12;
    static constexpr int threads = 128 * NG;
    static_assert(NG * 64 * NB <= 512, "TMEM has 512 columns");
    static constexpr int tmem_cols = NG * 64 * NB <= 32 ? 32 : NG * 64 * NB <= 64 ? 64 : NG * 64 * NB <= 128 ? 128 : NG * 64 * NB <= 256 ? 256 : 512;

    static __device__ __forceinline__ Group<NB> setup(unsigned char* smem, const uint4* __restrict__ amat) {
        const int tid = threadIdx.x;
        for (int i = tid; i < A_BYTES / 16; i += threads) reinterpret_cast<uint4*>(smem + offA)[i] = __ldg(amat + i);
        Group<NB> g;
        const int grp = tid >> 7;
        g.t = tid & 127; g.q = g.t >> 5; g.lane = tid & 31; g.j = g.lane & 15; g.c = g.lane >> 4; g.barid = 1 + grp;
        g.bbuf = smem + offB + grp * Group<NB>::B_BYTES;
        g.a_addr = smem_u32(smem + offA);
        g.b_addr = smem_u32(g.bbuf);
        g.bar = reinterpret_cast<uint64_t*>(smem + offBar) + grp;
        g.phase = 0;
        uint32_t* slot = reinterpret_cast<uint32_t*>(smem + offSlot);       // one allocation per CTA, 64 NB columns per group
        if (g.t == 0) {
            mbar_init(g.bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;");
        }
        if (tid < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "n"(tmem_cols));
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // A was written through the generic proxy
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        g.tmem = *slot + (uint32_t)(grp * 64 * NB);
        return g;
    }
    static __device__ __forceinline__ void teardown(const Group<NB>& g) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (threadIdx.x < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(g.tmem), "n"(tmem_cols));
    }
};

// host: the DFT-64 matrix in the byte order the kernels copy into shared memory
inline void build_tables(std::vector<__half>& amat) {
    const double pi = 3.14159265358979323846264338327950288;
    amat.assign(128 * 128, __float2half(0.f));
    for (int rho = 0; rho < 128; ++rho)
        for (int kap = 0; kap < 128; ++kap) {
            const int q = rho >> 5, c = (rho >> 4) & 1, j = rho & 15, k = 16 * q + j, cp = kap >> 6, i = kap & 63;
            const double th = 2.0 * pi * (double)((k * i) & 63) / 64.0;
            const double v = (c == cp) ? cos(th) : (c == 0 ? sin(th) : -sin(th));
            amat[(size_t)(((rho >> 3) * 16 + (kap >> 3)) * 64 + (rho & 7) * 8 + (kap & 7))] = __float2half((float)v);
        }
}

}  // namespace tcfft
}  // namespace tcpk
