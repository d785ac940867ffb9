// mmafft.cuh -- length-4096 complex transforms whose radix-16 butterflies run on the tensor cores
// (warp-level mma.sync m16n8k16, fp16 operands, fp32 accumulators in registers), for fp16 storage.
//
// Why: the Stockham kernels of fft.cuh are bound by instruction issue (profiles/r1_kernels.md: 65-72 % issue
// active, 30 of 53 instructions per point are butterfly arithmetic) while the tensor pipe idles.  A radix-16
// butterfly over 8 positions is one real 32 x 32 by 32 x 8 product, i.e. four m16n8k16 MMAs per warp, and
// unlike tcgen05 (accumulators in TMEM, read back through the L1 data pipe: profiles/r1_tcfft.md) the result
// lands in the registers of the threads that twiddle and store it.  Measured rate of HMMA.16816.F32 on B200:
// one per 8.6 clk per SM sub-partition (profiles/r2_mma_rate.md), so 48 MMAs per 512 points cost 138 clk of
// tensor pipe against ~400 clk of issue for the same passes on the CUDA cores.
//
// Algorithm: in-place decimation in frequency, N = 16^3, slot s = d2 256 + d1 16 + d0:
//   pass 1: butterflies over d2 (stride 256), output (k2, beta = 16 d1 + d0) times W_4096^(k2 beta)
//   pass 2: butterflies over d1 (stride 16),  output (k1, d0) times W_256^(k1 d0)
//   pass 3: butterflies over d0 (stride 1),   output X[k0 256 + k1 16 + k2]: handed to the caller's epilogue
//           with its NATURAL index, so every transform reads and writes natural order and one set of
//           per-thread twiddles (20 complex registers) serves forward and inverse transforms alike.
// A transform is carried by a team of 256 threads = 8 warps.  NL lines that share the team (the two rows of an
// output row pair, the four columns of a grid strip) share its twiddles and sit INTERLEAVED in shared memory:
// element k of line l is word NL swz(k) + l of N NL half2 words, so one 4 NL-byte access moves element k of
// every line -- exactly the layout of the HBM arrays they come from (pass-1 row pairs, grid strips).  swz() is an
// XOR swizzle (no padding) that makes every access pattern below bank-conflict free.
//
// MMA mapping (PTX m16n8k16 fragments; g = lane / 4, c = lane % 4).  One MMA group = 8 butterflies:
//   B (K 32 x N 8): column n = butterfly g of the group; K index 2 q' + (0 re | 1 im) of input q';
//                   a thread holds q' in {c, c + 4, 8 + c, 12 + c} as 4 packed half2 registers.
//   A (M 32 x K 32): real form of W_16^(o j) times GAMMA, two 16-row tiles t; tile row g = re and g + 8 = im
//                   of output o = outmap(t, g); 16 registers per thread, from a table built in fp64.
//   D: a thread holds outputs outmap(0, g), outmap(1, g) of butterflies 2c and 2c + 1 (fp32).
// Inverse transforms use the same fragments with sign bits flipped (R_inv = D R D, D = diag(+re, -im)) and
// conjugated twiddles.  Zero-padded inputs skip the second K step, cropped outputs the second tile.
// Every pass works on batches of 4 / NL groups: all loads of a batch, then its 16 (8 independent chains of 2)
// MMAs, then twiddles, packing and stores, which gives the tensor pipe and the load pipe independent work.
//
// Accuracy: operands are rounded to fp16 once per pass (relative 2^-11, the rounding the fp16 path already
// applies at every HBM boundary); GAMMA = 1.86033... is chosen so that GAMMA x {1, cos pi/8, sin pi/8,
// cos pi/4} are all within 1.7e-5 of an fp16 number (3.0e-4 without it), which keeps the systematic error
// of the butterfly matrix below the data rounding; the factors 1/GAMMA ride in the twiddles (gain 1 overall).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcpk {
namespace mf {

constexpr int N = 4096;
constexpr int NT = 256;                                   // threads of a team
constexpr double GAMMA = 1.8603300443229513;
enum { AV_NAT = 0, AV_LO = 1, AV_LOC = 2, AV_COUNT = 3 };  // fragment tables: passes 1-2 | pass 3 | pass 3, centre crop
constexpr int ATAB_WORDS = AV_COUNT * 32 * 16;

// Bank swizzle of element index k for NL interleaved lines (a wavefront = 128 bytes = 32 / NL elements of 4 NL bytes).
// The digit that varies across the lanes of one access (d2 in passes 1 and 3, d1 in pass 2) is XORed into the low
// bits so that the 32 / NL lanes of a wavefront fall into distinct banks for every pattern of this file; derivation
// in DESIGN.md section 6.
template <int NL>
__host__ __device__ constexpr int swz(int k) {
    if (NL == 1) return k ^ (((k >> 8) & 3) << 3) ^ (((k >> 5) & 1) << 3);
    if (NL == 2) return k ^ (((k >> 8) & 1) ? 12 : 0) ^ (((k >> 9) & 1) ? 5 : 0) ^ (((k >> 4) & 1) ? 12 : 0) ^ (((k >> 5) & 1) ? 5 : 0);
    return k ^ ((((k >> 8) & 3) << 1) | ((k >> 8) & 1)) ^ ((((k >> 4) & 3) << 1) | ((k >> 4) & 1));
}

template <int NL> struct Vec;
template <> struct Vec<1> { using T = uint32_t; };
template <> struct Vec<2> { using T = uint2; };
template <> struct Vec<4> { using T = uint4; };
__device__ __forceinline__ uint32_t vget(uint32_t v, int) { return v; }
__device__ __forceinline__ uint32_t vget(const uint2& v, int l) { return l ? v.y : v.x; }
__device__ __forceinline__ uint32_t vget(const uint4& v, int l) { return l == 0 ? v.x : l == 1 ? v.y : l == 2 ? v.z : v.w; }
__device__ __forceinline__ void vmake(uint32_t& v, const uint32_t* w) { v = w[0]; }
__device__ __forceinline__ void vmake(uint2& v, const uint32_t* w) { v = make_uint2(w[0], w[1]); }
__device__ __forceinline__ void vmake(uint4& v, const uint32_t* w) { v = make_uint4(w[0], w[1], w[2], w[3]); }
// element k of all NL lines
template <int NL>
__device__ __forceinline__ typename Vec<NL>::T* elem(uint32_t* L, int k) { return reinterpret_cast<typename Vec<NL>::T*>(L + NL * swz<NL>(k)); }

struct AFrag { uint32_t a[2][2][4]; };                    // [tile][K step][register]
// Twiddles of a thread.  Pass 2 needs four (registers).  Pass 1 needs sixteen, W^(d2 beta) with beta = 8 warp + 64 group
// + 2c + e: the four of group 0 sit in a small shared-memory table base[2 tile + e][thread] and the others follow by the
// recurrence W^(d2 (beta + 64)) = W^(d2 beta) W_64^(d2), whose two factors step[tile] are registers.
typedef unsigned long long f32x2_t;
struct Tw2s { f32x2_t r, i; };
struct Twid {
    const float2* base;                                   // this thread's column: base[(2 t + e) * NT]
    float2 step[2];
    Tw2s t2[2];                                           // pass 2: [tile], butterflies 2c and 2c + 1 packed (real parts, imaginary parts)
};
constexpr int T1_BYTES = 4 * NT * 8;

// Byte offsets of the thread's accesses into the lines (element k of NL lines at byte 4 NL swz(k)).  In every pattern the
// bits the swizzle reads and flips come from the thread's own indices, never from the group, tile or input counters, so
// an access is one of these offsets plus a compile-time immediate.
template <int NL>
struct Offs {
    uint32_t r1, w1[2], r2, w2[2], r3[4];
};
template <int NL>
__device__ __forceinline__ void make_offs(Offs<NL>& o, int warp, int g, int c) {
    o.r1 = 4 * NL * swz<NL>(256 * c + 8 * warp + g);                           // + 4 NL (1024 i + 64 grp)
    const int b2 = 256 * (warp >> 1) + 8 * (warp & 1);
    o.r2 = 4 * NL * swz<NL>(b2 + 16 * c + g);                                  // + 4 NL (1024 grp + 64 i)
    const int b3 = 256 * (8 * (warp & 1) + g) + 16 * (warp >> 1) + 2 * c;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        o.w1[e] = 4 * NL * swz<NL>(256 * g + 8 * warp + 2 * c + e);            // + 4 NL (2048 t + 64 grp)
        o.w2[e] = 4 * NL * swz<NL>(b2 + 16 * g + 2 * c + e);                   // + 4 NL (1024 grp + 128 t)
        o.r3[e] = 4 * NL * swz<NL>(b3 + e);                                    // + 4 NL 64 grp
        o.r3[2 + e] = 4 * NL * swz<NL>(b3 + 8 + e);
    }
}

__device__ __forceinline__ void load_afrag(AFrag& f, const uint32_t* __restrict__ atab, int variant, int lane) {
    const uint4* p = reinterpret_cast<const uint4*>(atab + ((size_t)variant * 32 + lane) * 16);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const uint4 v = __ldg(p + q);
        f.a[q >> 1][q & 1][0] = v.x; f.a[q >> 1][q & 1][1] = v.y; f.a[q >> 1][q & 1][2] = v.z; f.a[q >> 1][q & 1][3] = v.w;
    }
}
// forward <-> inverse: registers 0, 2 hold re rows (flip the im column = high half), 1, 3 im rows (flip the re column)
__device__ __forceinline__ void flip_afrag(AFrag& f) {
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            f.a[t][s][0] ^= 0x80000000u; f.a[t][s][2] ^= 0x80000000u;
            f.a[t][s][1] ^= 0x00008000u; f.a[t][s][3] ^= 0x00008000u;
        }
}

// twiddles of the calling thread (tw = e^{-2 pi i t / 4096}); the butterfly matrices carry GAMMA each, so with
// s1 = 1/GAMMA and s2 = 1/GAMMA^2 a whole transform has gain 1
__device__ __forceinline__ void load_twid(Twid& T, float2* t1tab, const float2* __restrict__ tw, int warp, int g, int c, float s1, float s2) {
    float2* mine = t1tab + (warp * 32 + g * 4 + c);
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int d2 = g + 8 * t;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const float2 w = __ldg(&tw[(d2 * (8 * warp + 2 * c + e)) & (N - 1)]);
            mine[(2 * t + e) * NT] = make_float2(w.x * s1, w.y * s1);
        }
        const float2 v0 = __ldg(&tw[(16 * d2 * (8 * (warp & 1) + 2 * c)) & (N - 1)]);
        const float2 v1 = __ldg(&tw[(16 * d2 * (8 * (warp & 1) + 2 * c + 1)) & (N - 1)]);
        asm("mov.b64 %0, {%1, %2};" : "=l"(T.t2[t].r) : "f"(v0.x * s2), "f"(v1.x * s2));
        asm("mov.b64 %0, {%1, %2};" : "=l"(T.t2[t].i) : "f"(v0.y * s2), "f"(v1.y * s2));
        T.step[t] = __ldg(&tw[(64 * d2) & (N - 1)]);
    }
    T.base = mine;
}

__device__ __forceinline__ void mma_z(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ void mma_a(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// (re, im) fp32 -> half2 with saturation
__device__ __forceinline__ uint32_t pack_h2(float re, float im) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(im), "f"(re));
    return r;
}
// Packed fp32 pairs (sm_100 FMUL2 / FFMA2: two fp32 operations per issued instruction).  The accumulator of an MMA holds
// {re, re', im, im'} of two adjacent butterflies, so a pair of complex twiddle products is 2 FMUL2 + 2 FFMA2.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpk2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 neg2(f32x2 a) { return a ^ 0x8000000080000000ull; }
// twiddles of two adjacent butterflies: real parts, imaginary parts
struct Tw2 { f32x2 r, i; };
// acc = {re0, re1, im0, im1} times the twiddle pair (or its conjugate), packed to two half2 (re, im) words
template <bool INV>
__device__ __forceinline__ void twmul2(const float (&acc)[4], const Tw2& w, uint32_t& h0, uint32_t& h1) {
    const f32x2 re = pk2(acc[0], acc[1]), im = pk2(acc[2], acc[3]);
    const f32x2 yr = fma2(im, INV ? w.i : neg2(w.i), mul2(re, w.r));      // re wr -/+ im wi
    const f32x2 yi = fma2(re, INV ? neg2(w.i) : w.i, mul2(im, w.r));      // im wr +/- re wi
    float r0, r1, i0, i1;
    unpk2(yr, r0, r1);
    unpk2(yi, i0, i1);
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(h0) : "f"(i0), "f"(r0));
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(h1) : "f"(i1), "f"(r1));
}

template <bool INV>
__device__ __forceinline__ float2 twmul(float re, float im, float2 w) {       // (re + i im) w, or times conj(w)
    return INV ? make_float2(fmaf(im, w.y, re * w.x), fmaf(-re, w.y, im * w.x))
               : make_float2(fmaf(-im, w.y, re * w.x), fmaf(re, w.y, im * w.x));
}

// One butterfly group: b = the thread's 4 inputs; acc[t] = {re(2c), re(2c+1), im(2c), im(2c+1)} of output outmap(t, g)
template <bool KPRUNE, bool MPRUNE>
__device__ __forceinline__ void bfly(float (&acc)[2][4], const AFrag& A, uint32_t b0, uint32_t b1, uint32_t b2, uint32_t b3) {
#pragma unroll
    for (int t = 0; t < (MPRUNE ? 1 : 2); ++t) mma_z(acc[t], A.a[t][0], b0, b1);
    if (!KPRUNE) {
#pragma unroll
        for (int t = 0; t < (MPRUNE ? 1 : 2); ++t) mma_a(acc[t], A.a[t][1], b2, b3);
    }
}

constexpr int groups_per_batch(int NL) { return 4 / NL; }

template <int NL>
__device__ __forceinline__ typename Vec<NL>::T& at(uint32_t* L, uint32_t byte_off) {
    return *reinterpret_cast<typename Vec<NL>::T*>(reinterpret_cast<unsigned char*>(L) + byte_off);
}
// store the packed outputs at natural indices k0 (even) and k0 + 1 of all lines; o[e] = byte offset of k0 + e
template <int NL>
__device__ __forceinline__ void put2(uint32_t* L, const uint32_t (&o)[2], uint32_t imm, const uint32_t (&w0)[NL], const uint32_t (&w1)[NL]) {
    if constexpr (NL == 1) {
        at<2>(L, o[0] + imm) = make_uint2(w0[0], w1[0]);          // one line: k0 and k0 + 1 are adjacent words
    } else {
        vmake(at<NL>(L, o[0] + imm), w0);
        vmake(at<NL>(L, o[1] + imm), w1);
    }
}

// pass 1 (stride 256).  SRC_LINES: the inputs are in the lines (in place); otherwise in(k) returns the Vec<NL> at natural
// index k from somewhere else (a staging buffer, global memory).  Outputs go to the lines.
template <int NL, bool INV, bool KPRUNE, bool SRC_LINES, class In>
__device__ __forceinline__ void pass1(uint32_t* L, const AFrag& A, const Twid& T, const Offs<NL>& O, int warp, int g, int c, In in) {
    using V = typename Vec<NL>::T;
    constexpr int GB = groups_per_batch(NL), NB = 4 / GB, NI = KPRUNE ? 2 : 4;
    Tw2 cur[2];
    f32x2 sx[2], sy[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const float2 a = T.base[(2 * t) * NT], b = T.base[(2 * t + 1) * NT];
        cur[t].r = pk2(a.x, b.x);
        cur[t].i = pk2(a.y, b.y);
        sx[t] = pk2(T.step[t].x, T.step[t].x);
        sy[t] = pk2(T.step[t].y, T.step[t].y);
    }
#pragma unroll
    for (int bt = 0; bt < NB; ++bt) {
        V v[GB][4];
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                if constexpr (SRC_LINES) v[q][i] = at<NL>(L, O.r1 + 4 * NL * (1024 * i + 64 * (bt * GB + q)));
                else v[q][i] = in((c + 4 * i) * 256 + 8 * warp + 64 * (bt * GB + q) + g);
            }
        float acc[GB][NL][2][4];
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int l = 0; l < NL; ++l)
                bfly<KPRUNE, false>(acc[q][l], A, vget(v[q][0], l), vget(v[q][1], l), KPRUNE ? 0u : vget(v[q][2], l), KPRUNE ? 0u : vget(v[q][3], l));
#pragma unroll
        for (int q = 0; q < GB; ++q) {
            const int grp = bt * GB + q;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                uint32_t w0[NL], w1[NL];
#pragma unroll
                for (int l = 0; l < NL; ++l) twmul2<INV>(acc[q][l][t], cur[t], w0[l], w1[l]);
                put2<NL>(L, O.w1, 4 * NL * (2048 * t + 64 * grp), w0, w1);
                if (grp < 3) {          // next group: beta + 64, i.e. times step = sx + i sy
                    const f32x2 nr = fma2(cur[t].i, neg2(sy[t]), mul2(cur[t].r, sx[t]));
                    cur[t].i = fma2(cur[t].r, sy[t], mul2(cur[t].i, sx[t]));
                    cur[t].r = nr;
                }
            }
        }
    }
}

// pass 2 (stride 16), in place
template <int NL, bool INV>
__device__ __forceinline__ void pass2(uint32_t* L, const AFrag& A, const Twid& T, const Offs<NL>& O) {
    using V = typename Vec<NL>::T;
    constexpr int GB = groups_per_batch(NL), NB = 4 / GB;
#pragma unroll
    for (int bt = 0; bt < NB; ++bt) {
        V v[GB][4];
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int i = 0; i < 4; ++i) v[q][i] = at<NL>(L, O.r2 + 4 * NL * (1024 * (bt * GB + q) + 64 * i));
        float acc[GB][NL][2][4];
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int l = 0; l < NL; ++l) bfly<false, false>(acc[q][l], A, vget(v[q][0], l), vget(v[q][1], l), vget(v[q][2], l), vget(v[q][3], l));
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                uint32_t w0[NL], w1[NL];
#pragma unroll
                for (int l = 0; l < NL; ++l) twmul2<INV>(acc[q][l][t], Tw2{T.t2[t].r, T.t2[t].i}, w0[l], w1[l]);
                put2<NL>(L, O.w2, 4 * NL * (1024 * (bt * GB + q) + 128 * t), w0, w1);
            }
    }
}

// pass 3 (stride 1): the thread's inputs of group grp: digits (2c, 2c + 1) and (8 + 2c, 9 + 2c) of butterfly d2 = 8 h + g
template <int NL>
__device__ __forceinline__ void pass3_load(uint32_t* L, const Offs<NL>& O, int grp, typename Vec<NL>::T (&v)[4]) {
    if constexpr (NL == 1) {
        const uint2 lo = at<2>(L, O.r3[0] + 4 * 64 * grp), hi = at<2>(L, O.r3[2] + 4 * 64 * grp);
        v[0] = lo.x; v[1] = lo.y; v[2] = hi.x; v[3] = hi.y;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = at<NL>(L, O.r3[j] + 4 * NL * 64 * grp);
    }
}
// natural index of the thread's first output (butterfly 2c) of tile t: o 256 + d1 16 + 8 h + 2c; the second is + 1.
// CENTRE: tile 0 holds o in {0..3, 12..15} (the central half of the FFT-ordered axis), there is no tile 1.
template <bool CENTRE>
__device__ __forceinline__ int pass3_index(int t, int grp, int warp, int g, int c) {
    const int o = CENTRE ? (g < 4 ? g : g + 8) : g + 8 * t;
    return o * 256 + ((warp >> 1) + 4 * grp) * 16 + 8 * (warp & 1) + 2 * c;
}
// pass 3 with the outputs handed to the caller in natural order, two adjacent indices k0 (even), k0 + 1 at a time:
// epi(k0, y0[NL], y1[NL]) gets the NL lines of the team together.  TO_LINES (one line): the epilogue writes the line
// itself, so every input of the team is loaded before a block barrier and only then transformed.
template <int NL, bool MPRUNE, bool CENTRE, bool TO_LINES, class Epi>
__device__ __forceinline__ void pass3(uint32_t* L, const AFrag& A, const Offs<NL>& O, int warp, int g, int c, Epi epi) {
    using V = typename Vec<NL>::T;
    constexpr int GB = groups_per_batch(NL), NB = 4 / GB, NTILE = MPRUNE ? 1 : 2;
    static_assert(!TO_LINES || NL == 1, "line-to-line pass 3 is used by the row kernel only");
    const int kbase = pass3_index<CENTRE>(0, 0, warp, g, c);
#pragma unroll
    for (int bt = 0; bt < NB; ++bt) {
        V v[GB][4];
#pragma unroll
        for (int q = 0; q < GB; ++q) pass3_load<NL>(L, O, bt * GB + q, v[q]);
        if constexpr (TO_LINES) __syncthreads();          // NB == 1: all inputs of the team are in registers
        float acc[GB][NL][2][4];
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int l = 0; l < NL; ++l) bfly<false, MPRUNE>(acc[q][l], A, vget(v[q][0], l), vget(v[q][1], l), vget(v[q][2], l), vget(v[q][3], l));
#pragma unroll
        for (int q = 0; q < GB; ++q)
#pragma unroll
            for (int t = 0; t < NTILE; ++t) {
                float2 y0[NL], y1[NL];
#pragma unroll
                for (int l = 0; l < NL; ++l) {
                    y0[l] = make_float2(acc[q][l][t][0], acc[q][l][t][2]);
                    y1[l] = make_float2(acc[q][l][t][1], acc[q][l][t][3]);
                }
                epi(kbase + 2048 * t + 64 * (bt * GB + q), y0, y1);
            }
    }
}

}  // namespace mf
}  // namespace tcpk
