// fft.cuh -- batched shared-memory Stockham FFT for sm_100a (fp32 arithmetic).
//
// One transform of length N (power of two, 128..8192) is computed by a group of
// TG = N/16 threads; every thread keeps 16 complex values in registers per pass, so
// a pass is (N/16/R)... butterflies of radix R in {16, 8, 4, 2} per thread with
// NB*R = 16.  Passes exchange data through a padded shared-memory line (one pad
// element per 16, which makes the stride-16 writes of the first pass conflict free).
// The first pass reads through a caller-supplied loader and the last pass writes
// through a caller-supplied storer, so zero-padding, filtering, cropping, phase
// tables, deapodisation and dtype casts fuse into the transforms and the row never
// touches HBM in between.
//
// Autosort (Stockham) indexing: pass with radix R and Ns = product of earlier radices,
// butterfly b in [0, N/R):  inputs x[b + r N/R] * w^(r (b mod Ns)),  w = e^{-/+ 2 pi i/(Ns R)};
// outputs y[(b / Ns) Ns R + (b mod Ns) + r Ns].  Output is in natural order.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>

namespace tcpk {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// Two complex values that share every twiddle: two adjacent columns of the grid in the column pass
// of the 2D transform (one 8-byte global access, one 16-byte shared-memory access per element).
struct alignas(16) cpair { float2 a, b; };
__device__ __forceinline__ cpair cmul(cpair x, float2 w) { return cpair{cmul(x.a, w), cmul(x.b, w)}; }
__device__ __forceinline__ cpair cadd(cpair x, cpair y) { return cpair{cadd(x.a, y.a), cadd(x.b, y.b)}; }
__device__ __forceinline__ cpair csub(cpair x, cpair y) { return cpair{csub(x.a, y.a), csub(x.b, y.b)}; }

__host__ __device__ constexpr int pad_idx(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded_len(int N) { return N + (N >> 4); }

// multiply by -i (forward) or +i (inverse)
template <bool INV>
__device__ __forceinline__ float2 mul_mi(float2 a) {
    return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
template <bool INV>
__device__ __forceinline__ cpair mul_mi(cpair x) { return cpair{mul_mi<INV>(x.a), mul_mi<INV>(x.b)}; }
// multiply by e^{-/+ i phi} given (cos phi, sin phi)
template <bool INV>
__device__ __forceinline__ float2 mul_w(float2 a, float c, float s) {
    return INV ? make_float2(fmaf(-a.y, s, a.x * c), fmaf(a.x, s, a.y * c))
               : make_float2(fmaf(a.y, s, a.x * c), fmaf(-a.x, s, a.y * c));
}
template <bool INV>
__device__ __forceinline__ cpair mul_w(cpair x, float c, float s) { return cpair{mul_w<INV>(x.a, c, s), mul_w<INV>(x.b, c, s)}; }

template <bool INV, class T>
__device__ __forceinline__ void dft4(T& a0, T& a1, T& a2, T& a3) {
    T s02 = cadd(a0, a2), d02 = csub(a0, a2), s13 = cadd(a1, a3), d13 = csub(a1, a3);
    T jd = mul_mi<INV>(d13);
    a0 = cadd(s02, s13);
    a2 = csub(s02, s13);
    a1 = cadd(d02, jd);
    a3 = csub(d02, jd);
}

template <int R, bool INV>
struct Bfly;

template <bool INV>
struct Bfly<2, INV> {
    template <class T>
    static __device__ __forceinline__ void run(T* v) {
        T t = v[0];
        v[0] = cadd(t, v[1]);
        v[1] = csub(t, v[1]);
    }
};
template <bool INV>
struct Bfly<4, INV> {
    template <class T>
    static __device__ __forceinline__ void run(T* v) { dft4<INV>(v[0], v[1], v[2], v[3]); }
};
template <bool INV>
struct Bfly<8, INV> {
    template <class T>
    static __device__ __forceinline__ void run(T* v) {
        const float c = 0.70710678118654752440f;
        dft4<INV>(v[0], v[2], v[4], v[6]);   // E0..E3 in v0,v2,v4,v6
        dft4<INV>(v[1], v[3], v[5], v[7]);   // O0..O3 in v1,v3,v5,v7
        T o1 = mul_w<INV>(v[3], c, c);
        T o2 = mul_mi<INV>(v[5]);
        T o3 = mul_w<INV>(v[7], -c, c);
        T e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
        v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
        v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
        v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
        v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
    }
};
template <bool INV>
struct Bfly<16, INV> {
    template <class T>
    static __device__ __forceinline__ void run(T* v) {
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;  // cos, sin(pi/8)
        const float c2 = 0.70710678118654752440f;
        // step 1: for i0: A_i0[k1] = DFT4 over i1 of v[i0 + 4 i1]  (in place: v[i0 + 4 k1])
#pragma unroll
        for (int i0 = 0; i0 < 4; ++i0) dft4<INV>(v[i0], v[i0 + 4], v[i0 + 8], v[i0 + 12]);
        // step 2: twiddle A_i0[k1] *= w16^(i0 k1)
        v[5] = mul_w<INV>(v[5], c1, s1);      // i0=1,k1=1: t=1
        v[9] = mul_w<INV>(v[9], c2, c2);      // i0=1,k1=2: t=2
        v[13] = mul_w<INV>(v[13], s1, c1);    // i0=1,k1=3: t=3
        v[6] = mul_w<INV>(v[6], c2, c2);      // i0=2,k1=1: t=2
        v[10] = mul_mi<INV>(v[10]);           // i0=2,k1=2: t=4
        v[14] = mul_w<INV>(v[14], -c2, c2);   // i0=2,k1=3: t=6
        v[7] = mul_w<INV>(v[7], s1, c1);      // i0=3,k1=1: t=3
        v[11] = mul_w<INV>(v[11], -c2, c2);   // i0=3,k1=2: t=6
        v[15] = mul_w<INV>(v[15], -c1, -s1);  // i0=3,k1=3: t=9: cos(9pi/8)=-c1, sin(9pi/8)=-s1
        // step 3: for k1: X[k1 + 4 k0] = DFT4 over i0 of A_i0[k1] = v[i0 + 4 k1]
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) dft4<INV>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);
        // now v[4 k1 + k0] holds X[k1 + 4 k0]: transpose the 4x4 to natural order
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a + 1; b < 4; ++b) {
                T t = v[4 * a + b];
                v[4 * a + b] = v[4 * b + a];
                v[4 * b + a] = t;
            }
    }
};

// w^1 .. w^(R-1) by a shallow product tree (depth <= 4 keeps the rounding at a few ulp)
template <int R>
__device__ __forceinline__ void twiddle_powers(float2 w1, float2* w) {
    w[1] = w1;
    if (R > 2) { w[2] = cmul(w1, w1); w[3] = cmul(w[2], w1); }
    if (R > 4) { w[4] = cmul(w[2], w[2]); w[5] = cmul(w[4], w1); w[6] = cmul(w[4], w[2]); w[7] = cmul(w[4], w[3]); }
    if (R > 8) {
        w[8] = cmul(w[4], w[4]);
#pragma unroll
        for (int r = 9; r < 16; ++r) w[r] = cmul(w[8], w[r - 8]);
    }
}

// One Stockham pass of radix R over a length-N line held by TG = N/16 threads.
//   tw: table e^{-2 pi i t / N}, t in [0, N) (conjugated here for INV)
//   FIRST: inputs come from ld(index); else from s[pad_idx(index)]
//   LAST:  outputs go to st(index, value); else to s[pad_idx(index)]
// A loader / storer may take the thread's register slot (compile-time after unrolling) as an extra
// argument: the 16 outputs of a thread in the LAST pass of one transform and its 16 inputs in the FIRST
// pass of the next are the same elements when both passes are radix 16 over 16 N/16-strided points
// (tid + r N/16, slot r), so chained transforms can hand them over in registers instead of through
// shared memory.
template <class Load>
__device__ __forceinline__ auto call_ld(Load& ld, int i, int slot) {
    if constexpr (std::is_invocable_v<Load, int, int>) return ld(i, slot);
    else return ld(i);
}
template <class Store, class T>
__device__ __forceinline__ void call_st(Store& st, int i, T v, int slot) {
    if constexpr (std::is_invocable_v<Store, int, T, int>) st(i, v, slot);
    else st(i, v);
}

template <int N, int R, int NS, bool INV, bool FIRST, bool LAST, class T, class Load, class Store>
__device__ __forceinline__ void fft_pass(T* s, int tid, const float2* __restrict__ tw, Load ld, Store st) {
    constexpr int TG = N / 16;
    constexpr int NB = 16 / R;          // butterflies per thread
    T v[16];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = tid + q * TG;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = b + r * (N / R);
            if constexpr (FIRST) v[q * R + r] = call_ld(ld, i, q * R + r);
            else v[q * R + r] = s[pad_idx(i)];
        }
        if (NS > 1) {
            const int t = (b % NS) * (N / (NS * R));
            float2 w1 = __ldg(&tw[t]);
            if (INV) w1.y = -w1.y;
            float2 w[R];
            twiddle_powers<R>(w1, w);
#pragma unroll
            for (int r = 1; r < R; ++r) v[q * R + r] = cmul(v[q * R + r], w[r]);
        }
        Bfly<R, INV>::run(&v[q * R]);
    }
    __syncthreads();                    // everyone has read the line (a FIRST loader may read it too)
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = tid + q * TG;
        const int o = (b / NS) * (NS * R) + (b % NS);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if constexpr (LAST) call_st(st, o + r * NS, v[q * R + r], q * R + r);
            else s[pad_idx(o + r * NS)] = v[q * R + r];
        }
    }
    if (!LAST) __syncthreads();
}

// Register hand-over between chained transforms of length N: a thread's 16 outputs of the LAST pass
// (radix RL, 16 / RL butterflies b = tid + q N/16, outputs b + r N/RL, slot q RL + r) are the elements
// tid + (q + (16 / RL) r) N/16, i.e. exactly its 16 inputs of the next transform's FIRST pass (radix 16,
// input r' at tid + r' N/16, slot r') with r' = q + (16 / RL) r.
__host__ __device__ constexpr int fft_last_radix(int N) {
    return N == 128 ? 8 : N == 256 ? 16 : N == 8192 ? 2 : N / 256;      // plans below
}
template <int N>
__host__ __device__ constexpr int fft_chain_slot(int last_slot) {
    constexpr int RL = fft_last_radix(N);
    return last_slot / RL + (16 / RL) * (last_slot % RL);
}

// Full transform.  Radix plans: 128: 16,8 | 256: 16,16 | 512: 16,16,2 | 1024: 16,16,4 |
// 2048: 16,16,8 | 4096: 16,16,16 | 8192: 16,16,16,2.
// All threads of the CTA must call this together (it uses __syncthreads); `s` is the
// calling group's own padded line of padded_len(N) float2.
// NOTE: when the loader reads shared memory that the storer of a previous transform
// wrote, the caller must __syncthreads() between the two calls.
struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};

// `hook` runs once, right after the first pass (every thread of the group has consumed the loader's
// source by then: a caller may start refilling it).
template <int N, bool INV, class T, class Load, class Store, class Hook = NoHook>
__device__ __forceinline__ void fft_line(T* s, int tid, const float2* __restrict__ tw, Load ld, Store st, Hook hook = Hook()) {
    auto nold = [](int) { return T(); };
    auto nost = [](int, T) {};
    if constexpr (N == 128) {
        fft_pass<N, 16, 1, INV, true, false>(s, tid, tw, ld, nost);
        hook();
        fft_pass<N, 8, 16, INV, false, true>(s, tid, tw, nold, st);
    } else if constexpr (N == 256) {
        fft_pass<N, 16, 1, INV, true, false>(s, tid, tw, ld, nost);
        hook();
        fft_pass<N, 16, 16, INV, false, true>(s, tid, tw, nold, st);
    } else if constexpr (N == 8192) {
        fft_pass<N, 16, 1, INV, true, false>(s, tid, tw, ld, nost);
        hook();
        fft_pass<N, 16, 16, INV, false, false>(s, tid, tw, nold, nost);
        fft_pass<N, 16, 256, INV, false, false>(s, tid, tw, nold, nost);
        fft_pass<N, 2, 4096, INV, false, true>(s, tid, tw, nold, st);
    } else {
        constexpr int RL = N / 256;     // 2, 4, 8 or 16
        fft_pass<N, 16, 1, INV, true, false>(s, tid, tw, ld, nost);
        hook();
        fft_pass<N, 16, 16, INV, false, false>(s, tid, tw, nold, nost);
        fft_pass<N, RL, 256, INV, false, true>(s, tid, tw, nold, st);
    }
}

}  // namespace tcpk
