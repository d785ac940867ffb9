// k_grid_mma.cu -- S5 for fp16 storage: tile-owned gridding as a block-sparse contraction on the
// 5th-generation tensor cores (tcgen05, accumulators in TMEM).
//
//   F[cell][n] = sum_samples W[cell][sample] * G[sample][n],   n = (slice pair, re|im),
//   W[cell][sample] = phi(l1 - nu1) phi(l2 - nu2) inside the open box |l - nu| < m, else 0
//   (reading Q7).
//
// The weight W does not depend on the slice, and per-cell FMA gridding is bound by instruction
// issue, not by HBM (profiles/r1b: 1.18 G warp instructions per 16-slice chunk).  Here the CUDA cores
// only GENERATE W -- once per (sub-tile, sample), for all slices of the chunk -- and the multiply-
// accumulate over up to 32 slice pairs runs as dense 128 x N x 16 MMAs, which is a measured win
// (profiles/r1c) although only ~12 % of W is non-zero.
//
// Work decomposition (shared with k_grid_tile.cu): an item is a 32 x 32 region of cells (or a
// projection sub-range of a near-DC region); its chords -- runs of consecutive k of the rays that
// cross it -- are staged in shared memory in batches: the NN/2 spectra values of every sample,
// interleaved (one B-operand row), and the sample's first tap and tap distance, decided in fp64.
// The region is 8 sub-tiles of 16 x 8 cells = the M = 128 rows of one accumulator each
// (8 x NN TMEM columns).  Per batch, the samples that can touch a sub-tile are listed (a chord crosses
// a sub-tile box in one run), the lists are laid end to end in 16-column segments, and for every
// 64 columns: phase 1 writes the separable 1D weights (6 + 6 taps) and copies the B rows, phase 2
// forms the outer products into the MN-major A stage, and one thread issues the MMAs; two stages
// are ring-buffered on mbarriers signalled by tcgen05.commit.  Deterministic: fixed order, no atomics.
#include <math.h>

#include "grid_common.cuh"
#include "tcp_internal.h"

namespace tcpk {

constexpr int SUBX = 16, SUBY = 8, NSUB = 8;      // sub-tile = 128 cells; 2 x 4 sub-tiles per region
constexpr int MPB = 12;                           // chords per batch
constexpr int KC = 64;                            // columns (samples) per A/B stage
constexpr int NST = 2;                            // stages
constexpr int RUNMAX = 32;                        // >= samples of one chord inside a sub-tile's sample box
constexpr int COLMAX = NSUB * MPB * RUNMAX;       // flat column list capacity (segments are 16-aligned)
constexpr int A_LBO = (128 / 8) * 128;            // bytes between k-blocks of 8 columns in an A stage

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, no swizzle: start >> 4, leading (k-block) and stride (mn-block) byte offsets >> 4
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    uint32_t done = 0;
    while (!done)
        asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p;}"
                     : "=r"(done)
                     : "r"(smem_u32(b)), "r"(parity)
                     : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* b) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{.reg .pred p; setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;}" ::"r"(tmem_d),
                 "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
                 : "memory");
}

template <int NN> struct TmemLd;
template <> struct TmemLd<16> {
    static __device__ __forceinline__ void run(uint32_t taddr, uint32_t* r) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                       "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                     : "r"(taddr));
    }
};
template <> struct TmemLd<32> {
    static __device__ __forceinline__ void run(uint32_t taddr, uint32_t* r) {
        TmemLd<16>::run(taddr, r);
        TmemLd<16>::run(taddr + 16, r + 16);
    }
};

// bytes of dynamic shared memory, and the carve-up (all offsets multiples of 128)
template <int MH, int NN>
struct MmaSmem {
    static constexpr int KL = chord_len(MH);
    static constexpr int NSLOT = MPB * KL;
    static constexpr int GW = NN * 2 / 16;                   // uint4 per sample (B row)
    static constexpr int B_LBO = (NN / 8) * 128;
    static constexpr int offA = 0;                           // [NST][KC/8][16][8][8] half
    static constexpr int offB = offA + NST * KC * 256;       // [NST][KC/8][NN/8][8][8] half
    static constexpr int offMeta = offB + NST * KC * NN * 2; // [NSLOT] float4
    static constexpr int offG = offMeta + NSLOT * 16;        // [NSLOT][GW] uint4
    static constexpr int offWx = offG + NSLOT * GW * 16;     // [2][KC] uint4 (lx 0..7 | 8..15)
    static constexpr int offWy = offWx + 2 * KC * 16;        // [KC] uint4 (ly 0..7)
    static constexpr int offCol = offWy + KC * 16;           // [COLMAX] uint16
    static constexpr int offRec = offCol + COLMAX * 2;       // [MPB] ChordRec
    static constexpr int offRecj = offRec + MPB * 16;        // [MPB] int
    static constexpr int offHits = offRecj + 64;             // [NTHR] int2
    static constexpr int offRun = offHits + NTHR * 8;        // [NSUB][MPB] int (start | len << 16), then pre[NSUB][MPB] int
    static constexpr int offMisc = offRun + 2 * NSUB * MPB * 4;   // wcount[9], seg[9], flags
    static constexpr int offBar = offMisc + 128;             // mbarriers: free[NST], done
    static constexpr int total = offBar + 64;
};

// ---------------------------------------------------------------------------------------
// item: x = region (32 x 32 tile) index, y = split s | nsplit S << 16, z = first partial slot (-1: write the grid)
template <int MH, int NN>
__global__ void __launch_bounds__(NTHR, 2)
    grid_mma_kernel(const __half2* __restrict__ spec, __half2* __restrict__ grid, float2* __restrict__ partial,
                    const double2* __restrict__ trig, const int2* __restrict__ plan, const int4* __restrict__ items,
                    int nproj, int M, int npair, float alpha2) {
    using L = MmaSmem<MH, NN>;
    constexpr int KL = L::KL, GW = L::GW, NPG = NN / 2;
    extern __shared__ __align__(128) unsigned char smem[];
    float4* meta = reinterpret_cast<float4*>(smem + L::offMeta);
    uint4* gs = reinterpret_cast<uint4*>(smem + L::offG);
    uint4* wxs = reinterpret_cast<uint4*>(smem + L::offWx);
    uint4* wys = reinterpret_cast<uint4*>(smem + L::offWy);
    unsigned short* colslot = reinterpret_cast<unsigned short*>(smem + L::offCol);
    ChordRec* rec = reinterpret_cast<ChordRec*>(smem + L::offRec);
    int* recj = reinterpret_cast<int*>(smem + L::offRecj);
    int2* hits = reinterpret_cast<int2*>(smem + L::offHits);
    int* run = reinterpret_cast<int*>(smem + L::offRun);             // [NSUB][MPB] start | len << 16
    int* pre = run + NSUB * MPB;                                      // [NSUB][MPB] offset inside the segment
    int* wcount = reinterpret_cast<int*>(smem + L::offMisc);          // [9]
    int* seg = wcount + 9;                                            // [9] segment starts (columns), seg[8] = total
    uint32_t* shared_u32 = reinterpret_cast<uint32_t*>(seg + 9);      // [0] tmem base, [1] started mask
    uint64_t* bar_free = reinterpret_cast<uint64_t*>(smem + L::offBar);
    uint64_t* bar_done = bar_free + NST;

    const int n = M >> 1, tiles = M / TS;
    const int4 item = items[blockIdx.x];
    const int tile = item.x, split = item.y & 0xffff, nsplit = item.y >> 16;
    const int pg = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TX0 = (tile % tiles) * TS, TY0 = (tile / tiles) * TS;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) mbar_init(&bar_free[s], 1);
        mbar_init(bar_done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
        shared_u32[1] = 0;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&shared_u32[0])), "n"(NSUB * NN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = shared_u32[0];
    // instruction descriptor: D fp32, A/B fp16, both MN-major, N = NN, M = 128
    constexpr uint32_t IDESC = (1u << 4) | (1u << 15) | (1u << 16) | ((uint32_t)(NN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    uint32_t started = 0;          // thread 0: sub-tiles whose accumulator has been written
    uint32_t nfill = 0;            // stage fills so far (uniform)

    for (int img = 0; img < 4; ++img) {
        const int2 win = plan[tile * 4 + img];
        if (win.y == 0) continue;
        int X0 = (TX0 >= n) ? TX0 - M : TX0, Y0 = (TY0 >= n) ? TY0 - M : TY0;
        if (img & 1) X0 += (X0 == -n) ? M : -M;
        if (img & 2) Y0 += (Y0 == -n) ? M : -M;
        const float hw = (float)MH + 0.02f;
        const float bax = (float)X0 - hw, bbx = (float)(X0 + TS - 1) + hw;
        const float bay = (float)Y0 - hw, bby = (float)(Y0 + TS - 1) + hw;
        const int i_lo = (int)(((long long)win.y * split) / nsplit), i_hi = (int)(((long long)win.y * (split + 1)) / nsplit);

        for (int i0 = i_lo; i0 < i_hi; i0 += NTHR) {
            // ---- test 256 projections of the window, compact the hits in order
            const int i = i0 + tid;
            bool hit = false;
            int j = 0, kmin = 0, kmax = -1;
            if (i < i_hi) {
                j = win.x + i;
                if (j >= nproj) j -= nproj;
                const double2 cs = trig[j];
                hit = chord_range((float)cs.x, (float)cs.y, bax, bbx, bay, bby, (float)(n - 1), kmin, kmax);
            }
            const unsigned bal = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) wcount[warp] = __popc(bal);
            __syncthreads();
            int before = 0, nhit = 0;
#pragma unroll
            for (int w = 0; w < NTHR / 32; ++w) {
                const int cw = wcount[w];
                if (w < warp) before += cw;
                nhit += cw;
            }
            if (hit) {
                int cnt = kmax - kmin + 1;
                if (cnt > KL) cnt = KL;
                hits[before + __popc(bal & ((1u << lane) - 1u))] = make_int2(j, (kmin & 0xffff) | (cnt << 16));
            }
            __syncthreads();

            for (int b0 = 0; b0 < nhit; b0 += MPB) {
                const int nb = min(MPB, nhit - b0);
                if (tid < nb) {
                    const int2 h = hits[b0 + tid];
                    const double2 cs = trig[h.x];
                    ChordRec r;
                    r.c = (float)cs.x;
                    r.s = (float)cs.y;
                    r.inv = 0.f;
                    r.pack = h.y;
                    rec[tid] = r;
                    recj[tid] = h.x;
                }
                __syncthreads();
                // ---- stage the chords: one B row (NN halves) + the first tap and its distance per sample
                for (int idx = tid; idx < nb * KL; idx += NTHR) {
                    const int r = idx / KL, kl = idx - r * KL;
                    const int pk = rec[r].pack;
                    if (kl >= ((pk >> 16) & 0xff)) continue;
                    const int k = (int)(short)(pk & 0xffff) + kl;
                    const int jj = recj[r];
                    const double2 cs = trig[jj];
                    const double nu1 = (double)k * cs.x, nu2 = (double)k * cs.y;
                    // taps l = floor(nu) - m + 1 + t, t = 0..2m-1, distance d_t = l - nu; the open box
                    // |l - nu| < m keeps t iff d_t < m (d_0 > -m always).  d_0 is rounded to fp32 so that
                    // this test still decides as in fp64: exactly -m+1 only when nu is an integer.
                    const double f1 = floor(nu1) - (double)(MH - 1), f2 = floor(nu2) - (double)(MH - 1);
                    float d1 = (float)(f1 - nu1), d2 = (float)(f2 - nu2);
                    const float dint = -(float)(MH - 1);
                    if (d1 >= dint && (f1 - nu1) < (double)dint) d1 = __uint_as_float(__float_as_uint(dint) + 1u);   // next below
                    if (d2 >= dint && (f2 - nu2) < (double)dint) d2 = __uint_as_float(__float_as_uint(dint) + 1u);
                    meta[idx] = make_float4((float)(f1 - (double)X0), d1, (float)(f2 - (double)Y0), d2);
                    alignas(16) __half2 v[NPG];
#pragma unroll
                    for (int p = 0; p < NPG; ++p) {
                        const int pair = pg * NPG + p;
                        v[p] = (pair < npair) ? spec[((size_t)pair * nproj + jj) * M + (size_t)(k & (M - 1))] : czero<__half2>();
                    }
                    const uint4* vv = reinterpret_cast<const uint4*>(v);
#pragma unroll
                    for (int q = 0; q < GW; ++q) gs[(size_t)idx * GW + q] = vv[q];
                }
                __syncthreads();
                // ---- runs: chord r inside the sample box of sub-tile b = consecutive staged slots
                if (tid < nb * NSUB) {
                    const int r = tid / NSUB, b = tid - r * NSUB;
                    const ChordRec R = rec[r];
                    const int rk0 = (int)(short)(R.pack & 0xffff), rcnt = (R.pack >> 16) & 0xff;
                    const float sx = (float)(X0 + (b & 1) * SUBX), sy = (float)(Y0 + (b >> 1) * SUBY);
                    int k0, k1, len = 0, start = 0;
                    if (chord_range(R.c, R.s, sx - hw, sx + (float)(SUBX - 1) + hw, sy - hw, sy + (float)(SUBY - 1) + hw,
                                    (float)(n - 1), k0, k1)) {
                        k0 = max(k0, rk0);
                        k1 = min(k1, rk0 + rcnt - 1);
                        len = min(max(k1 - k0 + 1, 0), RUNMAX);
                        start = r * KL + (k0 - rk0);
                    }
                    run[b * MPB + r] = start | (len << 16);
                }
                __syncthreads();
                if (tid < NSUB) {                     // per sub-tile: offsets of its runs, total length
                    int off = 0;
                    for (int r = 0; r < nb; ++r) {
                        pre[tid * MPB + r] = off;
                        off += run[tid * MPB + r] >> 16;
                    }
                    wcount[tid] = off;
                }
                __syncthreads();
                {
                    int s0 = 0;
#pragma unroll
                    for (int b = 0; b < NSUB; ++b) {
                        if (tid == 0) seg[b] = s0;
                        const int len = wcount[b];
                        // fill: run slots, then padding up to a multiple of 16 columns
                        if (tid < nb * NSUB && (tid - (tid / NSUB) * NSUB) == b) {
                            const int r = tid / NSUB, rv = run[b * MPB + r], st = rv & 0xffff, ln = rv >> 16;
                            unsigned short* dst = colslot + s0 + pre[b * MPB + r];
                            for (int q = 0; q < ln; ++q) dst[q] = (unsigned short)(st + q);
                        }
                        const int padded = (len + 15) & ~15;
                        if (tid >= NTHR - 16 && s0 + len + (tid - (NTHR - 16)) < s0 + padded) colslot[s0 + len + (tid - (NTHR - 16))] = 0xffffu;
                        s0 += padded;
                    }
                    if (tid == 0) seg[NSUB] = s0;
                }
                __syncthreads();
                const int ncols = seg[NSUB];
                // ---- 64 columns at a time: weights -> A stage, spectra -> B stage, MMAs
                for (int c0 = 0; c0 < ncols; c0 += KC) {
                    const int st = nfill & (NST - 1);
                    if (nfill >= NST) mbar_wait(&bar_free[st], ((nfill / NST) - 1) & 1);   // MMAs that read this stage are done
                    unsigned char* As = smem + L::offA + st * (KC * 256);
                    unsigned char* Bs = smem + L::offB + st * (KC * NN * 2);
                    // phase 1: thread = (column, part); part 0: x taps, 1: y taps, 2..3: B row
                    {
                        const int cl = tid & (KC - 1), part = tid >> 6, col = c0 + cl;
                        const int slot = (col < ncols) ? (int)colslot[col] : 0xffff;
                        int b = 0;
#pragma unroll
                        for (int q = 1; q < NSUB; ++q) b += (col >= seg[q]);
                        if (part == 0) {
                            wxs[cl] = make_uint4(0, 0, 0, 0);
                            wxs[KC + cl] = make_uint4(0, 0, 0, 0);
                            if (slot != 0xffff) {
                                const float4 mt = meta[slot];
                                const int l0 = (int)mt.x - (b & 1) * SUBX;
                                __half* w = reinterpret_cast<__half*>(wxs);
#pragma unroll
                                for (int t = 0; t < 2 * MH; ++t) {
                                    const float d = mt.y + (float)t;
                                    const int lx = l0 + t;
                                    if ((unsigned)lx < (unsigned)SUBX && d < (float)MH)
                                        w[((lx >> 3) * KC + cl) * 8 + (lx & 7)] = __float2half_rn(ex2_approx(-alpha2 * d * d));
                                }
                            }
                        } else if (part == 1) {
                            wys[cl] = make_uint4(0, 0, 0, 0);
                            if (slot != 0xffff) {
                                const float4 mt = meta[slot];
                                const int l0 = (int)mt.z - (b >> 1) * SUBY;
                                __half* w = reinterpret_cast<__half*>(wys);
#pragma unroll
                                for (int t = 0; t < 2 * MH; ++t) {
                                    const float d = mt.w + (float)t;
                                    const int ly = l0 + t;
                                    if ((unsigned)ly < (unsigned)SUBY && d < (float)MH)
                                        w[cl * 8 + ly] = __float2half_rn(ex2_approx(-alpha2 * d * d));
                                }
                            }
                        } else {
                            // B row: n-block q of column cl at (cl / 8) * B_LBO + q * 128 + (cl % 8) * 16
#pragma unroll
                            for (int q = (part - 2) * (GW / 2); q < (part - 1) * (GW / 2); ++q) {
                                const uint4 v = (slot != 0xffff) ? gs[(size_t)slot * GW + q] : make_uint4(0, 0, 0, 0);
                                *reinterpret_cast<uint4*>(Bs + (cl >> 3) * L::B_LBO + q * 128 + (cl & 7) * 16) = v;
                            }
                        }
                    }
                    __syncthreads();
                    // phase 2: A[m = ly * 16 + lx][column] = wy[ly] * wx[lx], MN-major: 8 cells = 16 B
#pragma unroll
                    for (int u = tid; u < KC * SUBY; u += NTHR) {
                        const int cl = u & (KC - 1), ly = u >> 6;
                        const unsigned short wyb = reinterpret_cast<const unsigned short*>(wys)[cl * 8 + ly];
                        uint4 lo = make_uint4(0, 0, 0, 0), hi = lo;
                        if (wyb != 0) {
                            const __half wyh = __ushort_as_half(wyb);
                            const __half2 wy2 = __halves2half2(wyh, wyh);
                            const uint4 a = wxs[cl], c = wxs[KC + cl];
                            auto mul = [&](unsigned x) {
                                const __half2 p = __hmul2(*reinterpret_cast<const __half2*>(&x), wy2);
                                return *reinterpret_cast<const unsigned*>(&p);
                            };
                            lo = make_uint4(mul(a.x), mul(a.y), mul(a.z), mul(a.w));
                            hi = make_uint4(mul(c.x), mul(c.y), mul(c.z), mul(c.w));
                        }
                        unsigned char* dst = As + (cl >> 3) * A_LBO + (2 * ly) * 128 + (cl & 7) * 16;
                        *reinterpret_cast<uint4*>(dst) = lo;
                        *reinterpret_cast<uint4*>(dst + 128) = hi;
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    __syncthreads();
                    if (tid == 0) {
                        asm volatile("tcgen05.fence::after_thread_sync;");
                        const int nk = (min(KC, ncols - c0) + 15) >> 4;
                        const uint32_t a0 = smem_u32(As), b0a = smem_u32(Bs);
                        for (int kk = 0; kk < nk; ++kk) {
                            const int col = c0 + kk * 16;
                            int b = 0;
#pragma unroll
                            for (int q = 1; q < NSUB; ++q) b += (col >= seg[q]);
                            umma_f16(tmem + (uint32_t)(b * NN), umma_desc(a0 + kk * 2 * A_LBO, A_LBO, 128),
                                     umma_desc(b0a + kk * 2 * L::B_LBO, L::B_LBO, 128), IDESC, (started >> b) & 1u);
                            started |= 1u << b;
                        }
                        umma_commit(&bar_free[st]);
                    }
                    ++nfill;
                }
                __syncthreads();                      // staging buffers, runs and column list are reused
            }
        }
    }

    // ---- epilogue: wait for the MMAs, TMEM -> registers -> grid (or partial tile)
    if (tid == 0) {
        shared_u32[1] = started;
        if (started) umma_commit(bar_done);
    }
    __syncthreads();
    const uint32_t started_all = shared_u32[1];
    if (started_all) mbar_wait(bar_done, 0);
    asm volatile("tcgen05.fence::after_thread_sync;");
    {
        const int q = warp & 3, hsel = warp >> 2;
        const int mrow = q * 32 + lane, ly = mrow >> 4, lx = mrow & 15;
#pragma unroll 1
        for (int bb = 0; bb < NSUB / 2; ++bb) {
            const int b = hsel * (NSUB / 2) + bb;
            uint32_t r[NN];
            if ((started_all >> b) & 1u) {
                TmemLd<NN>::run(tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(b * NN), r);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            } else {
#pragma unroll
                for (int e = 0; e < NN; ++e) r[e] = 0u;
            }
            const int ry = (b >> 1) * SUBY + ly, rx = (b & 1) * SUBX + lx;      // region-relative cell
            if (item.z < 0) {
#pragma unroll
                for (int p = 0; p < NPG; ++p) {
                    const int pair = pg * NPG + p;
                    if (pair < npair)
                        grid[((size_t)pair * M + TY0 + ry) * M + TX0 + rx] = __floats2half2_rn(__uint_as_float(r[2 * p]), __uint_as_float(r[2 * p + 1]));
                }
            } else {
#pragma unroll
                for (int p = 0; p < NPG; ++p) {
                    const int pair = pg * NPG + p;
                    if (pair < npair)
                        partial[(((size_t)(item.z + split) * npair + pair) * TS + ry) * TS + rx] =
                            make_float2(__uint_as_float(r[2 * p]), __uint_as_float(r[2 * p + 1]));
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(NSUB * NN));
}

// ---------------------------------------------------------------------------------------
template <int MH, int NN>
static int launch_mma_t(const tcp_ctx* c, cudaStream_t st) {
    using L = MmaSmem<MH, NN>;
    auto kern = grid_mma_kernel<MH, NN>;
    TCP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::total));
    const double alpha = 3.14159265358979323846 / (1.4142135623730951 * MH);
    dim3 grid(c->g_nitems, (c->npair + NN / 2 - 1) / (NN / 2));
    kern<<<grid, NTHR, L::total, st>>>((const __half2*)c->spec, (__half2*)c->grid, c->g_partial, c->trig, c->g_plan, c->g_items,
                                       c->nproj, c->M, c->npair, (float)(alpha * 1.4426950408889634));
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

// Enqueue the tensor-core gridding of the spectrum into the grid (fp16 storage only); the plan
// kernel and the split-tile reduce are launched by launch_grid_tile's caller.
int launch_grid_mma_main(const tcp_ctx* c, cudaStream_t st) {
    if (!c->half_store) return set_error(TCP_EUNSUPPORTED, "tensor-core gridding needs fp16 storage");
    const bool wide = c->npair > 8;
    if (c->m == 3) return wide ? launch_mma_t<3, 32>(c, st) : launch_mma_t<3, 16>(c, st);
    return wide ? launch_mma_t<4, 32>(c, st) : launch_mma_t<4, 16>(c, st);
}

}  // namespace tcpk
