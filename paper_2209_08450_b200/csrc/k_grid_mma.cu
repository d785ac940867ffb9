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
// forms the outer products into the MN-major A stage.  Warp-specialised: 7 producer warps each build
// whole 32-column stages (one lane = one column, no block barrier inside the loop), 1 warp issues the
// MMAs in column order (fixed summation order => bitwise reproducible) from a ring of 4 stages
// guarded by full/empty mbarriers (tcgen05.commit frees a stage).
#include <math.h>
#include <stdio.h>

#include "grid_common.cuh"
#include "tcp_internal.h"

namespace tcpk {

constexpr int SUBX = 16, SUBY = 8, NSUB = 8;      // sub-tile = 128 cells; 2 x 4 sub-tiles per region
constexpr int MPB = 10;                           // chords per batch
constexpr int SC = 32;                            // columns (samples) per A/B stage = one producer warp
constexpr int NST = 4;                            // stages in the ring
constexpr int NPROD = 7;                          // producer warps; warp 7 issues the MMAs
constexpr int RUNMAX = 32;                        // >= samples of one chord inside a sub-tile's sample box
constexpr int COLMAX = NSUB * MPB * RUNMAX;       // flat column list capacity (segments are 16-aligned)
constexpr int A_LBO = (128 / 8) * 128;            // bytes between k-blocks of 8 columns in an A stage
constexpr int A_STAGE = SC * 256;                 // bytes of one A stage: [SC/8][16][8 columns][8 cells] half

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, no swizzle: start >> 4, leading (k-block) and stride (mn-block) byte offsets >> 4
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity, int tag = 0, int info = 0) {
    uint32_t done = 0;
#ifdef TCP_MBAR_WATCHDOG
    unsigned spins = 0;
#endif
    while (!done) {
        asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p;}"
                     : "=r"(done)
                     : "r"(smem_u32(b)), "r"(parity)
                     : "memory");
#ifdef TCP_MBAR_WATCHDOG
        if (!done && ++spins > (1u << 22)) {
            if ((threadIdx.x & 31) == 0)
                printf("mbar stuck: block %d,%d warp %d tag %d parity %u info %d\n", blockIdx.x, blockIdx.y, threadIdx.x >> 5, tag, parity, info);
            __trap();
        }
#endif
    }
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

__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}

// nu = k * (c_hi + c_lo) as floor + fraction, fp32 FMAs only (k exact, |k| < 2^13): the product's
// rounding error is recovered exactly by an FMA, so fl + frac = nu to ~1e-11 cells.
__device__ __forceinline__ void nu_split(float k, float c_hi, float c_lo, float& fl, float& frac) {
    const float p = k * c_hi;
    const float e = fmaf(k, c_hi, -p);
    const float t = fmaf(k, c_lo, e);
    fl = floorf(p);
    frac = (p - fl) + t;
    if (frac < 0.f) { fl -= 1.f; frac += 1.f; }
    else if (frac >= 1.f) { fl += 1.f; frac -= 1.f; }
}

// dynamic shared memory carve-up
template <int MH, int NN>
struct MmaSmem {
    static constexpr int KL = chord_len(MH);
    static constexpr int NSLOT = MPB * KL;
    static constexpr int GW = NN * 2 / 16;                   // uint4 per sample (B row)
    static constexpr int B_LBO = (NN / 8) * 128;
    static constexpr int B_STAGE = SC * NN * 2;
    static constexpr int offA = 0;                           // [NST] A stages
    static constexpr int offB = offA + NST * A_STAGE;        // [NST] B stages
    static constexpr int offMeta = offB + NST * B_STAGE;     // [NSLOT] float4: first tap x, d0x, first tap y, d0y
    static constexpr int offG = offMeta + NSLOT * 16;        // [NSLOT][GW] uint4
    static constexpr int offWs = offG + NSLOT * GW * 16;     // [NPROD][3][32] uint4: wx lo, wx hi, wy per lane
    static constexpr int offCol = offWs + NPROD * 3 * 32 * 16;   // [COLMAX] uint16
    static constexpr int offRec = offCol + COLMAX * 2;       // [MPB] ChordRec
    static constexpr int offRecj = offRec + MPB * 16;        // [MPB] int (padded to 64 B)
    static constexpr int offHits = offRecj + 64;             // [NTHR] int2
    static constexpr int offRun = offHits + NTHR * 8;        // run[NSUB][MPB], pre[NSUB][MPB] int
    static constexpr int offMisc = offRun + 2 * NSUB * MPB * 4;   // wcount[9], seg[9], tmem base, started
    static constexpr int offBar = offMisc + 128;             // mbarriers: full[NST], empty[NST], done
    static constexpr int total = offBar + 128;
};

// ---------------------------------------------------------------------------------------
// item: x = region (32 x 32 tile) index, y = split s | nsplit S << 16, z = first partial slot (-1: write the grid)
template <int MH, int NN>
__global__ void __launch_bounds__(NTHR, 2)
    grid_mma_kernel(const __half2* __restrict__ spec, __half2* __restrict__ grid, float2* __restrict__ partial,
                    const double2* __restrict__ trig, const float4* __restrict__ trigf, const int2* __restrict__ plan,
                    const int4* __restrict__ items, int nproj, int M, int npair, float alpha2) {
    using L = MmaSmem<MH, NN>;
    constexpr int KL = L::KL, GW = L::GW, NPG = NN / 2;
    extern __shared__ __align__(128) unsigned char smem[];
    float4* meta = reinterpret_cast<float4*>(smem + L::offMeta);
    uint4* gs = reinterpret_cast<uint4*>(smem + L::offG);
    unsigned short* colslot = reinterpret_cast<unsigned short*>(smem + L::offCol);
    ChordRec* rec = reinterpret_cast<ChordRec*>(smem + L::offRec);
    int* recj = reinterpret_cast<int*>(smem + L::offRecj);
    int2* hits = reinterpret_cast<int2*>(smem + L::offHits);
    int* run = reinterpret_cast<int*>(smem + L::offRun);             // [NSUB][MPB] start | len << 16
    int* pre = run + NSUB * MPB;                                      // [NSUB][MPB] offset inside the segment
    int* wcount = reinterpret_cast<int*>(smem + L::offMisc);          // [9]
    int* seg = wcount + 9;                                            // [9] segment starts (columns), seg[8] = total
    uint32_t* shared_u32 = reinterpret_cast<uint32_t*>(seg + 9);      // [0] tmem base, [1] started mask, [2] completed passes
    volatile uint32_t* prog = shared_u32 + 2;
    uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem + L::offBar);
    uint64_t* bar_empty = bar_full + NST;
    uint64_t* bar_done = bar_empty + NST;

    const int n = M >> 1, tiles = M / TS;
    const int4 item = items[blockIdx.x];
    const int tile = item.x, split = item.y & 0xffff, nsplit = item.y >> 16;
    const int pg = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TX0 = (tile % tiles) * TS, TY0 = (tile / tiles) * TS;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_empty[s], 1); }
        mbar_init(bar_done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
        shared_u32[1] = 0;
        shared_u32[2] = 0;
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
    uint32_t started = 0;          // issuer: sub-tiles whose accumulator has been written
    uint32_t gpass = 0;            // stages filled so far in this item (uniform)

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
                const float4 cs = trigf[j];
                hit = chord_range(cs.x, cs.z, bax, bbx, bay, bby, (float)(n - 1), kmin, kmax);
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
                    const float4 cs = trigf[h.x];
                    ChordRec r;
                    r.c = cs.x;
                    r.s = cs.z;
                    r.inv = 0.f;
                    r.pack = h.y;
                    rec[tid] = r;
                    recj[tid] = h.x;
                }
                __syncthreads();
                // ---- stage the chords: one B row (NN halves) + the first tap and its distance per sample.
                // taps l = floor(nu) - m + 1 + t, t = 0..2m-1, distance d_t = l - nu = d_0 + t; the open box
                // |l - nu| < m keeps t iff d_t < m (d_0 > -m always), and d_0 = -m+1 exactly iff nu is an integer
                for (int idx = tid; idx < nb * KL; idx += NTHR) {
                    const int r = idx / KL, kl = idx - r * KL;
                    const int pk = rec[r].pack;
                    if (kl >= ((pk >> 16) & 0xff)) continue;
                    const int k = (int)(short)(pk & 0xffff) + kl;
                    const int jj = recj[r];
                    const float4 cs = trigf[jj];
                    float f1, r1, f2, r2;
                    nu_split((float)k, cs.x, cs.y, f1, r1);
                    nu_split((float)k, cs.z, cs.w, f2, r2);
                    const float dint = -(float)(MH - 1);
                    float d1 = dint - r1, d2 = dint - r2;
                    if (r1 > 0.f && d1 >= dint) d1 = __uint_as_float(__float_as_uint(dint) + 1u);   // next below -m+1
                    if (r2 > 0.f && d2 >= dint) d2 = __uint_as_float(__float_as_uint(dint) + 1u);
                    meta[idx] = make_float4(f1 + dint - (float)X0, d1, f2 + dint - (float)Y0, d2);
                    const __half2* src = spec + ((size_t)(pg * NPG) * nproj + jj) * M + (size_t)(k & (M - 1));
                    const size_t pstride = (size_t)nproj * M;
                    alignas(16) __half2 v[NPG];
#pragma unroll
                    for (int p = 0; p < NPG; ++p) v[p] = (pg * NPG + p < npair) ? src[p * pstride] : czero<__half2>();
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
                        // run slots, then padding up to a multiple of 16 columns (one MMA K step = one sub-tile)
                        if (tid < nb * NSUB && (tid - (tid / NSUB) * NSUB) == b) {
                            const int r = tid / NSUB, rv = run[b * MPB + r], st = rv & 0xffff, ln = rv >> 16;
                            unsigned short* dst = colslot + s0 + pre[b * MPB + r];
                            for (int q = 0; q < ln; ++q) dst[q] = (unsigned short)(st + q);
                        }
                        const int padded = (len + 15) & ~15;
                        if (tid >= NTHR - 16 && len + (tid - (NTHR - 16)) < padded) colslot[s0 + len + (tid - (NTHR - 16))] = 0xffffu;
                        s0 += padded;
                    }
                    if (tid == 0) seg[NSUB] = s0;
                }
                __syncthreads();
                const int ncols = seg[NSUB];
                const int npass = (ncols + SC - 1) / SC;
                if (warp < NPROD) {
                    // ======== producers: one warp = one 32-column stage, one lane = one column ========
                    uint4* ws = reinterpret_cast<uint4*>(smem + L::offWs) + warp * 3 * 32;   // wx lo | wx hi | wy, [32 lanes]
                    for (int p = warp; p < npass; p += NPROD) {
                        const uint32_t gp = gpass + (uint32_t)p, st = gp % NST;
                        // the MMAs of pass gp - NST (same stage) must be complete.  An mbarrier wait only tells odd
                        // from even phases and producers of different rounds of a stage are different warps, so
                        // they follow the issuer's published count of completed passes instead
                        if (gp >= NST) {
#ifdef TCP_MBAR_WATCHDOG
                            unsigned spins = 0;
#endif
                            while (*prog + NST <= gp) {
#ifdef TCP_MBAR_WATCHDOG
                                if (++spins > (1u << 24)) { if (lane == 0) printf("prog stuck: block %d warp %d gp %u prog %u\n", blockIdx.x, warp, gp, *prog); __trap(); }
#endif
                            }
                            __threadfence_block();
                        }
                        unsigned char* As = smem + L::offA + st * A_STAGE;
                        unsigned char* Bs = smem + L::offB + st * L::B_STAGE;
                        const int col = p * SC + lane;
                        const int slot = (col < ncols) ? (int)colslot[col] : 0xffff;
                        int b = 0;
#pragma unroll
                        for (int q = 1; q < NSUB; ++q) b += (col >= seg[q]);
                        ws[lane] = make_uint4(0, 0, 0, 0);
                        ws[32 + lane] = make_uint4(0, 0, 0, 0);
                        ws[64 + lane] = make_uint4(0, 0, 0, 0);
                        unsigned char* brow = Bs + (lane >> 3) * L::B_LBO + (lane & 7) * 16;
                        if (slot != 0xffff) {
                            const float4 mt = meta[slot];
                            __half* wh = reinterpret_cast<__half*>(ws);
                            const int lx0 = (int)mt.x - (b & 1) * SUBX, ly0 = (int)mt.z - (b >> 1) * SUBY;
#pragma unroll
                            for (int t = 0; t < 2 * MH; ++t) {
                                const float dx = mt.y + (float)t, dy = mt.w + (float)t;
                                const int lx = lx0 + t, ly = ly0 + t;
                                if ((unsigned)lx < (unsigned)SUBX && dx < (float)MH)
                                    wh[((lx >> 3) * 32 + lane) * 8 + (lx & 7)] = __float2half_rn(ex2_approx(-alpha2 * dx * dx));
                                if ((unsigned)ly < (unsigned)SUBY && dy < (float)MH)
                                    wh[(64 + lane) * 8 + ly] = __float2half_rn(ex2_approx(-alpha2 * dy * dy));
                            }
#pragma unroll
                            for (int q = 0; q < GW; ++q) *reinterpret_cast<uint4*>(brow + q * 128) = gs[(size_t)slot * GW + q];
                        } else {
#pragma unroll
                            for (int q = 0; q < GW; ++q) *reinterpret_cast<uint4*>(brow + q * 128) = make_uint4(0, 0, 0, 0);
                        }
                        // A[m = ly * 16 + lx][column] = wy[ly] * wx[lx]; MN-major: 8 cells of a column = 16 B
                        const uint4 xa = ws[lane], xc = ws[32 + lane], yv = ws[64 + lane];
                        const unsigned yw[4] = {yv.x, yv.y, yv.z, yv.w};
                        unsigned char* arow = As + (lane >> 3) * A_LBO + (lane & 7) * 16;
#pragma unroll
                        for (int ly = 0; ly < SUBY; ++ly) {
                            const unsigned yb = (ly & 1) ? (yw[ly >> 1] >> 16) : (yw[ly >> 1] & 0xffffu);
                            uint4 lo = make_uint4(0, 0, 0, 0), hi = lo;
                            if (__any_sync(0xffffffffu, yb != 0)) {
                                const unsigned y2 = yb | (yb << 16);
                                auto mul = [&](unsigned x) {
                                    const __half2 pr = __hmul2(*reinterpret_cast<const __half2*>(&x), *reinterpret_cast<const __half2*>(&y2));
                                    return *reinterpret_cast<const unsigned*>(&pr);
                                };
                                lo = make_uint4(mul(xa.x), mul(xa.y), mul(xa.z), mul(xa.w));
                                hi = make_uint4(mul(xc.x), mul(xc.y), mul(xc.z), mul(xc.w));
                            }
                            *reinterpret_cast<uint4*>(arow + (2 * ly) * 128) = lo;
                            *reinterpret_cast<uint4*>(arow + (2 * ly + 1) * 128) = hi;
                        }
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&bar_full[st]);
                    }
                } else {
                    // ======== issuer: stages in column order ========
                    for (int p = 0; p < npass; ++p) {
                        const uint32_t gp = gpass + (uint32_t)p, st = gp % NST, round = gp / NST;
                        mbar_wait(&bar_full[st], round & 1, 2, (int)gp);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        if (lane == 0) {
                            const int nk = (min(SC, ncols - p * SC) + 15) >> 4;
                            const uint32_t a0 = smem_u32(smem + L::offA + st * A_STAGE), b0a = smem_u32(smem + L::offB + st * L::B_STAGE);
                            for (int kk = 0; kk < nk; ++kk) {
                                const int col = p * SC + kk * 16;
                                int b = 0;
#pragma unroll
                                for (int q = 1; q < NSUB; ++q) b += (col >= seg[q]);
                                umma_f16(tmem + (uint32_t)(b * NN), umma_desc(a0 + kk * 2 * A_LBO, A_LBO, 128),
                                         umma_desc(b0a + kk * 2 * L::B_LBO, L::B_LBO, 128), IDESC, (started >> b) & 1u);
                                started |= 1u << b;
                            }
                            umma_commit(&bar_empty[st]);
                            // observe the previous pass's completion (in order: no parity aliasing) and publish it
                            if (gp > 0) {
                                mbar_wait(&bar_empty[(gp - 1) % NST], ((gp - 1) / NST) & 1, 1, (int)gp);
                                *prog = gp;
                            }
                        }
                        __syncwarp();
                    }
                }
                gpass += (uint32_t)npass;
                __syncthreads();                      // staging buffers, runs and column list are reused
            }
        }
    }

    // ---- epilogue: wait for the MMAs, TMEM -> registers -> grid (or partial tile)
    if (tid == NPROD * 32) {
        shared_u32[1] = started;
        if (started) umma_commit(bar_done);
    }
    __syncthreads();
    const uint32_t started_all = shared_u32[1];
    if (started_all) mbar_wait(bar_done, 0, 3, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    {
        const int q = warp & 3, hsel = warp >> 2;
        const int mrow = q * 32 + lane, ly = mrow >> 4, lx = mrow & 15;
        const size_t pstride = (size_t)M * M;
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
                __half2* dst = grid + ((size_t)(pg * NPG) * M + TY0 + ry) * M + TX0 + rx;
#pragma unroll
                for (int p = 0; p < NPG; ++p)
                    if (pg * NPG + p < npair) dst[p * pstride] = __floats2half2_rn(__uint_as_float(r[2 * p]), __uint_as_float(r[2 * p + 1]));
            } else {
                float2* dst = partial + (((size_t)(item.z + split) * npair + pg * NPG) * TS + ry) * TS + rx;
#pragma unroll
                for (int p = 0; p < NPG; ++p)
                    if (pg * NPG + p < npair) dst[p * (TS * TS)] = make_float2(__uint_as_float(r[2 * p]), __uint_as_float(r[2 * p + 1]));
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
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
    kern<<<grid, NTHR, L::total, st>>>((const __half2*)c->spec, (__half2*)c->grid, c->g_partial, c->trig, c->trigf, c->g_plan,
                                       c->g_items, c->nproj, c->M, c->npair, (float)(alpha * 1.4426950408889634));
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

// Enqueue the tensor-core gridding of the spectrum into the grid (fp16 storage only); the plan
// kernel and the split-tile reduce are launched by launch_grid_tile.
int launch_grid_mma_main(const tcp_ctx* c, cudaStream_t st) {
    if (!c->half_store) return set_error(TCP_EUNSUPPORTED, "tensor-core gridding needs fp16 storage");
    const bool wide = c->npair > 8;
    if (c->m == 3) return wide ? launch_mma_t<3, 32>(c, st) : launch_mma_t<3, 16>(c, st);
    return wide ? launch_mma_t<4, 32>(c, st) : launch_mma_t<4, 16>(c, st);
}

}  // namespace tcpk
