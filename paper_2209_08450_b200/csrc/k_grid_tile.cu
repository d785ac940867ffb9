// k_grid_tile.cu -- S5 (default implementation): tile-owned, atomics-free gridding.
//
//   F[l2][l1] = sum_{j,k} G[j][k] phi(l1 - k cos_j) phi(l2 - k sin_j),  taps l = floor(nu) + a,
//   a = -m+1..m, phi(t) = exp(-alpha t^2), periodic in M      (reading Q7)
//
// Design:
//  * A CTA OWNS a 32 x 32 tile of Cartesian cells for NP slice pairs; a thread owns a 2 x 2 cell
//    block for all NP pairs (64 fp32 accumulators at NP = 8).  Nothing is scattered, no atomics,
//    the summation order is fixed => bitwise reproducible.
//  * The Gaussian weight of a (cell, sample) pair does not depend on the slice, so it is computed
//    once and applied to all NP pairs; with fp16 storage the multiply-accumulate is the sm_100
//    mixed-precision FMA (fma.rn.f32.f16 -> SASS FHFMA: fp32 accumulator, fp16 x fp16 product,
//    full FFMA rate, no conversion instructions).
//  * Samples near a tile are contiguous runs of k on the rays that cross the tile (the grid side
//    equals the padded row length M, so samples are one cell apart along a ray).  A plan kernel
//    finds, per tile, the angular window of projections that can cross it (theta is increasing);
//    the CTA tests those, stages the chords -- the NP spectra values of each sample, interleaved,
//    plus the sample's position -- in shared memory, and each thread then walks ITS OWN candidate
//    list (per-lane flattened loop: lanes do not wait for each other's rays).
//  * The tap decision floor(nu) is taken in fp64 at staging, exactly as the definition states it;
//    the per-thread arithmetic is fp32 on tile-relative coordinates (|x| < 64, error ~1e-6 cells).
//  * Tiles near DC collect most samples (density ~ 1/radius): they are split over several CTAs by
//    projection sub-ranges; the partial tiles are summed in split order by grid_reduce_kernel.
#include <math.h>

#include <algorithm>
#include <vector>

#include "grid_common.cuh"
#include "mmafft.cuh"
#include "tcp_internal.h"

namespace tcpk {

// ---------------------------------------------------------------------------------------
// Plan: per tile and periodic image, the window [ja, ja + count) (mod nproj) of projections whose
// ray can cross the tile.  One thread per (tile, image).
__global__ void grid_plan_kernel(const float* __restrict__ theta, int nproj, int M, int MH, int2* __restrict__ plan, int* __restrict__ counter) {
    const int n = M >> 1, tiles = M / TS;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < 64) counter[idx] = 0;          // work counters of the persistent tcgen05 gridding CTAs
    if (idx >= tiles * tiles * 4) return;
    const int img = idx & 3, tile = idx >> 2;
    const int tx = tile % tiles, ty = tile / tiles;
    int X0 = tx * TS, Y0 = ty * TS;
    if (X0 >= n) X0 -= M;
    if (Y0 >= n) Y0 -= M;
    // image shifts: cells at the negative edge also receive samples near +n (shift +M) and
    // cells at the positive edge samples near -n (shift -M)
    int sx = 0, sy = 0;
    bool valid = true;
    if (img & 1) { if (X0 == -n) sx = M; else if (X0 + TS == n) sx = -M; else valid = false; }
    if (img & 2) { if (Y0 == -n) sy = M; else if (Y0 + TS == n) sy = -M; else valid = false; }
    int2 out = make_int2(0, 0);
    if (valid) {
        const float PI_F = 3.14159265358979f;
        const float h = 0.5f * TS + (float)MH + 0.05f;
        const float xc = (float)(X0 + sx) + 0.5f * TS - 0.5f, yc = (float)(Y0 + sy) + 0.5f * TS - 0.5f;
        const float rho = sqrtf(xc * xc + yc * yc), rd = h * 1.41421357f;
        if (rho - rd <= (float)(n - 1)) {
            out = make_int2(0, nproj);
            if (rho > rd + 1.f) {
                const float delta = asinf(fminf(1.f, rd / rho)) + 2e-3f;
                if (delta < 0.5f * PI_F - 1e-2f) {
                    const float t0 = theta[0];
                    float a = atan2f(yc, xc) - delta - t0;
                    a -= PI_F * floorf(a / PI_F);                      // [0, pi)
                    int lo = 0, hi = nproj;                            // first j with theta[j] - t0 >= a
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        if (theta[mid] - t0 < a) lo = mid + 1; else hi = mid;
                    }
                    // window length: first cnt whose projection (theta increasing, + pi after the wrap) leaves
                    // [a, a + 2 delta]; monotone in cnt, so a second binary search
                    int clo = 0, chi = nproj;
                    while (clo < chi) {
                        const int mid = (clo + chi) >> 1;
                        int j = lo + mid;
                        float wrapped = 0.f;
                        if (j >= nproj) { j -= nproj; wrapped = PI_F; }
                        if ((theta[j] - t0) + wrapped - a > 2.f * delta) chi = mid; else clo = mid + 1;
                    }
                    out = make_int2(lo % nproj, clo);
                }
            }
        }
    }
    plan[idx] = out;
}

// ---------------------------------------------------------------------------------------
// item: x = tile index, y = split index s | nsplit S << 16, z = first partial slot (-1: write the grid)
template <int MH, int NP, class TC>
__global__ void __launch_bounds__(NTHR, 2)
    grid_tile_kernel(const TC* __restrict__ spec, TC* __restrict__ grid, float2* __restrict__ partial,
                     const double2* __restrict__ trig, const int2* __restrict__ plan, const int4* __restrict__ items,
                     int nproj, int M, int npair, float alpha2, const float* __restrict__ kbtab) {
    constexpr int KL = chord_len(MH);
    constexpr int PB = batch_records<TC>();
    constexpr int GW = NP * (int)sizeof(TC) / 16;           // uint4 words of spectrum per sample
    static_assert(PB <= MAXREC, "hit mask is 32 bits");
    static_assert(GW >= 1, "NP * sizeof(TC) must be a multiple of 16");

    extern __shared__ uint4 smem_u4[];
    float4* meta = reinterpret_cast<float4*>(smem_u4);                      // [PB*KL] qx, fx, qy, fy
    uint4* gs = smem_u4 + PB * KL;                                          // [PB*KL][GW]
    ChordRec* rec = reinterpret_cast<ChordRec*>(gs + PB * KL * GW);         // [PB]
    int* recj = reinterpret_cast<int*>(rec + PB);                           // [PB]
    int2* hits = reinterpret_cast<int2*>(recj + PB + (PB & 1));             // [NTHR] j, kmin | cnt << 16
    int* wcount = reinterpret_cast<int*>(hits + NTHR);                      // [NTHR/32 + 1]

    const int n = M >> 1, tiles = M / TS;
    const int4 item = items[blockIdx.x];
    const int tile = item.x, split = item.y & 0xffff, nsplit = item.y >> 16;
    const int pg = blockIdx.y;                                              // pair group
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // warp = 8 x 4 threads = 16 x 8 cells; CTA = 2 x 4 warps
    const int tx = (warp & 1) * 8 + (lane & 7), ty = (warp >> 1) * 4 + (lane >> 3);
    const int TX0 = (tile % tiles) * TS, TY0 = (tile / tiles) * TS;         // FFT-order origin
    const float cxa = (float)(2 * tx), cya = (float)(2 * ty);               // cell a, tile-relative

    float acc[4][NP][2];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int p = 0; p < NP; ++p) acc[c][p][0] = acc[c][p][1] = 0.f;

    for (int img = 0; img < 4; ++img) {
        const int2 win = plan[tile * 4 + img];
        if (win.y == 0) continue;                                           // uniform over the CTA
        int X0 = (TX0 >= n) ? TX0 - M : TX0, Y0 = (TY0 >= n) ? TY0 - M : TY0;
        if (img & 1) X0 += (X0 == -n) ? M : -M;
        if (img & 2) Y0 += (Y0 == -n) ? M : -M;
        const float hw = (float)MH + 0.02f;
        const float bax = (float)X0 - hw, bbx = (float)(X0 + TS - 1) + hw;  // sample box of the tile
        const float bay = (float)Y0 - hw, bby = (float)(Y0 + TS - 1) + hw;
        const float Bx = (float)X0 + cxa + 0.5f, By = (float)Y0 + cya + 0.5f;   // block centre
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

            for (int b0 = 0; b0 < nhit; b0 += PB) {
                const int nb = min(PB, nhit - b0);
                // ---- chord records
                if (tid < nb) {
                    const int2 h = hits[b0 + tid];
                    const double2 cs = trig[h.x];
                    ChordRec r;
                    r.c = (float)cs.x;
                    r.s = (float)cs.y;
                    const int dom = fabsf(r.s) > fabsf(r.c);
                    r.inv = 1.f / (dom ? r.s : r.c);
                    r.pack = h.y | (dom << 24);
                    rec[tid] = r;
                    recj[tid] = h.x;
                }
                __syncthreads();
                // ---- stage the chords: NP spectrum values + position of every sample
                for (int idx = tid; idx < nb * KL; idx += NTHR) {
                    const int r = idx / KL, kl = idx - r * KL;
                    const int pk = rec[r].pack;
                    if (kl >= ((pk >> 16) & 0xff)) continue;
                    const int k = (int)(short)(pk & 0xffff) + kl;
                    const int jj = recj[r];
                    const double2 cs = trig[jj];
                    const double nu1 = (double)k * cs.x, nu2 = (double)k * cs.y;
                    const double f1 = floor(nu1), f2 = floor(nu2);
                    // open box |l - nu| < m: 2m taps a = -m+1..m around floor(nu), stored so that
                    // e = cell - q = a - 1/2 and d = e - f = l - nu; when nu is an integer the tap a = m
                    // sits ON the box edge and is dropped: store q = floor(nu), f = 0, so e = d = a and
                    // the same test |e| < m keeps a = -m+1..m-1
                    const bool i1 = (nu1 == f1), i2 = (nu2 == f2);
                    meta[idx] = make_float4((float)(f1 - (double)X0) + (i1 ? 0.f : 0.5f), i1 ? 0.f : (float)(nu1 - f1) - 0.5f,
                                            (float)(f2 - (double)Y0) + (i2 ? 0.f : 0.5f), i2 ? 0.f : (float)(nu2 - f2) - 0.5f);
                    alignas(16) TC v[NP];
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        const int pair = pg * NP + p;
                        v[p] = (pair < npair) ? spec[((size_t)pair * nproj + jj) * M + (size_t)(k & (M - 1))] : czero<TC>();
                    }
                    const uint4* vv = reinterpret_cast<const uint4*>(v);
#pragma unroll
                    for (int q = 0; q < GW; ++q) gs[(size_t)idx * GW + q] = vv[q];
                }
                __syncthreads();
                // ---- which chords cross this thread's 2 x 2 block (widened by the support)?
                unsigned mask = 0;
                const float hb = (float)MH + 0.52f;
                for (int r = 0; r < nb; ++r) {
                    const ChordRec R = rec[r];
                    const float dperp = fmaf(By, R.c, -Bx * R.s);
                    if (fabsf(dperp) <= hb * (fabsf(R.c) + fabsf(R.s))) mask |= 1u << r;
                }
                // ---- per-lane flattened walk over (chord, sample) candidates
                int k = 0, kend = -1, base = 0;
                while (true) {
                    if (k > kend) {
                        bool got = false;
                        while (mask) {
                            const int r = __ffs(mask) - 1;
                            mask &= mask - 1;
                            const ChordRec R = rec[r];
                            const int dom = (R.pack >> 24) & 1, rk0 = (int)(short)(R.pack & 0xffff), rcnt = (R.pack >> 16) & 0xff;
                            const float kc = (dom ? By : Bx) * R.inv, hr = hb * fabsf(R.inv);
                            k = max(rk0, (int)ceilf(kc - hr));
                            kend = min(rk0 + rcnt - 1, (int)floorf(kc + hr));
                            base = r * KL - rk0;
                            if (k <= kend) { got = true; break; }
                        }
                        if (!got) break;
                    }
                    const int slot = base + k;
                    ++k;
                    const float4 mt = meta[slot];
                    // tap offsets: e = a - 1/2 (a = l - floor(nu), valid -m+1..m <=> |e| < m); d = l - nu
                    const float exa = cxa - mt.x, exb = exa + 1.f, eya = cya - mt.z, eyb = eya + 1.f;
                    const float dxa = exa - mt.y, dxb = dxa + 1.f, dya = eya - mt.w, dyb = dya + 1.f;
                    float wxa = tap_weight(kbtab, dxa, alpha2), wxb = tap_weight(kbtab, dxb, alpha2);
                    float wya = tap_weight(kbtab, dya, alpha2), wyb = tap_weight(kbtab, dyb, alpha2);
                    wxa = (fabsf(exa) < (float)MH) ? wxa : 0.f;
                    wxb = (fabsf(exb) < (float)MH) ? wxb : 0.f;
                    wya = (fabsf(eya) < (float)MH) ? wya : 0.f;
                    wyb = (fabsf(eyb) < (float)MH) ? wyb : 0.f;
                    const float w0 = wya * wxa, w1 = wya * wxb, w2 = wyb * wxa, w3 = wyb * wxb;
                    if constexpr (sizeof(TC) == 4) {
                        const __half2 h01 = __floats2half2_rn(w0, w1), h23 = __floats2half2_rn(w2, w3);
                        const unsigned u01 = *reinterpret_cast<const unsigned*>(&h01), u23 = *reinterpret_cast<const unsigned*>(&h23);
                        const unsigned short hw0 = u01 & 0xffffu, hw1 = u01 >> 16, hw2 = u23 & 0xffffu, hw3 = u23 >> 16;
#pragma unroll
                        for (int q = 0; q < GW; ++q) {
                            const uint4 g = gs[(size_t)slot * GW + q];
                            const unsigned gw[4] = {g.x, g.y, g.z, g.w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int p = q * 4 + e;
                                cfma_h(acc[0][p][0], acc[0][p][1], gw[e], hw0);
                                cfma_h(acc[1][p][0], acc[1][p][1], gw[e], hw1);
                                cfma_h(acc[2][p][0], acc[2][p][1], gw[e], hw2);
                                cfma_h(acc[3][p][0], acc[3][p][1], gw[e], hw3);
                            }
                        }
                    } else {
#pragma unroll
                        for (int q = 0; q < GW; ++q) {
                            const uint4 g = gs[(size_t)slot * GW + q];
                            const float gf[4] = {__uint_as_float(g.x), __uint_as_float(g.y), __uint_as_float(g.z), __uint_as_float(g.w)};
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int p = q * 2 + e;
                                acc[0][p][0] = fmaf(w0, gf[2 * e], acc[0][p][0]); acc[0][p][1] = fmaf(w0, gf[2 * e + 1], acc[0][p][1]);
                                acc[1][p][0] = fmaf(w1, gf[2 * e], acc[1][p][0]); acc[1][p][1] = fmaf(w1, gf[2 * e + 1], acc[1][p][1]);
                                acc[2][p][0] = fmaf(w2, gf[2 * e], acc[2][p][0]); acc[2][p][1] = fmaf(w2, gf[2 * e + 1], acc[2][p][1]);
                                acc[3][p][0] = fmaf(w3, gf[2 * e], acc[3][p][0]); acc[3][p][1] = fmaf(w3, gf[2 * e + 1], acc[3][p][1]);
                            }
                        }
                    }
                }
                __syncthreads();                                            // batch buffers are reused
            }
        }
    }

    // ---- epilogue: cells a (l1, l2), b (l1+1, l2), c (l1, l2+1), d (l1+1, l2+1)
    const int L1 = TX0 + 2 * tx, L2 = TY0 + 2 * ty;
    if (item.z < 0) {
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int pair = pg * NP + p;
            if (pair >= npair) break;
            TC* g0 = grid + ((size_t)pair * M + L2) * M + L1;
            if constexpr (sizeof(TC) == 4) {
                const __half2 a = f2h2_sat(make_float2(acc[0][p][0], acc[0][p][1])), b = f2h2_sat(make_float2(acc[1][p][0], acc[1][p][1]));
                const __half2 c = f2h2_sat(make_float2(acc[2][p][0], acc[2][p][1])), d = f2h2_sat(make_float2(acc[3][p][0], acc[3][p][1]));
                *reinterpret_cast<uint2*>(g0) = make_uint2(*reinterpret_cast<const unsigned*>(&a), *reinterpret_cast<const unsigned*>(&b));
                *reinterpret_cast<uint2*>(g0 + M) = make_uint2(*reinterpret_cast<const unsigned*>(&c), *reinterpret_cast<const unsigned*>(&d));
            } else {
                *reinterpret_cast<float4*>(g0) = make_float4(acc[0][p][0], acc[0][p][1], acc[1][p][0], acc[1][p][1]);
                *reinterpret_cast<float4*>(g0 + M) = make_float4(acc[2][p][0], acc[2][p][1], acc[3][p][0], acc[3][p][1]);
            }
        }
    } else {
        // partial tile [slot][pair][32][32] float2
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int pair = pg * NP + p;
            if (pair >= npair) break;
            float2* q0 = partial + (((size_t)(item.z + split) * npair + pair) * TS + 2 * ty) * TS + 2 * tx;
            *reinterpret_cast<float4*>(q0) = make_float4(acc[0][p][0], acc[0][p][1], acc[1][p][0], acc[1][p][1]);
            *reinterpret_cast<float4*>(q0 + TS) = make_float4(acc[2][p][0], acc[2][p][1], acc[3][p][0], acc[3][p][1]);
        }
    }
}

// ---------------------------------------------------------------------------------------
// Sum the partial tiles of a split tile in split order and write the grid.
// red: x = tile, y = first slot, z = S.  One CTA per (split tile, pair); a thread sums 4 cells.
template <class TC>
__global__ void __launch_bounds__(NTHR) grid_reduce_kernel(const float2* __restrict__ partial, TC* __restrict__ grid,
                                                           const int4* __restrict__ red, int M, int npair, int strip, int rswz) {
    const int4 r = red[blockIdx.x];
    const int pair = blockIdx.y, tiles = M / TS;
    const int row = threadIdx.x >> 3, col = (threadIdx.x & 7) * 4;
    float2 a[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) a[e] = make_float2(0.f, 0.f);
    for (int s = 0; s < r.z; ++s) {
        const float4* p = reinterpret_cast<const float4*>(partial + (((size_t)(r.y + s) * npair + pair) * TS + row) * TS + col);
        const float4 u = p[0], v = p[1];
        a[0].x += u.x; a[0].y += u.y; a[1].x += u.z; a[1].y += u.w;
        a[2].x += v.x; a[2].y += v.y; a[3].x += v.z; a[3].y += v.w;
    }
    const int gr = (r.x / tiles) * TS + row, gc = (r.x % tiles) * TS + col;     // col is a multiple of 4
    TC* g = grid + (size_t)pair * M * M;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int c1 = gc + e;
        st_c(g, strip ? ((size_t)(c1 / strip) * M + (rswz ? mf::swz<4>(gr) : gr)) * strip + (c1 % strip) : (size_t)gr * M + c1, a[e]);
    }
}

// ---------------------------------------------------------------------------------------
// Host: work items.  A tile's load is estimated from its distance to DC assuming angles spread
// evenly over [0, pi) (only the balance depends on it, not the result); tiles above the cap are
// split by projection sub-range; items are issued heaviest first.
int grid_tile_setup(tcp_ctx* c) {
    const int M = c->M, n = c->n, tiles = M / TS, MH = c->m;
    const double h = 0.5 * TS + MH, rd = h * 1.4142135623730951;
    const double chord_avg = 0.9 * (TS + 2 * MH);
    // cap: a fraction of one CTA slot's fair share (148 SMs x 2 CTAs), see below
    double total = 0;
    std::vector<double> est((size_t)tiles * tiles);
    for (int ty = 0; ty < tiles; ++ty)
        for (int tx = 0; tx < tiles; ++tx) {
            int X0 = tx * TS, Y0 = ty * TS;
            if (X0 >= n) X0 -= M;
            if (Y0 >= n) Y0 -= M;
            const double xc = X0 + 0.5 * TS - 0.5, yc = Y0 + 0.5 * TS - 0.5, rho = sqrt(xc * xc + yc * yc);
            double np = 0;
            if (rho - rd <= n - 1) {
                np = c->nproj;
                if (rho > rd + 1.0) np = std::min<double>(np, c->nproj * 2.0 * asin(std::min(1.0, rd / rho)) / 3.14159265358979 * 0.75);
            }
            // Samples lie at radius <= n and reach MH cells further; rd bounds the tile's half diagonal plus MH, so a tile whose
            // centre is more than n + rd + 2 from DC (the corners of the grid, a fifth of it) receives nothing, nor do its periodic
            // images, which are further still: it gets no work item and is never written; the grid is zeroed once instead.
            const bool empty = rho - rd > n + 2;
            est[(size_t)ty * tiles + tx] = empty ? -1.0 : np * chord_avg + 64.0;        // + fixed per-tile cost
            if (!empty) total += est[(size_t)ty * tiles + tx];
        }
    // the floor keeps the per-item fixed cost small against its work; a grid with fewer tiles than CTA slots (M <= 512) is
    // bound by the latency of one CTA's walk instead, and splits four times finer (C1: gridding 0.142 -> 0.054 ms)
    const double floor_ = tiles * tiles < 2 * 148 ? 512.0 : 2048.0;
    const double cap = std::max(floor_, total / (148.0 * 2.0) / 3.0);      // a third of a slot's fair share (a sixth measured 9 % slower at C3: more partial tiles to write and sum)
    struct It { double w; int4 v; };
    std::vector<It> its;
    std::vector<int4> red;
    int nslots = 0;
    for (int t = 0; t < tiles * tiles; ++t) {
        if (est[t] < 0.0) continue;              // no sample can reach the tile: no item, its cells stay zero (tcp_ctx::grid_dirty)
        int S = (int)ceil(est[t] / cap);
        S = std::max(1, std::min(S, std::min(64, c->nproj)));
        int slot0 = -1;
        if (S > 1) { slot0 = nslots; nslots += S; red.push_back(make_int4(t, slot0, S, 0)); }
        for (int s = 0; s < S; ++s) its.push_back({est[t] / S, make_int4(t, s | (S << 16), slot0, 0)});
    }
    std::stable_sort(its.begin(), its.end(), [](const It& a, const It& b) { return a.w > b.w; });
    std::vector<int4> items;
    for (auto& it : its) items.push_back(it.v);
    c->g_nitems = (int)items.size();
    c->g_nred = (int)red.size();
    TCP_CUDA_CHECK(cudaMalloc((void**)&c->g_items, items.size() * sizeof(int4)));
    TCP_CUDA_CHECK(cudaMemcpy(c->g_items, items.data(), items.size() * sizeof(int4), cudaMemcpyHostToDevice));
    c->bytes += items.size() * sizeof(int4);
    if (!red.empty()) {
        TCP_CUDA_CHECK(cudaMalloc((void**)&c->g_red, red.size() * sizeof(int4)));
        TCP_CUDA_CHECK(cudaMemcpy(c->g_red, red.data(), red.size() * sizeof(int4), cudaMemcpyHostToDevice));
        const size_t pb = (size_t)nslots * c->npair * TS * TS * sizeof(float2);
        cudaError_t e = cudaMalloc((void**)&c->g_partial, pb);
        if (e != cudaSuccess) return set_error(TCP_ENOMEM, "cudaMalloc(%zu) failed: %s", pb, cudaGetErrorString(e));
        c->bytes += pb + red.size() * sizeof(int4);
    }
    TCP_CUDA_CHECK(cudaMalloc((void**)&c->g_plan, (size_t)tiles * tiles * 4 * sizeof(int2)));
    TCP_CUDA_CHECK(cudaMalloc((void**)&c->g_counter, 64 * sizeof(int)));
    c->bytes += (size_t)tiles * tiles * 4 * sizeof(int2);
    if (c->half_store) return grid_mma_cache_setup(c);
    return TCP_OK;
}

void grid_tile_free(tcp_ctx* c) {
    cudaFree(c->g_items); cudaFree(c->g_red); cudaFree(c->g_partial); cudaFree(c->g_plan); cudaFree(c->g_counter);
    grid_mma_cache_free(c);
}

template <int MH, int NP, class TC>
static int launch_tile_t(const tcp_ctx* c, cudaStream_t st) {
    constexpr int KL = chord_len(MH), PB = batch_records<TC>();
    const size_t smem = (size_t)PB * KL * (16 + NP * sizeof(TC)) + (size_t)PB * (sizeof(ChordRec) + 4) + 8 +
                        NTHR * sizeof(int2) + (NTHR / 32 + 1) * sizeof(int);
    auto kern = grid_tile_kernel<MH, NP, TC>;
    TCP_SMEM(kern, (int)smem);
    const double alpha = 3.14159265358979323846 / (1.4142135623730951 * MH);
    dim3 grid(c->g_nitems, (c->npair + NP - 1) / NP);
    kern<<<grid, NTHR, smem, st>>>((const TC*)c->spec, (TC*)c->grid, c->g_partial, c->trig, c->g_plan, c->g_items, c->nproj,
                                   c->M, c->npair, c->kbtab ? (float)(1.0 / ((double)MH * MH)) : (float)(alpha * 1.4426950408889634), c->kbtab);
    TCP_CUDA_CHECK(cudaGetLastError());
    return TCP_OK;
}

template <int MH, class TC>
static int launch_tile_np(const tcp_ctx* c, cudaStream_t st) {
    return (c->npair > 4) ? launch_tile_t<MH, 8, TC>(c, st) : launch_tile_t<MH, 4, TC>(c, st);
}

// plan -> main kernel (CUDA-core FMA tile kernel, or the tcgen05 kernel of k_grid_mma.cu for fp16
// storage) -> sum of the split near-DC tiles
int launch_grid_tile(const tcp_ctx* c, const float* theta, cudaStream_t st) {
    const int tiles = c->M / TS, nplan = tiles * tiles * 4;
    grid_plan_kernel<<<(nplan + 127) / 128, 128, 0, st>>>(theta, c->nproj, c->M, c->m, c->g_plan, c->g_counter);
    TCP_CUDA_CHECK(cudaGetLastError());
    int rc;
    if (c->grid_impl == TCP_GRID_MMA) rc = launch_grid_mma_main(c, theta, st);
    else if (c->m == 2) rc = c->half_store ? launch_tile_np<2, __half2>(c, st) : launch_tile_np<2, float2>(c, st);
    else if (c->m == 3) rc = c->half_store ? launch_tile_np<3, __half2>(c, st) : launch_tile_np<3, float2>(c, st);
    else rc = c->half_store ? launch_tile_np<4, __half2>(c, st) : launch_tile_np<4, float2>(c, st);
    if (rc) return rc;
    if (c->g_nred) {
        if (c->half_store)
            grid_reduce_kernel<__half2><<<dim3(c->g_nred, c->npair), NTHR, 0, st>>>(c->g_partial, (__half2*)c->grid, c->g_red, c->M, c->npair, c->grid_strip, ifft2_on_mma(c) ? 1 : 0);
        else
            grid_reduce_kernel<float2><<<dim3(c->g_nred, c->npair), NTHR, 0, st>>>(c->g_partial, (float2*)c->grid, c->g_red, c->M, c->npair, c->grid_strip, ifft2_on_mma(c) ? 1 : 0);
        TCP_CUDA_CHECK(cudaGetLastError());
    }
    return TCP_OK;
}

}  // namespace tcpk
