// force_mixed.cuh -- mixed-precision variant of the one-sided O(N^2) kick (Fig. 1
// contrasts FP32 and FP64 runs of the same code on both of its GPUs).  What is computed is the H_B kick of
// force_tiles.cuh (Eq. 5, 98) and the same pair list; what changes is the arithmetic of the pairs that are
// out of reach of every critical radius (all but ~1e-6 of them), which runs on the FP32 pipe on double-single
// positions (nb_force_mixedds_kernel below; the Newton-III counterpart is force_symds.cuh).  Pairs whose fp32 r^2 is
// within reach of a critical radius (margin 2^-18: far above the fp32 rounding of r^2), and every self term, take the
// EXACT fp64 path of force_tiles.cuh: the changeover weight, the pair test r^2 < rc^2 and the pair list are
// bit-identical to the fp64 kernel's.  Tolerance reading: DESIGN.md S25.
// (Round 2's first version -- fp64 differences and conversions, fp32 for the rest -- was no faster than the fp64 kernel:
// the differences stayed on the FP64 pipe.  It is gone; with one i-body per thread (small N, latency-bound launches) the
// host runs the fp64 kernel, which meets the mixed tolerance trivially.)
#pragma once
#include "force_tiles.cuh"

namespace nbk {

// The one-sided counterpart of force_symds.cuh (semi-active mode, N below the Newton-III threshold; I = 2 or 4): 32-byte
// JRecDs records stream through the TMA ring, dx = fl(fl(xjh - xih) + fl(xjl - xil)) with the (high, low) partial
// differences in one packed FADD2, everything after the differences on two i-bodies at a time (FMUL2 / FFMA2), fp32 sums
// per 128-body tile, fp64 across tiles.  A j within reach of a critical radius (fp32 pre-filter, margin 2^-18; always the
// self term) takes the exact fp64 path with the fp64 record read from global memory (rare).  Tolerance: S25.
template <int I, bool PAIRS, int MINB>
__global__ void __launch_bounds__(kForceThreads, MINB) nb_force_mixedds_kernel(const ForceParams p) {
    static_assert(I == 2 || I == 4, "packed arithmetic takes the i-bodies two at a time");
    constexpr int H = I / 2;
    __shared__ __align__(128) JRecDs sm[kStages][kTileJ];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ __align__(8) uint64_t empty[kStages];

    const int t = threadIdx.x;
    const int i0 = blockIdx.x * (kForceThreads * I) + t;
    const int tile_begin = blockIdx.y * p.tiles_per_split;
    int tile_end = tile_begin + p.tiles_per_split;
    if (tile_end > p.tiles_total) tile_end = p.tiles_total;
    const int ntiles = tile_end - tile_begin;
    constexpr unsigned kTileBytes = kTileJ * sizeof(JRecDs);
    constexpr int kAhead = kStages - 2;

    if (t == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kForceThreads / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (t == 0) {
#pragma unroll
        for (int n = 0; n < kAhead; ++n)
            if (n < ntiles) {
                mbar_expect_tx(&full[n], kTileBytes);
                tma_bulk_g2s(&sm[n][0], p.jds + (size_t)(tile_begin + n) * kTileJ, kTileBytes, &full[n]);
            }
    }

    double xi[I], yi[I], zi[I], rci[I];
    float2 nxa[I], nya[I], nza[I];   // the i-bodies, negated, as (high, low)
    float thr_i = 0.0f;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + k * kForceThreads;
        if (i < p.N) {
            xi[k] = p.x[3 * (size_t)i]; yi[k] = p.x[3 * (size_t)i + 1]; zi[k] = p.x[3 * (size_t)i + 2];
            rci[k] = p.rcrit[i];
        } else {
            xi[k] = kFarI; yi[k] = kFarI; zi[k] = kFarI; rci[k] = 0.0;
        }
        const JRecDs r = make_jrecds(xi[k], yi[k], zi[k], 0.0, rci[k] * rci[k]);
        nxa[k] = make_float2(-r.xh, -r.xl); nya[k] = make_float2(-r.yh, -r.yl); nza[k] = make_float2(-r.zh, -r.zl);
        thr_i = fmaxf(thr_i, r.thr);
    }
    double ox[I], oy[I], oz[I];
#pragma unroll
    for (int k = 0; k < I; ++k) { ox[k] = 0.0; oy[k] = 0.0; oz[k] = 0.0; }

    for (int it = 0; it < ntiles; ++it) {
        const int st = it % kStages;
        {
            const int n = it + kAhead;
            if (n < ntiles) {
                const int sn = n % kStages;
                if (n >= kStages) mbar_wait(&empty[sn], (unsigned)((n / kStages - 1) & 1));
                if (t == 0) {
                    mbar_expect_tx(&full[sn], kTileBytes);
                    tma_bulk_g2s(&sm[sn][0], p.jds + (size_t)(tile_begin + n) * kTileJ, kTileBytes, &full[sn]);
                }
            }
        }
        mbar_wait(&full[st], (unsigned)((it / kStages) & 1));

        float2 fx[H], fy[H], fz[H];   // fp32 sums of this tile, bodies (2g, 2g+1)
#pragma unroll
        for (int g = 0; g < H; ++g) { fx[g] = make_float2(0.f, 0.f); fy[g] = fx[g]; fz[g] = fx[g]; }
        const int jbase = (tile_begin + it) * kTileJ;
        const float4 *tile = reinterpret_cast<const float4 *>(&sm[st][0]);
#pragma unroll 4
        for (int jj = 0; jj < kTileJ; ++jj) {
            const float4 a = tile[2 * jj];        // (xh, xl, yh, yl)
            const float4 b = tile[2 * jj + 1];    // (zh, zl, G m, threshold)
            const float2 jx = make_float2(a.x, a.y), jy = make_float2(a.z, a.w), jz = make_float2(b.x, b.y);
            float2 dx[H], dy[H], dz[H], r2[H];
#pragma unroll
            for (int g = 0; g < H; ++g) {
                const float2 x0 = __fadd2_rn(jx, nxa[2 * g]), x1 = __fadd2_rn(jx, nxa[2 * g + 1]);
                const float2 y0 = __fadd2_rn(jy, nya[2 * g]), y1 = __fadd2_rn(jy, nya[2 * g + 1]);
                const float2 z0 = __fadd2_rn(jz, nza[2 * g]), z1 = __fadd2_rn(jz, nza[2 * g + 1]);
                dx[g] = make_float2(__fadd_rn(x0.x, x0.y), __fadd_rn(x1.x, x1.y));
                dy[g] = make_float2(__fadd_rn(y0.x, y0.y), __fadd_rn(y1.x, y1.y));
                dz[g] = make_float2(__fadd_rn(z0.x, z0.y), __fadd_rn(z1.x, z1.y));
                r2[g] = __ffma2_rn(dz[g], dz[g], __ffma2_rn(dy[g], dy[g], __fmul2_rn(dx[g], dx[g])));
            }
            float mn = fminf(r2[0].x, r2[0].y);
#pragma unroll
            for (int g = 1; g < H; ++g) mn = fminf(mn, fminf(r2[g].x, r2[g].y));
            if (__any_sync(0xffffffffu, mn <= fmaxf(thr_i, b.w))) {
                // exact fp64 path for this j (self term, pairs within reach of a critical radius), straight into the fp64 sums
                const double4 *q = reinterpret_cast<const double4 *>(p.jrec + (size_t)jbase + jj);
                slow_path<I, PAIRS>(p, q[0], q[1], jbase + jj, xi, yi, zi, rci, i0, ox, oy, oz);
            } else {
                const float2 gmj = make_float2(b.z, b.z);
#pragma unroll
                for (int g = 0; g < H; ++g) {
                    float2 y0;
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0.x) : "f"(r2[g].x));
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0.y) : "f"(r2[g].y));
                    const float2 s = __fmul2_rn(__fmul2_rn(__fmul2_rn(y0, y0), y0), gmj);
                    fx[g] = __ffma2_rn(s, dx[g], fx[g]); fy[g] = __ffma2_rn(s, dy[g], fy[g]); fz[g] = __ffma2_rn(s, dz[g], fz[g]);
                }
            }
        }
#pragma unroll
        for (int g = 0; g < H; ++g) {
            ox[2 * g] += (double)fx[g].x; oy[2 * g] += (double)fy[g].x; oz[2 * g] += (double)fz[g].x;
            ox[2 * g + 1] += (double)fx[g].y; oy[2 * g + 1] += (double)fy[g].y; oz[2 * g + 1] += (double)fz[g].y;
        }
        __syncwarp();
        if ((t & 31) == 0) mbar_arrive(&empty[st]);
    }

    double *out = p.part + (size_t)blockIdx.y * p.N * 3;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + k * kForceThreads;
        if (i < p.N) { out[3 * (size_t)i] = ox[k]; out[3 * (size_t)i + 1] = oy[k]; out[3 * (size_t)i + 2] = oz[k]; }
    }
}

}  // namespace nbk
