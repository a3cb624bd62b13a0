// force_tiles.cuh -- the O(N^2) kernel: changeover-weighted pairwise accelerations (H_B kick,
// PAPER.md:86 Eq. 5) and, from the same tiles, the close-encounter pair list
// (PAPER.md:94, 98, 106).  fp64 FMA chains on the plain FP64 pipe; no tensor cores (this is not a
// dense contraction: r_ij^2 from a Gram matrix would cancel catastrophically for close pairs).
//
// Grid: blockIdx.x = i-block of kForceThreads*I bodies (I bodies per thread, in registers),
//       blockIdx.y = j-split (a contiguous range of j-tiles).  Each CTA streams its j-range through
//       a four-stage shared-memory ring filled by TMA bulk copies (cp.async.bulk, full/empty mbarriers) of
//       64-byte JRec records; every lane of a warp reads the same j => pure broadcasts.
// Out:  part[split][i][3], summed in split order by nb_kickv_kernel (deterministic two-level sum).
//
// Fast path, per interaction, FP64-pipe instructions (15):
//   dx,dy,dz = x_j - x_i                                  3 DADD
//   r2 = dx*dx + dy*dy + dz*dz                            1 DMUL + 2 DFMA
//   y0 = MUFU.RSQ64H(r2)  (~2^-20 relative, 21-bit mantissa; XU pipe, not FP64)
//   u  = y0*y0            (exact: 42 bits)                1 DMUL
//   e  = 1 - r2*u                                         1 DFMA
//   h  = G m_j (1 + 3/2 e + 15/8 e^2)  [(1-e)^(-3/2), next term 35/16 e^3 < 2^-56]   2 DFMA
//   s  = (u*y0) * h      = G m_j / r^3                    2 DMUL
//   a += s * (dx,dy,dz)                                   3 DFMA
// The encounter test never touches the FP64 pipe: positive doubles order like their high words, so
// min_k hi32(r2_k) <= max(hi32(rc_i^2), hi32(rc_j^2)) + 1 is a conservative integer pre-filter; a
// warp vote sends the (rare) hits, and every self term (r2 = 0), to the exact slow path.
#pragma once
#include "kepler.cuh"  // rcp_fast, rsqrt_fast, sqrt_from_rsqrt
#include "nb_common.cuh"

namespace nbk {

struct ForceParams {
    const JRec *jrec;            // [tiles_total * kTileJ] staged j-bodies (padded)
    const JRecDs *jds;           // [tiles_total * kTileJ] double-single records (mixed-precision kernel, I >= 2) or nullptr
    const double *x;             // [N,3] i-side positions
    const double *rcrit;         // [N]   i-side critical radii
    double *part;                // [nsplit, N, 3] partial accelerations
    int32_t *pairs;              // [cap,2] or nullptr
    unsigned long long *npairs;  // device counter
    long long *status;           // device int64[ST_COUNT]
    long long cap;
    int N;
    int Nj;           // number of force-exerting bodies (= n_active)
    int tiles_total;  // ceil(Nj / kTileJ)
    int tiles_per_split;
    int kind;  // changeover shape
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(addr), "r"(parity)
            : "memory");
    } while (!ok);
}

// MUFU.RSQ64H: reciprocal square root seed from the high word of a double (low word of the
// result is zero).  +0 -> +inf, never reached on the fast path (hi32(0) = 0 always votes slow).
__device__ __forceinline__ double rsqrt_seed(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
}

// Kick weight W(r; rc) between the end points (readings S1, S2).  Reciprocals from the MUFU
// seed with one third-order correction (~1 ulp, kepler.cuh): the exact path is not rare with the full Eq. 7 radius.
__device__ __forceinline__ double changeover_weight(double r, double rc, int kind) {
    const double t0 = r - 0.1 * rc;
    if (t0 <= 0.0) return 0.0;
    const double y = t0 * rcp_fast(0.9 * rc);
    if (y >= 1.0) return 1.0;
    if (kind == 1) return y * y * y * (10.0 + y * (-15.0 + 6.0 * y));
    return (y * y) * rcp_fast(2.0 * y * y - 2.0 * y + 1.0);
}

// W / r^3 for a pair inside rc (r2 > 0): no IEEE divide or square root
__device__ __forceinline__ double weighted_inv_r3(const double r2, const double rc, const bool inside, const int kind) {
    const double id = rsqrt_fast(r2);
    const double W = inside ? changeover_weight(sqrt_from_rsqrt(r2, id), rc, kind) : 1.0;
    return W * (id * id * id);
}

// Warp-aggregated append of encounter pairs (a3): one atomicAdd per warp-hit reserves the slots,
// lanes take them in lane order; overflow keeps counting, drops the writes and is reported.
// Must be called by all 32 lanes.
__device__ __forceinline__ void pair_append(int32_t *pairs, unsigned long long *npairs, long long *status,
                                            const long long cap, const bool emit, const int i, const int j) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned mask = __ballot_sync(0xffffffffu, emit);
    if (mask) {
        const int leader = __ffs(mask) - 1;
        const int cnt = __popc(mask);
        unsigned long long base = 0;
        if ((int)lane == leader) {
            base = atomicAdd(npairs, (unsigned long long)cnt);
            const long long end = (long long)base + cnt;
            const long long kept_end = end < cap ? end : cap;
            const long long kept = kept_end > (long long)base ? kept_end - (long long)base : 0;
            if (kept < cnt) status_add(status, ST_PAIR_DROPPED, cnt - kept);
        }
        base = __shfl_sync(0xffffffffu, base, leader);
        if (emit) {
            const long long pos = (long long)base + __popc(mask & ((1u << lane) - 1u));
            if (pos < cap) {
                const int lo = i < j ? i : j, hi = i < j ? j : i;
                reinterpret_cast<int2 *>(pairs)[pos] = make_int2(lo, hi);
            }
        }
    }
}

// Exact path for one j against this thread's I bodies: self term, strict r2 < rc_ij^2 pair test,
// changeover weight, IEEE sqrt/divide, warp-aggregated pair append.  Entered warp-uniformly.
template <int I, bool PAIRS>
__device__ __forceinline__ void slow_path(const ForceParams &p, const double4 A, const double4 B, const int j,
                                          const double (&xi)[I], const double (&yi)[I], const double (&zi)[I],
                                          const double (&rci)[I], const int i0, double (&ax)[I], double (&ay)[I],
                                          double (&az)[I], const bool mine = true) {
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + k * kForceThreads;
        const bool valid = mine && (i < p.N) && (j < p.Nj) && (i != j);
        const double dx = A.x - xi[k], dy = A.y - yi[k], dz = A.z - zi[k];
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        const double rc = fmax(rci[k], B.w);
        const double rc2 = rc * rc;
        const bool inside = valid && (r2 < rc2);
        if (valid) {
            if (r2 == 0.0) {
                if (!inside) status_add(p.status, ST_SINGULAR, 1);  // rc == 0 and coincident: contributes 0
            } else {
                const double wr3 = weighted_inv_r3(r2, rc, inside, p.kind);
                if (wr3 != 0.0) {
                    const double f = A.w * wr3;
                    ax[k] = __fma_rn(f, dx, ax[k]);
                    ay[k] = __fma_rn(f, dy, ay[k]);
                    az[k] = __fma_rn(f, dz, az[k]);
                }
            }
        }
        if (PAIRS) {
            // each unordered pair once: (i<j) among active bodies; passive i (>= Nj) sees j once only
            pair_append(p.pairs, p.npairs, p.status, p.cap, inside && (i < j || i >= p.Nj), i, j);
        }
    }
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// One j against the thread's I bodies: differences, r^2 and the running minimum of the high words.
template <int I>
struct JWork {
    double4 A, B;  // A = x, y, z, G m ; B = 3/2 G m, 15/8 G m, rc^2, rc
    double dx[I], dy[I], dz[I], r2[I];
    int mn, thr;
    __device__ __forceinline__ void load(const JRec *rec, const double (&xi)[I], const double (&yi)[I],
                                         const double (&zi)[I], const int thr_i) {
        const double4 *q = reinterpret_cast<const double4 *>(rec);
        A = q[0];
        B = q[1];
        thr = max(thr_i, __double2hiint(B.z) + 1);
        mn = 0x7fffffff;
#pragma unroll
        for (int k = 0; k < I; ++k) {
            dx[k] = __dsub_rn(A.x, xi[k]);
            dy[k] = __dsub_rn(A.y, yi[k]);
            dz[k] = __dsub_rn(A.z, zi[k]);
            r2[k] = __fma_rn(dz[k], dz[k], __fma_rn(dy[k], dy[k], __dmul_rn(dx[k], dx[k])));
            mn = min(mn, __double2hiint(r2[k]));
        }
    }
};

// The work of one CTA of kForceThreads threads: i-block bx, j-split by.  sm / full / empty: the CTA's shared-memory ring and
// its barriers, NOT yet initialised (a persistent caller -- step_small.cuh -- invalidates them between work items).
// BF: branch-free tile loop (latency-bound launches: few CTAs of one or two tiles each -- small N; measured N = 2048:
// 22.6 -> 16.5 us, but +6 % where the FP64 pipe is the limit, N = 65536 and the semi-active config)
template <int I, bool PAIRS, bool BF>
__device__ __forceinline__ void force_tiles_cta(const ForceParams &p, const int bx, const int by, JRec (*sm)[kTileJ],
                                                uint64_t *full, uint64_t *empty) {
    const int t = threadIdx.x;
    const int i0 = bx * (kForceThreads * I) + t;
    const int tile_begin = by * p.tiles_per_split;
    int tile_end = tile_begin + p.tiles_per_split;
    if (tile_end > p.tiles_total) tile_end = p.tiles_total;
    const int ntiles = tile_end - tile_begin;
    constexpr unsigned kTileBytes = kTileJ * sizeof(JRec);
    constexpr int kAhead = kStages - 2;  // tiles in flight ahead of the one being consumed

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
                tma_bulk_g2s(&sm[n][0], p.jrec + (size_t)(tile_begin + n) * kTileJ, kTileBytes, &full[n]);
            }
    }

    // i-bodies in registers
    double xi[I], yi[I], zi[I], rci[I];
    int thr_i = 0;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + k * kForceThreads;
        if (i < p.N) {
            xi[k] = p.x[3 * (size_t)i];
            yi[k] = p.x[3 * (size_t)i + 1];
            zi[k] = p.x[3 * (size_t)i + 2];
            rci[k] = p.rcrit[i];
        } else {
            xi[k] = kFarI; yi[k] = kFarI; zi[k] = kFarI; rci[k] = 0.0;
        }
        thr_i = max(thr_i, __double2hiint(rci[k] * rci[k]));
    }
    thr_i += 1;

    double ox[I], oy[I], oz[I];  // outer (per-CTA) sums; inner sums are flushed once per tile
#pragma unroll
    for (int k = 0; k < I; ++k) { ox[k] = 0.0; oy[k] = 0.0; oz[k] = 0.0; }

    for (int it = 0; it < ntiles; ++it) {
        const int st = it % kStages;
        {
            // refill the stage that tile it - 2 used.  Every thread takes the (almost always already
            // satisfied) wait so that control flow stays warp-uniform; one thread issues the copy.
            const int n = it + kAhead;
            if (n < ntiles) {
                const int sn = n % kStages;
                if (n >= kStages) mbar_wait(&empty[sn], (unsigned)((n / kStages - 1) & 1));
                if (t == 0) {
                    mbar_expect_tx(&full[sn], kTileBytes);
                    tma_bulk_g2s(&sm[sn][0], p.jrec + (size_t)(tile_begin + n) * kTileJ, kTileBytes, &full[sn]);
                }
            }
        }
        mbar_wait(&full[st], (unsigned)((it / kStages) & 1));

        double ax[I], ay[I], az[I];
#pragma unroll
        for (int k = 0; k < I; ++k) { ax[k] = 0.0; ay[k] = 0.0; az[k] = 0.0; }
        const int jbase = (tile_begin + it) * kTileJ;
        const JRec *tile = &sm[st][0];

        auto fast = [&](const JWork<I> &w, const double (&y0)[I]) {
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const double u = __dmul_rn(y0[k], y0[k]);
                const double e = __fma_rn(-w.r2[k], u, 1.0);
                const double h = __fma_rn(e, __fma_rn(e, w.B.y, w.B.x), w.A.w);
                const double s = __dmul_rn(__dmul_rn(u, y0[k]), h);
                ax[k] = __fma_rn(s, w.dx[k], ax[k]);
                ay[k] = __fma_rn(s, w.dy[k], ay[k]);
                az[k] = __fma_rn(s, w.dz[k], az[k]);
            }
        };

        if (BF) {
            // Branch-free form (as in force_sym.cuh): a lane within reach of a critical radius (always the self term)
            // feeds +inf to its seeds -- its I pairs contribute exactly 0 -- and sets a bit; the flagged j of each
            // group of 32 are then evaluated exactly by the lanes that flagged them.  No vote and no branch per j, so
            // consecutive j overlap in the FP64 pipe: what a CTA with a single tile (small N, semi-active) is short of.
            for (int g0 = 0; g0 < kTileJ; g0 += 32) {
                unsigned bits = 0u;
#pragma unroll 4
                for (int jj = 0; jj < 32; ++jj) {
                    JWork<I> cur;
                    cur.load(tile + g0 + jj, xi, yi, zi, thr_i);
                    const bool hit = cur.mn <= cur.thr;
                    bits |= (hit ? 1u : 0u) << jj;
                    const int kill = hit ? 0x7ff00000 : 0;
                    double y0[I];
#pragma unroll
                    for (int k = 0; k < I; ++k)
                        y0[k] = rsqrt_seed(__hiloint2double(max(__double2hiint(cur.r2[k]), kill), 0));
                    fast(cur, y0);
                }
                unsigned any = __reduce_or_sync(0xffffffffu, bits);
                while (any) {
                    const int jj = __ffs(any) - 1;
                    any &= any - 1u;
                    const double4 *q = reinterpret_cast<const double4 *>(tile + g0 + jj);
                    slow_path<I, PAIRS>(p, q[0], q[1], jbase + g0 + jj, xi, yi, zi, rci, i0, ax, ay, az, ((bits >> jj) & 1u) != 0u);
                }
            }
        } else {
#pragma unroll 4
        for (int jj = 0; jj < kTileJ; ++jj) {
            JWork<I> cur;
            cur.load(tile + jj, xi, yi, zi, thr_i);
            double y0[I];
#pragma unroll
            for (int k = 0; k < I; ++k) y0[k] = rsqrt_seed(cur.r2[k]);
            if (__any_sync(0xffffffffu, cur.mn <= cur.thr))
                slow_path<I, PAIRS>(p, cur.A, cur.B, jbase + jj, xi, yi, zi, rci, i0, ax, ay, az);
            else
                fast(cur, y0);
        }
        }
#pragma unroll
        for (int k = 0; k < I; ++k) { ox[k] += ax[k]; oy[k] += ay[k]; oz[k] += az[k]; }
        __syncwarp();
        if ((t & 31) == 0) mbar_arrive(&empty[st]);  // this warp is done with stage st
    }

    double *out = p.part + (size_t)by * p.N * 3;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + k * kForceThreads;
        if (i < p.N) {
            out[3 * (size_t)i] = ox[k];
            out[3 * (size_t)i + 1] = oy[k];
            out[3 * (size_t)i + 2] = oz[k];
        }
    }
}

// MINB = CTAs per SM the register allocation is capped for.
template <int I, bool PAIRS, int MINB, bool BF>
__global__ void __launch_bounds__(kForceThreads, MINB) nb_force_tiles_kernel(const ForceParams p) {
    __shared__ __align__(128) JRec sm[kStages][kTileJ];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ __align__(8) uint64_t empty[kStages];
    force_tiles_cta<I, PAIRS, BF>(p, blockIdx.x, blockIdx.y, sm, full, empty);
}

}  // namespace nbk
