// force_sym.cuh -- Newton-III form of the O(N^2) kick for the fully active case (Eq. 5,
// PAPER.md:98; pair list PAPER.md:94, 98, 106).  Each unordered pair {i,j} is evaluated ONCE and
// its r^-3 serves both bodies: 20 FP64-pipe instructions per unordered pair = 10 per ordered
// interaction, against 15 in the one-sided tile kernel (force_tiles.cuh), which stays the kernel of
// the semi-active mode and of small N.
//
// Work unit: a super-tile (A, B), A <= B, of S x S bodies; one CTA of W warps per super-tile (W = 4 for S >= 512,
// 2 for S = 256, 1 for S = 128 at I = 4: always 12 warps per SM; the small tiles are what keeps the tail of a
// mid-sized problem short -- a lone CTA runs hardly faster than one of many).
//   * B's bodies (x, y | z, Gm | threshold word; doubled-block layout, see SymParams) are staged
//     ONCE in shared memory by three TMA bulk copies; B's accelerations accumulate in shared memory (jS).
//   * A's bodies are taken in chunks of 32*W*I; every lane holds I of them in registers together
//     with their accumulators.
//   * A warp meets a block of 32 j-bodies by ROTATION: lane l starts with j = l, evaluates its I
//     pairs, then the three j-accumulators move one lane down (6 SHFL) while the next j's constants
//     come from shared memory; after 32 rotations every (i, j) pair of the 32I x 32 block has been
//     visited exactly once and the j-accumulators are back in their home lanes.  No reduction
//     arithmetic is spent on the j side.
//   * Warps of a CTA work on different j-units in a skewed order (unit = (step + warp) mod units)
//     with one __syncthreads per step, so shared accumulators are never touched by two warps at a
//     time and the summation order is fixed: results are bit-reproducible, no atomics.
// Output: part[slot][n][3]; super-tile (A,B) writes slot B for A's bodies (i side) and slot A for
// B's bodies (j side); every (slot, body) is written exactly once per evaluation and
// nb_kickv_kernel adds the slots in order.
//
// Diagonal super-tiles (A == B): a warp's 32I-block against a 32-block q is evaluated symmetrically
// if q lies above the block, skipped if below (the mirrored visit covers it), and "mixed" if q is one
// of the block's own 32-blocks: all ordered pairs are evaluated, only the i side is kept.
#pragma once
#include "force_tiles.cuh"
#include "sort_staging.cuh"

namespace nbk {

struct SymParams {
    // staged by nb_prep_kernel in the DOUBLED-BLOCK layout: every block of 32 bodies is stored twice in a
    // row (entry of body n, copy h: (n >> 5) * 64 + 32 h + (n & 31)), so that the j-body lane l meets in
    // rotation r sits at block + l + r with no wrap-around arithmetic.  Padding bodies sit far away at
    // distinct places with zero mass.
    const double2 *sxy;          // [2 Npad] (x, y)
    const double2 *szg;          // [2 Npad] (z, G m)
    const int *sthr;             // [2 Npad] hi32(rcrit^2) + 1
    const double *rcrit;         // [N]    exact critical radii (slow path only), indexed by BODY
    const int *perm;             // [Npad] staged position -> body (sorted staging, sort_staging.cuh) or nullptr
    const BlockBound *bnd;       // [nsb]  azimuth / radius / rc bounds of every staged super-block, or nullptr
    // partial accelerations.  Whole grid in one launch (col0 = 0, ncols = nsb): part_i = part_j = [slots, N, 3],
    // stride_i = stride_j = N, goff = 0 -- tile (A, B) writes slot B for A's bodies and slot A for B's.
    // BANDED (large N: the slots of the whole grid would be 24 N^2 / S bytes): one launch per band of ncols tile
    // columns B = col0 .. col0 + ncols - 1; the i sides go to part_i[B - col0][N] and the j sides of the band's bodies to
    // part_j[A][ncols S] (goff = col0 S), both folded into acc by nb_bandsum_kernel before the next band reuses them.
    double *part_i, *part_j;
    long long stride_i, stride_j;
    int goff, col0, ncols;
    int32_t *pairs;              // [cap,2] or nullptr
    unsigned long long *npairs;  // device counter
    long long *status;           // device int64[ST_COUNT]
    long long cap;
    int N;
    int S;      // super-block size: multiple of 128*I and of 128*U
    int nsb;    // super-blocks = Npad / S
    int U;      // 32-blocks per skew unit (S / (32 U) >= 4)
    int xcols;  // TAIL SPLITTING: the strict tiles of the last xcols columns B run as kSymSplit CTAs each, one per
                // part of B's bodies; part q > 0 of column T-1-c writes its i side to the extra slot nsb + c (kSymSplit-1) + q-1
    int kind;   // changeover shape
};

// rotations unrolled in the hot loop: 4 with the encounter test, 2 without (measured)
constexpr int kSymUnrollTest = 4, kSymUnrollFar = 2;
// Tail of the grid: a lone CTA runs hardly faster than one of many, so the end of the launch costs about one CTA
// duration whatever the number of CTAs left.  The tiles launched last are therefore cut into kSymSplit parts along B
// (S / kSymSplit j-bodies each, all of A): short CTAs, and many of them.  The j side of a part goes to slot A as usual
// (its bodies are its own); the i sides of the parts are kSymSplit partial sums for A's bodies: part 0 takes slot B, the
// others one extra slot each per split column (valid for the bodies in front of that column; nb_kickv_kernel knows).
constexpr int kSymSplit = 4;
__host__ __device__ constexpr long long sym_split_tiles(long long T, long long C) { return C * (T - 1) - C * (C - 1) / 2; }
__host__ __device__ constexpr long long sym_grid(long long T, long long C) {
    return T * (T + 1) / 2 + (kSymSplit - 1) * sym_split_tiles(T, C);
}
// CTAs of the launch that covers the tile columns col0 .. col0 + ncols - 1 (banded evaluation, no tail splitting)
__host__ __device__ constexpr long long sym_band_grid(long long col0, long long ncols) {
    return ncols + (col0 + ncols) * (col0 + ncols - 1) / 2 - col0 * (col0 - 1) / 2;
}
__host__ __device__ constexpr int sym_slots(int T, int C) { return T + (kSymSplit - 1) * C; }
__host__ __device__ constexpr size_t sym_smem_bytes(int S) { return (size_t)S * (32 + 32 + 24 + 8) + 16; }

// Exact evaluation of the lane's I pairs against body j (deferred pass; entered by the lanes that
// flagged rotation r, whose fast-path contributions were forced to exactly 0).  Returns the j-side
// contribution in (cx,cy,cz); emit[k] says whether pair k goes on the list.
//   mixed: only the i side is kept by the caller and a pair is emitted from its i < j visit only.
template <int I, bool SORTED>
__device__ __forceinline__ void sym_exact(const SymParams &p, const double2 xy, const double2 zg, const int thrj,
                                          const int j, const bool mixed, const double (&xi)[I], const double (&yi)[I],
                                          const double (&zi)[I], const double (&ngi)[I], const int i0,
                                          double (&ax)[I], double (&ay)[I], double (&az)[I], double &cx, double &cy,
                                          double &cz, bool (&emit)[I]) {
    // i, j are STAGED POSITIONS (the real bodies hold positions 0 .. N-1); with sorted staging perm gives the body
    const double rcj = j < p.N ? p.rcrit[SORTED ? p.perm[j] : j] : 0.0;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = i0 + 32 * k;
        emit[k] = false;
        const bool valid = (i < p.N) && (j < p.N) && (i != j);
        if (!valid) continue;  // padding bodies have zero mass both ways; the self term is skipped
        const double dx = __dsub_rn(xy.x, xi[k]), dy = __dsub_rn(xy.y, yi[k]), dz = __dsub_rn(zg.x, zi[k]);
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        // the body's own threshold word, reloaded from the staged array (kept out of the rotation loop's registers)
        const int thr_i = p.sthr[(size_t)(i >> 5) * 64 + (i & 31)];
        double f;  // W / r^3
        if (__double2hiint(r2) > max(thr_i, thrj)) {
            // flagged only because a lane-mate (say a giant planet) has a large critical radius: this pair is out of
            // reach, W = 1 -- same arithmetic as the rotation loop
            const double y0 = rsqrt_seed(r2);
            const double u = __dmul_rn(y0, y0);
            const double e = __fma_rn(-r2, u, 1.0);
            f = __dmul_rn(__dmul_rn(u, y0), __fma_rn(e, __fma_rn(e, 1.875, 1.5), 1.0));
        } else {
            const double rc = fmax(p.rcrit[SORTED ? p.perm[i] : i], rcj);
            const bool inside = r2 < rc * rc;
            emit[k] = inside && (!mixed || i < j);
            if (r2 == 0.0) {
                // rc == 0 and coincident: contributes 0; counted once per ordered interaction
                if (!inside) status_add(p.status, ST_SINGULAR, mixed ? 1 : 2);
                continue;
            }
            f = weighted_inv_r3(r2, rc, inside, p.kind);
        }
        const double si = zg.y * f, sj = ngi[k] * f;
        ax[k] = __fma_rn(si, dx, ax[k]); ay[k] = __fma_rn(si, dy, ay[k]); az[k] = __fma_rn(si, dz, az[k]);
        cx = __fma_rn(sj, dx, cx); cy = __fma_rn(sj, dy, cy); cz = __fma_rn(sj, dz, cz);
    }
}

// One warp, one block of 32 j-bodies (shared-memory arrays qxy/qzg/qthr of the doubled block: 64
// entries each), 32 rotations.
// On return (bx,by,bz) of lane l hold the sums for j = jbase + l.
//
// The rotation loop is branch-free so that consecutive rotations overlap in the FP64 pipe: a lane
// whose smallest r^2 is within reach of a critical radius (integer test on the high words; always
// true for the self term, r^2 = 0) replaces its rsqrt seeds by 0 -- u = 0, e = 1, r^-3 = 0: its I pairs
// contribute exactly 0 to both sides -- and sets bit r of a mask.  After the 32 rotations the
// (rare) flagged rotations are evaluated exactly, and their j-side contributions are handed to the
// home lanes of the j-bodies.
//
// TEST = false (sorted staging, super-tiles whose arcs are out of each other's reach): no test, no mask, no exact pass.
template <int I, bool PAIRS, bool TEST, bool SORTED>
__device__ __forceinline__ void sym_block(const SymParams &p, const double2 *__restrict__ qxy,
                                          const double2 *__restrict__ qzg, const int *__restrict__ qthr,
                                          const int jbase, const bool mixed, const double (&xi)[I],
                                          const double (&yi)[I], const double (&zi)[I], const double (&ngi)[I],
                                          const int thr_lane, const int i0, double (&ax)[I], double (&ay)[I],
                                          double (&az)[I], double &bx, double &by, double &bz) {
    const int lane = threadIdx.x & 31;
    const int down = (lane + 1) & 31;  // the lane whose j-sums this lane takes over after each rotation
    bx = 0.0; by = 0.0; bz = 0.0;
    unsigned bits = 0u, rbit = 1u;
    const double2 *__restrict__ lxy = qxy + lane;
    const double2 *__restrict__ lzg = qzg + lane;
    const int *__restrict__ lthr = qthr + lane;
#pragma unroll(TEST ? kSymUnrollTest : kSymUnrollFar)
    for (int r = 0; r < 32; ++r) {
        const double2 xy = lxy[r];
        const double2 zg = lzg[r];
        const int thrj = TEST ? lthr[r] : 0;
        double dx[I], dy[I], dz[I], r2[I];
        int mn = 0x7fffffff;
#pragma unroll
        for (int k = 0; k < I; ++k) {
            dx[k] = __dsub_rn(xy.x, xi[k]);
            dy[k] = __dsub_rn(xy.y, yi[k]);
            dz[k] = __dsub_rn(zg.x, zi[k]);
            r2[k] = __fma_rn(dz[k], dz[k], __fma_rn(dy[k], dy[k], __dmul_rn(dx[k], dx[k])));
            if (TEST) mn = min(mn, __double2hiint(r2[k]));
        }
        int kill = 0;
        if (TEST) {
            const bool hit = mn <= max(thr_lane, thrj);
            if (hit) bits |= rbit;
            rbit <<= 1;
            // a flagged lane feeds +inf to the seed: rsqrt(+inf) = +0, so y0 = u = r^-3 = 0 for its I pairs
            kill = hit ? 0x7ff00000 : 0;
        }
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const double y0 = TEST ? rsqrt_seed(__hiloint2double(max(__double2hiint(r2[k]), kill), 0)) : rsqrt_seed(r2[k]);
            const double u = __dmul_rn(y0, y0);                          // exact (y0 has 21 bits)
            const double e = __fma_rn(-r2[k], u, 1.0);                   // 1 - r2 y0^2
            const double q = __fma_rn(e, __fma_rn(e, 1.875, 1.5), 1.0);  // (1-e)^(-3/2), next term < 2^-56
            const double b = __dmul_rn(__dmul_rn(u, y0), q);             // r^-3
            const double si = __dmul_rn(b, zg.y);                        // G m_j / r^3
            const double sj = __dmul_rn(b, ngi[k]);                      // -G m_i / r^3
            if (TEST) {
                // neighbours share one operand (dx, sj, dy, si, dz): measured fastest in the loop with the test
                ax[k] = __fma_rn(si, dx[k], ax[k]);
                bx = __fma_rn(sj, dx[k], bx);
                by = __fma_rn(sj, dy[k], by);
                ay[k] = __fma_rn(si, dy[k], ay[k]);
                az[k] = __fma_rn(si, dz[k], az[k]);
                bz = __fma_rn(sj, dz[k], bz);
            } else {
                // side by side: -1.3 % in the test-free loop
                ax[k] = __fma_rn(si, dx[k], ax[k]);
                ay[k] = __fma_rn(si, dy[k], ay[k]);
                az[k] = __fma_rn(si, dz[k], az[k]);
                bx = __fma_rn(sj, dx[k], bx);
                by = __fma_rn(sj, dy[k], by);
                bz = __fma_rn(sj, dz[k], bz);
            }
        }
        bx = __shfl_sync(0xffffffffu, bx, down);
        by = __shfl_sync(0xffffffffu, by, down);
        bz = __shfl_sync(0xffffffffu, bz, down);
    }
    unsigned any = TEST ? __reduce_or_sync(0xffffffffu, bits) : 0u;
    while (any) {
        const int r = __ffs(any) - 1;
        any &= any - 1u;
        const int src = (lane + r) & 31;
        double cx = 0.0, cy = 0.0, cz = 0.0;
        bool emit[I];
#pragma unroll
        for (int k = 0; k < I; ++k) emit[k] = false;
        if ((bits >> r) & 1u)
            sym_exact<I, SORTED>(p, lxy[r], lzg[r], lthr[r], jbase + src, mixed, xi, yi, zi, ngi, i0, ax, ay, az, cx, cy, cz, emit);
        if (PAIRS) {
#pragma unroll
            for (int k = 0; k < I; ++k) {
                int ib = i0 + 32 * k, jb = jbase + src;
                if (SORTED && emit[k]) { ib = p.perm[ib]; jb = p.perm[jb]; }  // the list holds BODY indices
                pair_append(p.pairs, p.npairs, p.status, p.cap, emit[k], ib, jb);
            }
        }
        // body j = jbase + h met lane (h - r) & 31 in rotation r; its sums live in lane h
        const int from = (lane - r) & 31;
        bx += __shfl_sync(0xffffffffu, cx, from);
        by += __shfl_sync(0xffffffffu, cy, from);
        bz += __shfl_sync(0xffffffffu, cz, from);
    }
}


// The work of one super-tile after B is staged: chunks of A against the blocks of B, then the slot writes.
template <int I, int W, bool PAIRS, bool TEST, bool SORTED>
__device__ __forceinline__ void sym_tile(const SymParams &p, const int A, const int B, const bool diag, const int S,
                                         const volatile int *ti,
                                         const double2 *bxy, const double2 *bzg, const int *bthr, double *jsx, double *jsy,
                                         double *jsz) {
    // ti (shared memory, re-read where needed so that none of it occupies a register across the rotation loops):
    // [0] jS, the number of staged j-bodies (all of B unless the tile is split), [1] position of the first of them,
    // [2] Uq, 32-blocks per skew unit, [3] the slot of the i side
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int nunits = ti[0] / (32 * ti[2]);
    constexpr int kThreads = 32 * W;
    const int nchunks = S / (kThreads * I);
    for (int c = 0; c < nchunks; ++c) {
        const int P = (c * W + w) * I;                  // first 32-block of this warp's i-block within A
        const int i0 = A * S + P * 32 + lane;           // global index of the lane's first i-body
        double xi[I], yi[I], zi[I], ngi[I], ax[I], ay[I], az[I];
        int thr_lane = 0;
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const size_t en = (size_t)((i0 >> 5) + k) * 64 + lane;  // first copy of body i0 + 32 k
            const double2 a = p.sxy[en];
            const double2 b = p.szg[en];
            xi[k] = a.x; yi[k] = a.y; zi[k] = b.x; ngi[k] = -b.y;
            thr_lane = max(thr_lane, p.sthr[en]);
            ax[k] = 0.0; ay[k] = 0.0; az[k] = 0.0;
        }
        for (int step = 0; step < nunits; ++step) {
            int unit = step + w;
            if (unit >= nunits) unit -= nunits;
            const int Uq = ti[2];
            for (int uu = 0; uu < Uq; ++uu) {
                const int q = unit * Uq + uu;  // 32-block of the staged part of B
                bool mixed = false;
                if (diag) {
                    if (q < P) continue;          // the mirrored visit covers it
                    mixed = q < P + I;
                }
                double bx, by, bz;
                sym_block<I, PAIRS, TEST, SORTED>(p, bxy + q * 64, bzg + q * 64, bthr + q * 64, ti[1] + q * 32, mixed, xi, yi, zi,
                                    ngi, thr_lane, i0, ax, ay, az, bx, by, bz);
                if (!mixed) {
                    const int n = q * 32 + lane;
                    jsx[n] += bx; jsy[n] += by; jsz[n] += bz;
                }
            }
            __syncthreads();
        }
        if (diag) {
            // A's bodies are B's bodies: both sides of the diagonal tile go to the same slot
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const int n = P * 32 + 32 * k + lane;
                jsx[n] += ax[k]; jsy[n] += ay[k]; jsz[n] += az[k];
            }
            __syncthreads();
        } else {
            double *out = p.part_i + (size_t)ti[3] * p.stride_i * 3;
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const int i = i0 + 32 * k;
                if (i < p.N) {
                    out[3 * (size_t)i] = ax[k];
                    out[3 * (size_t)i + 1] = ay[k];
                    out[3 * (size_t)i + 2] = az[k];
                }
            }
        }
    }
    // j side (and, on the diagonal, both sides) -> slot A for B's bodies
    double *out = p.part_j + (size_t)A * p.stride_j * 3;
    const int jS = ti[0], j0 = ti[1];
    for (int n = t; n < jS; n += kThreads) {
        const long long g = (long long)j0 + n;
        if (g < p.N) {
            out[3 * (g - p.goff)] = jsx[n];
            out[3 * (g - p.goff) + 1] = jsy[n];
            out[3 * (g - p.goff) + 2] = jsz[n];
        }
    }
}

template <int I, int W, bool PAIRS, int MINB, bool SORTED>
__global__ void __launch_bounds__(32 * W, MINB) nb_force_sym_kernel(const SymParams p) {
    constexpr int kThreads = 32 * W;
    extern __shared__ __align__(16) unsigned char sym_smem[];
    const int S = p.S;
    double2 *bxy = reinterpret_cast<double2 *>(sym_smem);
    double2 *bzg = bxy + 2 * S;
    double *jsx = reinterpret_cast<double *>(bzg + 2 * S);
    double *jsy = jsx + S;
    double *jsz = jsy + S;
    int *bthr = reinterpret_cast<int *>(jsz + S);
    uint64_t *bar = reinterpret_cast<uint64_t *>(bthr + 2 * S);  // S*96 bytes in: 8-byte aligned

    const int t = threadIdx.x;

    // super-tile of this CTA: the diagonal tiles (about half the work each) first -- measured: half-cost tiles at the
    // START take the CTAs of an SM out of lock step, -1.9 % at N = 65536 --, then the strict pairs A < B column by
    // column, the last xcols columns cut into kSymSplit parts each (see kSymSplit)
    const int T = p.nsb;
    const int c1 = p.col0 + p.ncols;                                  // columns of this launch: col0 .. c1 - 1
    const long long first = (long long)p.col0 * (p.col0 - 1) / 2;     // strict tiles in front of the band
    const long long nstrict = (long long)c1 * (c1 - 1) / 2 - first;
    const long long nwhole = nstrict - sym_split_tiles(T, p.xcols);   // strict tiles that run as one CTA (xcols > 0: whole grid only)
    int A, B, part = 0, nparts = 1;
    if ((int)blockIdx.x < p.ncols) {
        A = B = p.col0 + (int)blockIdx.x;
    } else {
        long long idx = (long long)blockIdx.x - p.ncols;
        if (idx >= nwhole) {
            const long long k = idx - nwhole;
            idx = nwhole + k / kSymSplit;
            part = (int)(k % kSymSplit);
            nparts = kSymSplit;
        }
        idx += first;
        B = (int)((1.0 + sqrt(1.0 + 8.0 * (double)idx)) * 0.5);
        while ((long long)B * (B - 1) / 2 > idx) --B;
        while ((long long)(B + 1) * B / 2 <= idx) ++B;
        A = (int)(idx - (long long)B * (B - 1) / 2);
    }
    const int jS = S / nparts, joff = part * jS;
    __shared__ int tinfo[4];
    if (t == 0) {
        tinfo[0] = jS;
        tinfo[1] = B * S + joff;
        tinfo[2] = nparts == 1 ? p.U : (p.U / kSymSplit > 0 ? p.U / kSymSplit : 1);
        tinfo[3] = part == 0 ? B - p.col0 : T + (T - 1 - B) * (kSymSplit - 1) + part - 1;
    }
    const bool diag = (A == B);

    if (t == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const unsigned b16 = (unsigned)jS * 32u, b4 = (unsigned)jS * 8u;
        const size_t first = ((size_t)B * S + joff) * 2;   // doubled-block layout
        mbar_expect_tx(bar, 2u * b16 + b4);
        tma_bulk_g2s(bxy, p.sxy + first, b16, bar);
        tma_bulk_g2s(bzg, p.szg + first, b16, bar);
        tma_bulk_g2s(bthr, p.sthr + first, b4, bar);
    }
    for (int n = t; n < jS; n += kThreads) { jsx[n] = 0.0; jsy[n] = 0.0; jsz[n] = 0.0; }
    __syncthreads();  // barrier initialised and accumulators zeroed before anyone proceeds
    mbar_wait(bar, 0);

    // sorted staging: if the arcs of A and B are out of each other's reach no pair of this super-tile can meet a
    // critical radius -- the whole tile runs without the encounter test
    bool far = false;
    if (SORTED && !diag) {
        const BlockBound ba = p.bnd[A], bb = p.bnd[B];
        far = arcs_are_far(ba.phi_lo, ba.phi_hi, ba.r_min, ba.rc_max, bb.phi_lo, bb.phi_hi, bb.r_min, bb.rc_max);
    }
    if (SORTED && far) sym_tile<I, W, PAIRS, false, SORTED>(p, A, B, diag, S, tinfo, bxy, bzg, bthr, jsx, jsy, jsz);
    else sym_tile<I, W, PAIRS, true, SORTED>(p, A, B, diag, S, tinfo, bxy, bzg, bthr, jsx, jsy, jsz);
}

}  // namespace nbk
