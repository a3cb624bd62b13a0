// force_symds.cuh -- Newton-III form of the MIXED-PRECISION kick (Fig. 1 contrasts FP32
// and FP64 runs of the same code on both of its GPUs).  What is computed is the H_B kick of force_sym.cuh (PAPER.md:86
// Eq. 5, 98) and the same pair list; what changes is the arithmetic of the pairs that are out of reach of every critical
// radius (all but ~1e-6 of them), which runs ENTIRELY on the FP32 pipe:
//   * positions are staged as double-single, x = xh + xl with xh = fl32(x), xl = fl32(x - xh) (48 bits together);
//     dx = fl(fl(xjh - xih) + fl(xjl - xil)) carries a relative error of ~2.5 * 2^-24 OF THE DIFFERENCE ITSELF: the
//     cancellation of nearby positions happens between the high parts (exactly, by Sterbenz, when they are close) and
//     the low parts restore what fl32(x) lost -- no fp64 subtraction, no conversion;
//   * r^2, MUFU.RSQ, its cube, the two mass products, six FFMA: 22 FP32 instructions per UNORDERED pair, both sides
//     served (the fp64 kernel: 20 FP64 instructions, on a pipe half as wide);
//   * the j-sums travel through the warp as in force_sym.cuh; fp32 sums over ONE visit of a 32-body block (32 terms on
//     the i side, 64 + 64 on the j side), fp64 from there on;
//   * packed fp32x2 instructions (FADD2 / FMUL2 / FFMA2) wherever two values take the same operation: the kernel is
//     bound by instruction issue.
// Pairs whose fp32 r^2 is within reach of a critical radius (margin 2^-18: far above the fp32 rounding of r^2), and
// every self term, are killed in the fp32 loop (r^2 replaced by +inf, so rsqrt gives 0: they contribute exactly 0 to both sides) and
// re-evaluated by the EXACT fp64 pass of force_sym.cuh (sym_exact) from the fp64 staged arrays: the changeover weight,
// the pair test r^2 < rc^2 and the pair list are bit-identical to the fp64 kernel's.  Tolerance reading: DESIGN.md S25.
// Same super-tile decomposition, skewed unit order, slots, determinism and sorted staging (test-free far tiles) as
// nb_force_sym_kernel, banded evaluation included; no tail splitting.
#pragma once
#include "force_sym.cuh"

namespace nbk {

struct SymDsParams {
    SymParams sp;      // fp64 staged arrays (exact pass), slots, pair list, geometry, perm / bnd of the sorted staging: as nb_force_sym_kernel
    const float4 *sa;  // [2 Npad] (xh, xl, yh, yl)                                  doubled-block layout
    const float4 *sb;  // [2 Npad] (zh, zl, fl32(G m), rc^2 (1 + 2^-18) rounded up)
};

constexpr int kDsI = 4;   // i-bodies per lane
__host__ __device__ constexpr size_t symds_smem_bytes(int S) { return (size_t)S * (32 + 32 + 24) + 16; }

__device__ __forceinline__ float rsqrt_f32(const float a) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a));
    return y;
}

// One warp, one block of 32 j-bodies, 32 rotations in fp32; then the exact fp64 pass for the flagged rotations.
// On return lane l holds in (bx,by,bz) the fp64 sums for j = jbase + l; the i-side sums of the visit are ADDED to AX/AY/AZ.
// The kernel is bound by instruction issue, not by the FP32 pipe (ncu: issue slots 79 % busy, FMA pipe 62 %, with scalar
// instructions), so the arithmetic is written with the packed fp32x2 instructions of sm_100 (FADD2 / FMUL2 / FFMA2: two
// lanes per issue slot, each rounded as the scalar instruction would): the (high, low) partial differences of a coordinate
// in one FADD2, everything after the differences on two i-bodies at a time.  nxa/nya/nza: the lane's i-bodies, NEGATED,
// as (high, low) pairs; ngi2: -G m_i of bodies (2g, 2g+1).
// TEST = false (sorted staging, super-tiles whose arcs are out of each other's reach): no pre-filter, no kill, no exact pass.
template <bool PAIRS, bool TEST, bool SORTED>
__device__ __forceinline__ void symds_block(const SymDsParams &p, const float4 *__restrict__ qa, const float4 *__restrict__ qb,
                                            const int jbase, const bool mixed, const float2 (&nxa)[kDsI], const float2 (&nya)[kDsI],
                                            const float2 (&nza)[kDsI], const float2 (&ngi2)[kDsI / 2], const float thr_lane,
                                            const int i0, double (&AX)[kDsI], double (&AY)[kDsI], double (&AZ)[kDsI], double &bx,
                                            double &by, double &bz) {
    constexpr int I = kDsI, H = kDsI / 2;
    const int lane = threadIdx.x & 31;
    const int down = (lane + 1) & 31;
    float2 ax[H], ay[H], az[H];                       // i-side sums of bodies (2g, 2g+1)
    float2 fx = make_float2(0.0f, 0.0f), fy = fx, fz = fx;   // travelling j-side sums: even and odd i-bodies apart
#pragma unroll
    for (int g = 0; g < H; ++g) { ax[g] = make_float2(0.0f, 0.0f); ay[g] = ax[g]; az[g] = ax[g]; }
    unsigned bits = 0u, rbit = 1u;
    const float4 *__restrict__ la = qa + lane;
    const float4 *__restrict__ lb = qb + lane;
    const float kInf = __int_as_float(0x7f800000);
#pragma unroll(TEST ? 4 : 8)
    for (int r = 0; r < 32; ++r) {
        const float4 a = la[r];                       // (xh, xl, yh, yl)
        const float4 b = lb[r];                       // (zh, zl, G m, threshold)
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
        float kill = 0.0f;
        if (TEST) {
            float mn = fminf(r2[0].x, r2[0].y);
#pragma unroll
            for (int g = 1; g < H; ++g) mn = fminf(mn, fminf(r2[g].x, r2[g].y));
            const bool hit = mn <= fmaxf(thr_lane, b.w);
            if (hit) bits |= rbit;
            rbit <<= 1;
            kill = hit ? kInf : 0.0f;                 // rsqrt(+inf) = 0: a flagged lane's I pairs contribute exactly 0
        }
        const float2 gmj = make_float2(b.z, b.z);
#pragma unroll
        for (int g = 0; g < H; ++g) {
            const float2 y0 = TEST ? make_float2(rsqrt_f32(fmaxf(r2[g].x, kill)), rsqrt_f32(fmaxf(r2[g].y, kill)))
                                   : make_float2(rsqrt_f32(r2[g].x), rsqrt_f32(r2[g].y));
            const float2 y3 = __fmul2_rn(__fmul2_rn(y0, y0), y0);
            const float2 si = __fmul2_rn(y3, gmj);            // G m_j / r^3
            const float2 sj = __fmul2_rn(y3, ngi2[g]);        // -G m_i / r^3
            ax[g] = __ffma2_rn(si, dx[g], ax[g]); ay[g] = __ffma2_rn(si, dy[g], ay[g]); az[g] = __ffma2_rn(si, dz[g], az[g]);
            fx = __ffma2_rn(sj, dx[g], fx); fy = __ffma2_rn(sj, dy[g], fy); fz = __ffma2_rn(sj, dz[g], fz);
        }
        fx.x = __shfl_sync(0xffffffffu, fx.x, down); fx.y = __shfl_sync(0xffffffffu, fx.y, down);
        fy.x = __shfl_sync(0xffffffffu, fy.x, down); fy.y = __shfl_sync(0xffffffffu, fy.y, down);
        fz.x = __shfl_sync(0xffffffffu, fz.x, down); fz.y = __shfl_sync(0xffffffffu, fz.y, down);
    }
    bx = (double)fx.x + (double)fx.y; by = (double)fy.x + (double)fy.y; bz = (double)fz.x + (double)fz.y;
#pragma unroll
    for (int g = 0; g < H; ++g) {
        AX[2 * g] += (double)ax[g].x; AY[2 * g] += (double)ay[g].x; AZ[2 * g] += (double)az[g].x;
        AX[2 * g + 1] += (double)ax[g].y; AY[2 * g + 1] += (double)ay[g].y; AZ[2 * g + 1] += (double)az[g].y;
    }

    if (!TEST) return;
    unsigned any = __reduce_or_sync(0xffffffffu, bits);
    if (any == 0u) return;
    // exact fp64 pass (rare): the lane's i-bodies from the fp64 staged arrays
    const SymParams &sp = p.sp;
    double xi[I], yi[I], zi[I], ngd[I];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const size_t en = (size_t)((i0 >> 5) + k) * 64 + lane;
        const double2 u = sp.sxy[en], w = sp.szg[en];
        xi[k] = u.x; yi[k] = u.y; zi[k] = w.x; ngd[k] = -w.y;
    }
    while (any) {
        const int r = __ffs(any) - 1;
        any &= any - 1u;
        const int src = (lane + r) & 31;
        double cx = 0.0, cy = 0.0, cz = 0.0;
        bool emit[I];
#pragma unroll
        for (int k = 0; k < I; ++k) emit[k] = false;
        if ((bits >> r) & 1u) {
            const int j = jbase + src;
            const size_t ej = (size_t)(j >> 5) * 64 + (j & 31);
            sym_exact<I, SORTED>(sp, sp.sxy[ej], sp.szg[ej], sp.sthr[ej], j, mixed, xi, yi, zi, ngd, i0, AX, AY, AZ, cx, cy, cz, emit);
        }
        if (PAIRS) {
#pragma unroll
            for (int k = 0; k < I; ++k) {
                int ib = i0 + 32 * k, jb = jbase + src;
                if (SORTED && emit[k]) { ib = sp.perm[ib]; jb = sp.perm[jb]; }   // the list holds BODY indices
                pair_append(sp.pairs, sp.npairs, sp.status, sp.cap, emit[k], ib, jb);
            }
        }
        const int from = (lane - r) & 31;
        bx += __shfl_sync(0xffffffffu, cx, from);
        by += __shfl_sync(0xffffffffu, cy, from);
        bz += __shfl_sync(0xffffffffu, cz, from);
    }
}

// One CTA of W warps per super-tile (A, B), A <= B, S = 128 W bodies a side: B staged once (two TMA bulk copies of the
// float4 arrays), B's fp64 sums in shared memory, A's bodies in registers four per lane; diagonal tiles first.
template <int W, bool PAIRS, bool SORTED>
__global__ void __launch_bounds__(32 * W, 16 / W) nb_force_symds_kernel(const SymDsParams p) {
    constexpr int I = kDsI, kThreads = 32 * W;
    extern __shared__ __align__(16) unsigned char symds_smem[];
    const SymParams &sp = p.sp;
    const int S = sp.S;
    float4 *ba = reinterpret_cast<float4 *>(symds_smem);
    float4 *bb = ba + 2 * S;
    double *jsx = reinterpret_cast<double *>(bb + 2 * S);
    double *jsy = jsx + S;
    double *jsz = jsy + S;
    uint64_t *bar = reinterpret_cast<uint64_t *>(jsz + S);
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;

    // tile of this CTA among the columns col0 .. col0 + ncols - 1 of the launch (the whole grid, or one band of the banded
    // evaluation: force_sym.cuh SymParams): the diagonal tiles first, then the strict pairs A < B column by column
    int A, B;
    if ((int)blockIdx.x < sp.ncols) {
        A = B = sp.col0 + (int)blockIdx.x;
    } else {
        const long long idx = (long long)blockIdx.x - sp.ncols + (long long)sp.col0 * (sp.col0 - 1) / 2;
        B = (int)((1.0 + sqrt(1.0 + 8.0 * (double)idx)) * 0.5);
        while ((long long)B * (B - 1) / 2 > idx) --B;
        while ((long long)(B + 1) * B / 2 <= idx) ++B;
        A = (int)(idx - (long long)B * (B - 1) / 2);
    }
    const bool diag = (A == B);
    if (t == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const unsigned bytes = (unsigned)S * 32u;            // 2 S float4
        const size_t first = (size_t)B * S * 2;
        mbar_expect_tx(bar, 2u * bytes);
        tma_bulk_g2s(ba, p.sa + first, bytes, bar);
        tma_bulk_g2s(bb, p.sb + first, bytes, bar);
    }
    for (int n = t; n < S; n += kThreads) { jsx[n] = 0.0; jsy[n] = 0.0; jsz[n] = 0.0; }
    __syncthreads();
    mbar_wait(bar, 0);

    // sorted staging: arcs of A and B out of each other's reach => no pair of this super-tile can meet a critical radius
    bool far = false;
    if (SORTED && !diag) {
        const BlockBound ba_ = sp.bnd[A], bb_ = sp.bnd[B];
        far = arcs_are_far(ba_.phi_lo, ba_.phi_hi, ba_.r_min, ba_.rc_max, bb_.phi_lo, bb_.phi_hi, bb_.r_min, bb_.rc_max);
    }
    const int nunits = S / (32 * sp.U);
    const int nchunks = S / (kThreads * I);
    for (int c = 0; c < nchunks; ++c) {
        const int P = (c * W + w) * I;
        const int i0 = A * S + P * 32 + lane;
        float2 nxa[I], nya[I], nza[I], ngi2[I / 2];
        float ngi[I];
        double AX[I], AY[I], AZ[I];
        float thr_lane = 0.0f;
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const size_t en = (size_t)((i0 >> 5) + k) * 64 + lane;
            const float4 a = p.sa[en], b = p.sb[en];
            nxa[k] = make_float2(-a.x, -a.y); nya[k] = make_float2(-a.z, -a.w); nza[k] = make_float2(-b.x, -b.y);
            ngi[k] = -b.z;
            thr_lane = fmaxf(thr_lane, b.w);
            AX[k] = 0.0; AY[k] = 0.0; AZ[k] = 0.0;
        }
#pragma unroll
        for (int g = 0; g < I / 2; ++g) ngi2[g] = make_float2(ngi[2 * g], ngi[2 * g + 1]);
        for (int step = 0; step < nunits; ++step) {
            int unit = step + w;
            if (unit >= nunits) unit -= nunits;
            for (int uu = 0; uu < sp.U; ++uu) {
                const int q = unit * sp.U + uu;
                bool mixed = false;
                if (diag) {
                    if (q < P) continue;
                    mixed = q < P + I;
                }
                double bx, by, bz;
                if (SORTED && far)
                    symds_block<PAIRS, false, SORTED>(p, ba + q * 64, bb + q * 64, B * S + q * 32, mixed, nxa, nya, nza, ngi2, thr_lane, i0, AX, AY, AZ, bx, by, bz);
                else
                    symds_block<PAIRS, true, SORTED>(p, ba + q * 64, bb + q * 64, B * S + q * 32, mixed, nxa, nya, nza, ngi2, thr_lane, i0, AX, AY, AZ, bx, by, bz);
                if (!mixed) {
                    const int n = q * 32 + lane;
                    jsx[n] += bx; jsy[n] += by; jsz[n] += bz;
                }
            }
            __syncthreads();
        }
        if (diag) {
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const int n = P * 32 + 32 * k + lane;
                jsx[n] += AX[k]; jsy[n] += AY[k]; jsz[n] += AZ[k];
            }
            __syncthreads();
        } else {
            double *out = sp.part_i + (size_t)(B - sp.col0) * sp.stride_i * 3;
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const int i = i0 + 32 * k;
                if (i < sp.N) { out[3 * (size_t)i] = AX[k]; out[3 * (size_t)i + 1] = AY[k]; out[3 * (size_t)i + 2] = AZ[k]; }
            }
        }
    }
    double *out = sp.part_j + (size_t)A * sp.stride_j * 3;
    for (int n = t; n < S; n += kThreads) {
        const long long g = (long long)B * S + n;
        if (g < sp.N) { out[3 * (g - sp.goff)] = jsx[n]; out[3 * (g - sp.goff) + 1] = jsy[n]; out[3 * (g - sp.goff) + 2] = jsz[n]; }
    }
}

}  // namespace nbk
