// nb_common.cuh -- shared device-side types and helpers of libnbkick (CUDA path only).
// Nothing here is shared with oracle/ (the CPU checker); see DESIGN.md "independence".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbk {

// One staged j-body, 64 bytes = four 16-byte shared-memory broadcasts.
// Built once per force evaluation by nb_prep_kernel (O(N)), consumed by the O(N^2) tile kernel.
//   gm = G m_j, c1 = 3/2 G m_j, c2 = 15/8 G m_j : coefficients of the rsqrt-cube correction
//   polynomial G m_j (1 + 3/2 e + 15/8 e^2)     (see force_tiles.cuh)
//   rc2 = rcrit_j^2, rc = rcrit_j                (pair test / changeover)
struct __align__(16) JRec {
    double x, y, z, gm;
    double c1, c2, rc2, rc;
};
static_assert(sizeof(JRec) == 64, "JRec must be 64 bytes");

// fp32 range: r^2 below this (r < 1e-15 in the caller's units) goes to the exact fp64 path whatever the critical radii -- the cube
// of an fp32 reciprocal square root would leave the fp32 range long before the fp64 kernel has any difficulty
constexpr float kDsMinR2 = 1.0e-30f;

// stages body `pos` (position in the doubled-block layout) for the Newton-III mixed-precision kernel (force_symds.cuh):
// double-single position (xh + xl), fl32(G m), and rc^2 rounded up with a 2^-18 margin; called by nb_prep_kernel
__device__ __forceinline__ void symds_stage(float4 *sa, float4 *sb, const int pos, const double x, const double y, const double z,
                                            const double gm, const double rc2) {
    const float xh = __double2float_rn(x), yh = __double2float_rn(y), zh = __double2float_rn(z);
    const float xl = __double2float_rn(x - (double)xh), yl = __double2float_rn(y - (double)yh), zl = __double2float_rn(z - (double)zh);
    const float thr = fmaxf(__double2float_ru(rc2) * 1.0000038f, kDsMinR2);
    const size_t en = (size_t)(pos >> 5) * 64 + (pos & 31);
    // (high, low) of a coordinate sit side by side: one packed fp32x2 add forms both partial differences
    const float4 a = make_float4(xh, xl, yh, yl), b = make_float4(zh, zl, __double2float_rn(gm), thr);
    sa[en] = a; sa[en + 32] = a;
    sb[en] = b; sb[en + 32] = b;
}

// One staged j-body of the one-sided mixed-precision kernel on double-single positions (force_mixed.cuh, nb_force_mixedds_kernel):
// 32 bytes, (high, low) of a coordinate side by side.  Padding records sit far away with zero mass.
struct __align__(16) JRecDs {
    float xh, xl, yh, yl;
    float zh, zl, gm, thr;   // thr = rc^2 (1 + 2^-18) rounded up
};
static_assert(sizeof(JRecDs) == 32, "JRecDs must be 32 bytes");
__device__ __forceinline__ JRecDs make_jrecds(const double x, const double y, const double z, const double gm, const double rc2) {
    JRecDs r;
    r.xh = __double2float_rn(x); r.yh = __double2float_rn(y); r.zh = __double2float_rn(z);
    r.xl = __double2float_rn(x - (double)r.xh); r.yl = __double2float_rn(y - (double)r.yh); r.zl = __double2float_rn(z - (double)r.zh);
    r.gm = __double2float_rn(gm); r.thr = fmaxf(__double2float_ru(rc2) * 1.0000038f, kDsMinR2);
    return r;
}

constexpr int kForceThreads = 128;  // threads per force CTA
constexpr int kTileJ = 128;         // j-bodies per shared-memory stage (8 KB)
constexpr int kStages = 4;          // TMA ring depth (2 tiles in flight ahead of the consumer)
constexpr int kBodyThreads = 256;   // threads per CTA of the O(N) kernels
constexpr double kFarJ = 1.0e30;    // padding j-records sit here with zero mass
constexpr double kFarI = -1.0e30;   // padding i-lanes sit here; their sums are discarded

// status counters (device int64[8]); meanings in include/nbkick.h nb_status
enum { ST_PAIR_DROPPED = 0, ST_KEPLER_FAIL = 1, ST_NONFINITE = 2, ST_SINGULAR = 3, ST_GROUP_SKIPPED = 4, ST_BS_FAIL = 5, ST_MIDPOINT_FAIL = 6, ST_ABSORBED = 7, ST_COUNT = 8 };

__device__ __forceinline__ void status_add(long long *status, int which, long long n) {
    atomicAdd(reinterpret_cast<unsigned long long *>(status + which), static_cast<unsigned long long>(n));
}

// Deterministic block-wide sum of three doubles (fixed tree, blockDim.x == kBodyThreads).
// Every thread returns the same totals.
__device__ __forceinline__ void block_sum3(double &a, double &b, double &c, double *sm /* [3*kBodyThreads] */) {
    const int t = threadIdx.x;
    sm[t] = a;
    sm[kBodyThreads + t] = b;
    sm[2 * kBodyThreads + t] = c;
    __syncthreads();
#pragma unroll
    for (int s = kBodyThreads / 2; s > 0; s >>= 1) {
        if (t < s) {
            sm[t] += sm[t + s];
            sm[kBodyThreads + t] += sm[kBodyThreads + t + s];
            sm[2 * kBodyThreads + t] += sm[2 * kBodyThreads + t + s];
        }
        __syncthreads();
    }
    a = sm[0];
    b = sm[kBodyThreads];
    c = sm[2 * kBodyThreads];
    __syncthreads();
}

// Sum of per-block momentum partials part[nblk,3] in a fixed order: every CTA that calls this
// gets bit-identical totals (thread t adds blocks t, t+256, ... in order; then the fixed tree).
__device__ __forceinline__ void reduce_partials3(const double *__restrict__ part, int nblk, double &sx, double &sy,
                                                 double &sz, double *sm) {
    double a = 0.0, b = 0.0, c = 0.0;
    for (int k = threadIdx.x; k < nblk; k += kBodyThreads) {
        a += part[3 * k];
        b += part[3 * k + 1];
        c += part[3 * k + 2];
    }
    block_sum3(a, b, c, sm);
    sx = a;
    sy = b;
    sz = c;
}

}  // namespace nbk
