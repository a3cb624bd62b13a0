// sort_staging.cuh -- azimuthal ordering of the bodies staged for the Newton-III kernel (force_sym.cuh).
//
// The rotation loop must test every pair against its critical radius because bodies with neighbouring
// indices sit anywhere in the disk.  Staging the bodies sorted by azimuth makes every super-block of S bodies
// an arc, and two arcs whose angular gap g satisfies 2 r_min sin(g/2) > rc_max cannot hold an encounter
// pair: the CTA of such a super-tile (all but the ~3 T near-diagonal ones of T(T+1)/2) runs rotation loops
// without the test.  Only the STAGED copies are permuted; x, v, acc, the pair list and everything the
// caller sees keep the caller's indexing (perm maps back).
//
//   key      bucket of atan2(y, x) (a few bodies per bucket)            nb_sort_key_kernel
//   offsets  exclusive scan of the histogram                             nb_sort_scan_kernel
//   scatter  bodies to their bucket segment in arrival order             nb_sort_scatter_kernel
//   rank     ascending body index inside the bucket -> deterministic     nb_sort_rank_kernel
//            perm[pos] = body, pos_of[body] = pos; padding bodies keep the tail positions N .. Npad-1
//   bounds   per super-block of staged positions: azimuth interval, smallest cylindrical radius, largest
//            critical radius (computed from the staged data itself)     nb_sort_bounds_kernel
#pragma once
#include "groups.cuh"  // grp_block_scan2

namespace nbk {

struct SortScratch {
    int *key;     // [N]  bucket of each body
    int *hist;    // [NB + 1] bucket counts, then exclusive offsets
    int *cursor;  // [NB]
    int *tmp;     // [N]
    int *perm;    // [Npad] staged position -> body (>= N: padding)
    int *pos_of;  // [N]    body -> staged position
    int NB;
};

struct BlockBound {
    double phi_lo, phi_hi, r_min, rc_max;  // a block of padding only: r_min = +inf
};

__global__ void __launch_bounds__(kGrpThreads) nb_sort_clear_kernel(SortScratch s, int N, int Npad) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i <= s.NB) s.hist[i] = 0;
    if (i < s.NB) s.cursor[i] = 0;
    if (i >= N && i < Npad) s.perm[i] = i;  // padding keeps the tail
}

__global__ void __launch_bounds__(kGrpThreads) nb_sort_key_kernel(SortScratch s, const double *__restrict__ x, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= N) return;
    const double phi = atan2(x[3 * (size_t)i + 1], x[3 * (size_t)i]);  // (-pi, pi]; NaN falls into bucket 0
    int b = (int)((phi + 3.14159265358979323846) * (s.NB / 6.28318530717958647692));
    if (!(b >= 0)) b = 0;
    if (b >= s.NB) b = s.NB - 1;
    s.key[i] = b;
    atomicAdd(s.hist + b, 1);
}

// one CTA: exclusive scan of hist[0 .. NB) in place, hist[NB] = total
__global__ void __launch_bounds__(kGrpScanBlock) nb_sort_scan_kernel(SortScratch s) {
    __shared__ int sm[66];
    int run = 0;
    for (int base = 0; base < s.NB; base += kGrpScanBlock) {
        const int k = base + threadIdx.x;
        int a = k < s.NB ? s.hist[k] : 0, b = 0, ta, tb;
        grp_block_scan2(a, b, ta, tb, sm);
        (void)tb;
        if (k < s.NB) s.hist[k] = a + run;
        run += ta;
    }
    if (threadIdx.x == 0) s.hist[s.NB] = run;
}

__global__ void __launch_bounds__(kGrpThreads) nb_sort_scatter_kernel(SortScratch s, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= N) return;
    const int b = s.key[i];
    s.tmp[s.hist[b] + atomicAdd(s.cursor + b, 1)] = i;
}

__global__ void __launch_bounds__(kGrpThreads) nb_sort_rank_kernel(SortScratch s, int N) {
    const int p = blockIdx.x * kGrpThreads + threadIdx.x;
    if (p >= N) return;
    const int i = s.tmp[p], b = s.key[i];
    const int lo = s.hist[b], hi = s.hist[b + 1];
    int rank = 0;
    for (int q = lo; q < hi; ++q) rank += (s.tmp[q] < i) ? 1 : 0;
    s.perm[lo + rank] = i;
    s.pos_of[i] = lo + rank;
}

// one CTA per super-block of S staged positions (doubled-block arrays)
__global__ void __launch_bounds__(kGrpThreads) nb_sort_bounds_kernel(const double2 *__restrict__ sxy, const int *__restrict__ perm,
                                                                    const double *__restrict__ rcrit, int N, int S,
                                                                    BlockBound *__restrict__ bnd) {
    __shared__ double red[4][kGrpThreads / 32];
    const int sb = blockIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double lo = 1e300, hi = -1e300, rmin = INFINITY, rc = 0.0;
    for (int k = threadIdx.x; k < S; k += kGrpThreads) {
        const int pos = sb * S + k, body = perm[pos];
        if (body < N) {
            const double2 xy = sxy[(size_t)(pos >> 5) * 64 + (pos & 31)];
            const double phi = atan2(xy.y, xy.x);
            lo = fmin(lo, phi); hi = fmax(hi, phi);
            rmin = fmin(rmin, sqrt(xy.x * xy.x + xy.y * xy.y));
            rc = fmax(rc, rcrit[body]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        rmin = fmin(rmin, __shfl_xor_sync(0xffffffffu, rmin, o));
        rc = fmax(rc, __shfl_xor_sync(0xffffffffu, rc, o));
    }
    if (lane == 0) { red[0][w] = lo; red[1][w] = hi; red[2][w] = rmin; red[3][w] = rc; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < kGrpThreads / 32; ++k) {
            lo = fmin(lo, red[0][k]); hi = fmax(hi, red[1][k]); rmin = fmin(rmin, red[2][k]); rc = fmax(rc, red[3][k]);
        }
        BlockBound b; b.phi_lo = lo; b.phi_hi = hi; b.r_min = rmin; b.rc_max = rc; bnd[sb] = b;
    }
}

// true if no body of arc a can be within reach of a body of arc b: the chord between two points at cylindrical
// radii >= r and azimuths at least g apart is >= 2 r sin(g/2) >= r g (1 - g^2/24) for g <= 1 (and > 0.95 r beyond)
__device__ __forceinline__ bool arcs_are_far(const double a_lo, const double a_hi, const double a_r, const double a_rc,
                                             const double b_lo, const double b_hi, const double b_r, const double b_rc) {
    const double kTwoPiS = 6.28318530717958647692;
    if (!(a_r < 1e299) || !(b_r < 1e299)) return true;  // an arc of padding only
    double g1 = b_lo - a_hi, g2 = a_lo - b_hi;          // gap going one way round, and the other
    if (g1 < 0.0) g1 += kTwoPiS;
    if (g2 < 0.0) g2 += kTwoPiS;
    if (a_lo <= b_hi && b_lo <= a_hi) return false;     // the intervals overlap
    const double g = fmin(g1, g2);
    const double r = fmin(a_r, b_r);
    const double chord = g <= 1.0 ? r * g * (1.0 - g * g * (1.0 / 24.0)) : 0.95 * r;
    return chord > fmax(a_rc, b_rc) * 1.00001;          // the integer pre-filter reaches 2^-20 beyond rc^2
}

}  // namespace nbk
