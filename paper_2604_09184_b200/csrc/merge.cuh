// merge.cuh -- perfect merging of colliding bodies ("N-body simulations often treat collisions as
// perfect mergers"; radii may be inflated by a constant factor f; reading S21).
//   collision   r_ij < f (R_i + R_j) for a row (i, j) of the pair list, strict, decided in fp64 on r^2 -- tested
//               inside the hooking kernel of groups.cuh (GroupFilter), so no second list is written;
//   clusters    connected components of the contact graph (groups.cuh: label, ordered member lists);
//   merger      the smallest index survives: m <- sum m_k, x <- sum m_k x_k / sum m_k, v likewise (members in
//               index order: deterministic), R <- cbrt(sum R_k^3); all-massless clusters keep the survivor's x, v;
//   compaction  stable partition of x, v, m, R by the alive flag (exclusive scan in index order).
#pragma once
#include "groups.cuh"

namespace nbk {

// one thread per cluster
__global__ void __launch_bounds__(kGrpThreads) nb_mrg_merge_kernel(double *__restrict__ x, double *__restrict__ v,
                                                                  double *__restrict__ m, double *__restrict__ R,
                                                                  const int *__restrict__ members,
                                                                  const int *__restrict__ gstart,
                                                                  const long long *__restrict__ gstat,
                                                                  int *__restrict__ alive) {
    const long long g = (long long)blockIdx.x * kGrpThreads + threadIdx.x;
    if (g >= gstat[0]) return;
    const int g0 = gstart[g], g1 = gstart[g + 1];
    const int s = members[g0];
    double mt = 0.0, mx0 = 0.0, mx1 = 0.0, mx2 = 0.0, mv0 = 0.0, mv1 = 0.0, mv2 = 0.0, vol = 0.0;
    for (int k = g0; k < g1; ++k) {
        const int b = members[k];
        const double mb = m[b], rb = R[b];
        // unfused multiply / add in index order: the sums are the definition's, bit for bit
        mt = __dadd_rn(mt, mb);
        mx0 = __dadd_rn(mx0, __dmul_rn(mb, x[3 * (size_t)b]));
        mx1 = __dadd_rn(mx1, __dmul_rn(mb, x[3 * (size_t)b + 1]));
        mx2 = __dadd_rn(mx2, __dmul_rn(mb, x[3 * (size_t)b + 2]));
        mv0 = __dadd_rn(mv0, __dmul_rn(mb, v[3 * (size_t)b]));
        mv1 = __dadd_rn(mv1, __dmul_rn(mb, v[3 * (size_t)b + 1]));
        mv2 = __dadd_rn(mv2, __dmul_rn(mb, v[3 * (size_t)b + 2]));
        vol = __dadd_rn(vol, __dmul_rn(__dmul_rn(rb, rb), rb));
        if (k > g0) alive[b] = 0;
    }
    if (mt > 0.0) {
        x[3 * (size_t)s] = mx0 / mt; x[3 * (size_t)s + 1] = mx1 / mt; x[3 * (size_t)s + 2] = mx2 / mt;
        v[3 * (size_t)s] = mv0 / mt; v[3 * (size_t)s + 1] = mv1 / mt; v[3 * (size_t)s + 2] = mv2 / mt;
    }
    m[s] = mt;
    R[s] = cbrt(vol);
}

__global__ void __launch_bounds__(kGrpThreads) nb_mrg_alive_init_kernel(int *__restrict__ alive, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i < N) alive[i] = 1;
}

// per-block totals of (alive, alive among the first n_active)
__global__ void __launch_bounds__(kGrpScanBlock) nb_mrg_blocksum_kernel(const int *__restrict__ alive, int N, int n_active,
                                                                       int *__restrict__ bsum) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    int a = (i < N && alive[i]) ? 1 : 0, b = (a && i < n_active) ? 1 : 0, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    if (threadIdx.x == 0) { bsum[2 * blockIdx.x] = ta; bsum[2 * blockIdx.x + 1] = tb; }
}

__global__ void __launch_bounds__(kGrpScanBlock) nb_mrg_topscan_kernel(int *__restrict__ bsum, int nblk, int N,
                                                                      const long long *__restrict__ gstat,
                                                                      const long long *__restrict__ ncoll,
                                                                      long long *__restrict__ mstat) {
    __shared__ int sm[66];
    int run_a = 0, run_b = 0;
    for (int base = 0; base < nblk; base += kGrpScanBlock) {
        const int k = base + threadIdx.x;
        int a = k < nblk ? bsum[2 * k] : 0, b = k < nblk ? bsum[2 * k + 1] : 0, ta, tb;
        grp_block_scan2(a, b, ta, tb, sm);
        if (k < nblk) { bsum[2 * k] = a + run_a; bsum[2 * k + 1] = b + run_b; }
        run_a += ta;
        run_b += tb;
    }
    if (threadIdx.x == 0) { mstat[0] = run_a; mstat[1] = *ncoll; mstat[2] = N - run_a; mstat[3] = run_b; (void)gstat; }
}

// alive bodies to their new slots of the temporary arrays t8[8][N_old-sized stride]
__global__ void __launch_bounds__(kGrpScanBlock) nb_mrg_scatter_kernel(const double *__restrict__ x, const double *__restrict__ v,
                                                                      const double *__restrict__ m, const double *__restrict__ R,
                                                                      const int *__restrict__ alive, const int *__restrict__ bsum,
                                                                      int N, double *__restrict__ t8) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    const bool live = i < N && alive[i];
    int a = live ? 1 : 0, b = 0, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    (void)tb;
    if (live) {
        const size_t d = (size_t)(a + bsum[2 * blockIdx.x]);
#pragma unroll
        for (int c = 0; c < 3; ++c) { t8[8 * d + c] = x[3 * (size_t)i + c]; t8[8 * d + 3 + c] = v[3 * (size_t)i + c]; }
        t8[8 * d + 6] = m[i];
        t8[8 * d + 7] = R[i];
    }
}

__global__ void __launch_bounds__(kGrpThreads) nb_mrg_copyback_kernel(double *__restrict__ x, double *__restrict__ v,
                                                                     double *__restrict__ m, double *__restrict__ R,
                                                                     const double *__restrict__ t8,
                                                                     const long long *__restrict__ mstat) {
    const long long d = (long long)blockIdx.x * kGrpThreads + threadIdx.x;
    if (d >= mstat[0]) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) { x[3 * d + c] = t8[8 * d + c]; v[3 * d + c] = t8[8 * d + 3 + c]; }
    m[d] = t8[8 * d + 6];
    R[d] = t8[8 * d + 7];
}

}  // namespace nbk
