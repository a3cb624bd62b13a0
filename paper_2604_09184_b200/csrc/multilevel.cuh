// multilevel.cuh -- multi-level changeover ("introducing higher-level changeover functions ... the
// symplectic integrator reduces the time step level by level for the affected bodies.  Only the last level is then
// performed with the inner direct integrator.  Every level needs again a smooth changeover function"; DESIGN.md
// reading S23): the hybrid split of PAPER.md:84-86 (Eq. 4, 5) applied again to H_A, level after level.
//
// With W_k(r) = W(r; rc_k,ij), rc_k,i = max(hill_i, vel_i / 2^k) (Eq. 7 with the level's time step dt / 2^k), and
// Omega_l = prod_{k<=l} [1 - W_k], the bodies of the step's pair list P_0 are advanced over dt by
//     advance(l, tau):  l == L: Bulirsch-Stoer (encounter.cuh) over tau for the groups of P_L, pair weight Omega_L
//                       else twice, h = tau / 2:  P_{l+1} = pairs of P_l closer than rc_{l+1} now
//                                                 kick h/2 with weight Omega_l W_{l+1} over P_l
//                                                 bodies of P_l not in P_{l+1}: Kepler drift h;  advance(l + 1, h)
//                                                 kick h/2 over P_l
//
// Data: the pair list becomes a per-body adjacency (CSR, partners ascending: every sum has a fixed order, no fp64
// atomics, bit-reproducible); each slot carries `depth` = the deepest level the pair is listed at (the nested lists
// P_0 >= P_1 >= ... as ONE array, no compaction); each body carries bdepth = max over its slots.  A pair is seen from
// both ends; both ends take the same decision (r^2 is formed from the same squares, rc_ij is symmetric).
// One thread per body throughout; O(|P_0|) work per kick, 2^(l+1) + 1 kicks at level l.
#pragma once
#include "encounter.cuh"    // one_minus_weight
#include "force_tiles.cuh"  // changeover_weight
#include "groups.cuh"
#include "kepler.cuh"

namespace nbk {

constexpr int kMaxLevels = 8;  // intermediate levels L (time step dt / 2^L at the innermost)

struct MlScratch {
    int *deg;      // [N]      pairs per body
    int *off;      // [N + 1]  first slot of every body
    int *cur;      // [N]      fill cursor
    int *bdepth;   // [N]      deepest level the body is listed at (-1: in no pair)
    int *adj_tmp;  // [2 cap]  partners in arrival order
    int *own;      // [2 cap]  body that owns the slot
    int *adj;      // [2 cap]  partners, ascending inside a body's segment
    signed char *depth;  // [2 cap] deepest level the pair of the slot is listed at
    int *bsum;     // [ceil(N / 1024) + 1] block totals of the offset scan
    long long cap; // rows of the pair list that can be held
};

struct MlParams {
    double *x, *v;               // [N,3]
    const double *m;             // [N]
    const double *hill, *vel;    // [N] the two terms of Eq. 7: rc_k = max(hill, vel / 2^k)
    MlScratch s;
    long long *status;
    double G, mu;
    int N, kind, L;
};

// ---- adjacency (once per step) ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(kGrpThreads) nb_ml_clear_kernel(MlScratch s, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i < N) { s.deg[i] = 0; s.cur[i] = 0; s.bdepth[i] = -1; }
}

__global__ void __launch_bounds__(kGrpThreads) nb_ml_degree_kernel(MlScratch s, const int2 *__restrict__ pairs,
                                                                  const long long *__restrict__ npairs, long long cap, int N,
                                                                  long long *status) {
    long long n = *npairs;
    if (n > cap) n = cap;
    if (n > s.cap) n = s.cap;
    for (long long e = (long long)blockIdx.x * kGrpThreads + threadIdx.x; e < n; e += (long long)gridDim.x * kGrpThreads) {
        const int2 ab = pairs[e];
        if (ab.x < 0 || ab.y < 0 || ab.x >= N || ab.y >= N || ab.x == ab.y) continue;  // counted by the group kernels
        atomicAdd(s.deg + ab.x, 1);
        atomicAdd(s.deg + ab.y, 1);
    }
    (void)status;
}

// exclusive scan of deg -> off (three launches: block totals, top scan, offsets)
__global__ void __launch_bounds__(kGrpScanBlock) nb_ml_scan1_kernel(MlScratch s, int N) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    int a = i < N ? s.deg[i] : 0, b = 0, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    if (threadIdx.x == 0) s.bsum[blockIdx.x] = ta;
}
__global__ void __launch_bounds__(kGrpScanBlock) nb_ml_scan2_kernel(MlScratch s, int nblk, int N) {
    __shared__ int sm[66];
    int run = 0;
    for (int base = 0; base < nblk; base += kGrpScanBlock) {
        const int k = base + threadIdx.x;
        int a = k < nblk ? s.bsum[k] : 0, b = 0, ta, tb;
        grp_block_scan2(a, b, ta, tb, sm);
        if (k < nblk) s.bsum[k] = a + run;
        run += ta;
    }
    if (threadIdx.x == 0) s.off[N] = run;
}
__global__ void __launch_bounds__(kGrpScanBlock) nb_ml_scan3_kernel(MlScratch s, int N) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    int a = i < N ? s.deg[i] : 0, b = 0, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    if (i < N) s.off[i] = a + s.bsum[blockIdx.x];
}

__global__ void __launch_bounds__(kGrpThreads) nb_ml_fill_kernel(MlScratch s, const int2 *__restrict__ pairs,
                                                                const long long *__restrict__ npairs, long long cap, int N) {
    long long n = *npairs;
    if (n > cap) n = cap;
    if (n > s.cap) n = s.cap;
    for (long long e = (long long)blockIdx.x * kGrpThreads + threadIdx.x; e < n; e += (long long)gridDim.x * kGrpThreads) {
        const int2 ab = pairs[e];
        if (ab.x < 0 || ab.y < 0 || ab.x >= N || ab.y >= N || ab.x == ab.y) continue;
        const int sa = s.off[ab.x] + atomicAdd(s.cur + ab.x, 1);
        const int sb = s.off[ab.y] + atomicAdd(s.cur + ab.y, 1);
        s.adj_tmp[sa] = ab.y; s.own[sa] = ab.x;
        s.adj_tmp[sb] = ab.x; s.own[sb] = ab.y;
    }
}

// one thread per slot: rank of the partner inside its body's segment (a pair is listed once, so partners are distinct)
__global__ void __launch_bounds__(kGrpThreads) nb_ml_sort_kernel(MlScratch s, int N) {
    const long long nslots = s.off[N];
    for (long long q = (long long)blockIdx.x * kGrpThreads + threadIdx.x; q < nslots; q += (long long)gridDim.x * kGrpThreads) {
        const int i = s.own[q], b = s.adj_tmp[q];
        const int lo = s.off[i], hi = s.off[i + 1];
        int rank = 0;
        for (int t = lo; t < hi; ++t) rank += (s.adj_tmp[t] < b) ? 1 : 0;
        s.adj[lo + rank] = b;
        s.depth[lo + rank] = 0;       // everything starts in P_0
        if (q == lo) s.bdepth[i] = 0;
    }
}

// ---- the operators of a level ----------------------------------------------------------------------------------
// r^2 exactly as the definition writes it (the listing decision r^2 < rc^2 is an integer-valued result)
__device__ __forceinline__ double ml_r2(const double dx, const double dy, const double dz) {
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}
// level l: [detect] P_{l+1} among the slots of P_l, then napply kicks of h with weight Omega_l W_{l+1} over P_l
// (napply = 2: the closing kick of one substep and the opening kick of the next share the accelerations; two roundings).
template <bool DETECT>
__global__ void __launch_bounds__(kGrpThreads) nb_ml_kick_kernel(const MlParams p, const int l, const double h, const int napply) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= p.N) return;
    if (p.s.bdepth[i] < l) return;   // not in P_l
    const int lo = p.s.off[i], hi = p.s.off[i + 1];
    const double xi = p.x[3 * (size_t)i], yi = p.x[3 * (size_t)i + 1], zi = p.x[3 * (size_t)i + 2];
    const double hill_i = p.hill[i], vel_i = p.vel[i];
    const double sc_next = ldexp(1.0, -(l + 1));
    double ax = 0.0, ay = 0.0, az = 0.0;
    int bd = -1;
    for (int q = lo; q < hi; ++q) {
        int dq = p.s.depth[q];
        if (dq < l) { bd = max(bd, dq); continue; }   // listed at a shallower level only
        const int j = p.s.adj[q];
        const double dx = p.x[3 * (size_t)j] - xi, dy = p.x[3 * (size_t)j + 1] - yi, dz = p.x[3 * (size_t)j + 2] - zi;
        const double r2 = ml_r2(dx, dy, dz);
        const double hill = fmax(hill_i, p.hill[j]), vel = fmax(vel_i, p.vel[j]);
        const double rc_next = fmax(hill, vel * sc_next);
        if (DETECT) {
            dq = (r2 < rc_next * rc_next) ? l + 1 : l;
            p.s.depth[q] = (signed char)dq;
        }
        bd = max(bd, dq);
        if (r2 == 0.0) continue;
        const double id = rsqrt_fast(r2);
        const double r = sqrt_from_rsqrt(r2, id);
        double w = 1.0, sc = 1.0;
        for (int k = 0; k <= l && w != 0.0; ++k, sc *= 0.5) w *= one_minus_weight(r, fmax(hill, vel * sc), p.kind);
        if (w == 0.0) continue;
        w *= (r < rc_next) ? changeover_weight(r, rc_next, p.kind) : 1.0;
        if (w == 0.0) continue;
        const double f = p.G * p.m[j] * w * (id * id * id);
        ax += f * dx; ay += f * dy; az += f * dz;
    }
    if (DETECT) p.s.bdepth[i] = bd;
    double vx = p.v[3 * (size_t)i], vy = p.v[3 * (size_t)i + 1], vz = p.v[3 * (size_t)i + 2];
    for (int a = 0; a < napply; ++a) { vx = vx + h * ax; vy = vy + h * ay; vz = vz + h * az; }
    p.v[3 * (size_t)i] = vx; p.v[3 * (size_t)i + 1] = vy; p.v[3 * (size_t)i + 2] = vz;
}

// Kepler drift over h of the bodies whose deepest listing is exactly level l (at the innermost level: of the bodies the
// direct solver does not take, flag == 0: groups beyond its cap)
__global__ void __launch_bounds__(kGrpThreads) nb_ml_drift_kernel(const MlParams p, const int l, const double h,
                                                                 const int *__restrict__ taken) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= p.N) return;
    if (p.s.bdepth[i] != l) return;
    if (taken != nullptr && taken[i] != 0) return;
    double X0 = p.x[3 * (size_t)i], X1 = p.x[3 * (size_t)i + 1], X2 = p.x[3 * (size_t)i + 2];
    double V0 = p.v[3 * (size_t)i], V1 = p.v[3 * (size_t)i + 1], V2 = p.v[3 * (size_t)i + 2];
    if (kepler_elliptic_fast(X0, X1, X2, V0, V1, V2, p.mu, h) != 0) {
        double X[3] = {X0, X1, X2}, V[3] = {V0, V1, V2};
        if (kepler_universal(X, V, p.mu, h) != 0) status_add(p.status, ST_KEPLER_FAIL, 1);
        X0 = X[0]; X1 = X[1]; X2 = X[2]; V0 = V[0]; V1 = V[1]; V2 = V[2];
    }
    p.x[3 * (size_t)i] = X0; p.x[3 * (size_t)i + 1] = X1; p.x[3 * (size_t)i + 2] = X2;
    p.v[3 * (size_t)i] = V0; p.v[3 * (size_t)i + 1] = V1; p.v[3 * (size_t)i + 2] = V2;
}

// union-find hooking over the slots listed at the innermost level (the edges of P_L); groups.cuh does the rest
__global__ void __launch_bounds__(kGrpThreads) nb_ml_hook_kernel(GroupScratch g, const MlScratch s, const int L, int N,
                                                                long long *__restrict__ gstat) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= N) return;
    if (s.bdepth[i] < L) return;
    volatile int *parent = g.parent;
    int cnt = 0;
    for (int q = s.off[i]; q < s.off[i + 1]; ++q) {
        if (s.depth[q] < L) continue;
        const int j = s.adj[q];
        if (j < i) continue;          // each edge once
        ++cnt;
        int ra = i, rb = j;
        while (true) {
            ra = grp_find(parent, ra);
            rb = grp_find(parent, rb);
            if (ra == rb) break;
            const int hi = ra > rb ? ra : rb, lo = ra > rb ? rb : ra;
            if (atomicCAS(g.parent + hi, hi, lo) == hi) break;
        }
    }
    if (cnt) atomicAdd(reinterpret_cast<unsigned long long *>(gstat + 3), (unsigned long long)cnt);
}

// bodies in no pair of the step's list are the only ones the plain drift kernel moves
__global__ void __launch_bounds__(kGrpThreads) nb_ml_listed_kernel(const MlScratch s, int N, int *__restrict__ listed) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i < N) listed[i] = s.bdepth[i] >= 0 ? 1 : 0;
}

}  // namespace nbk
