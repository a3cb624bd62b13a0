// groups.cuh -- independent close-encounter groups ("finding independent close encounter
// groups and integrating them independently"): the connected components of the graph
// whose vertices are the bodies and whose edges are the pairs of the list nb_kick / nb_step emit.
//
// Integer work throughout; every output is unique (label = smallest index of the group, groups ordered
// by label, members ascending), so results are bit-exact whatever the order in which threads run:
//   1. hooking:   lock-free union-find over the edges; a root is only ever hooked under a SMALLER root
//                 (atomicCAS), so parent[i] <= i always holds and the final root of a component is its
//                 smallest index; finds use path halving (any ancestor is a valid parent: plain stores).
//   2. compress:  label[i] = root(i); size[root]++ (integer atomics: deterministic totals).
//   3. offsets:   exclusive scan in index order over the leaders (label[i] == i, size >= 2) of
//                 (1, size[i]) -> group number and first slot of every group.
//   4. members:   small groups: scatter with an atomic cursor, then a rank sort inside the segment;
//                 groups of >= kGiant members: one CTA per group compacts the indicator
//                 (label[i] == L) over all bodies in index order (no O(size^2) work).
#pragma once
#include "nb_common.cuh"

namespace nbk {

constexpr int kGrpThreads = 256;
constexpr int kGrpScanBlock = 1024;  // bodies per block of the offset scan
constexpr int kGiant = 2048;         // groups at least this large are compacted by an indicator scan

struct GroupScratch {
    int *parent;    // [N]
    int *size;      // [N]  members of the group led by i (valid at roots)
    int *segstart;  // [N]  first slot of the group led by i
    int *cursor;    // [N]  scatter cursor of the group led by i
    int *tmp;       // [N]  members before the rank sort
    int *bsum;      // [2 * nblk] per-block (leaders, members)
    int *giant;     // [N / kGiant + 2] leaders of giant groups
    int *ngiant;    // [1]
};

__device__ __forceinline__ int grp_find(volatile int *parent, int x) {
    int p = parent[x];
    while (p != x) {
        const int gp = parent[p];
        if (gp != p) parent[x] = gp;  // path halving: gp is an ancestor of x, and stays one
        x = p;
        p = gp;
    }
    return x;
}

__global__ void __launch_bounds__(kGrpThreads) nb_grp_init_kernel(GroupScratch s, int *__restrict__ label,
                                                                 int *__restrict__ members, int *__restrict__ gstart,
                                                                 long long *__restrict__ gstat, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i < N) { s.parent[i] = i; s.size[i] = 0; s.cursor[i] = 0; s.segstart[i] = 0; s.tmp[i] = -1; members[i] = -1; label[i] = i; }
    if (i < N / 2 + 2) gstart[i] = -1;
    if (i < 4) gstat[i] = 0;
    if (i == 0) *s.ngiant = 0;
}

// Optional edge filter of the hooking kernel (merge.cuh): an edge counts only if the two bodies are in
// contact, r_ij < f (R_i + R_j); x == nullptr: every row is an edge.
struct GroupFilter {
    const double *x;       // [N,3] or nullptr
    const double *radius;  // [N]
    double f;
    long long *nhit;       // rows that passed the filter
};

__global__ void __launch_bounds__(kGrpThreads) nb_grp_hook_kernel(GroupScratch s, const int2 *__restrict__ pairs,
                                                                 const long long *__restrict__ npairs, long long cap,
                                                                 int N, long long *__restrict__ gstat,
                                                                 long long *__restrict__ status, const GroupFilter flt) {
    long long n = *npairs;
    if (n > cap) n = cap;
    if (n < 0) n = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) gstat[3] = n;
    volatile int *parent = s.parent;
    for (long long e = (long long)blockIdx.x * kGrpThreads + threadIdx.x; e < n; e += (long long)gridDim.x * kGrpThreads) {
        const int2 ab = pairs[e];
        if (ab.x < 0 || ab.y < 0 || ab.x >= N || ab.y >= N || ab.x == ab.y) { status_add(status, ST_NONFINITE, 1); continue; }
        if (flt.x != nullptr) {
            const double dx = flt.x[3 * (size_t)ab.y] - flt.x[3 * (size_t)ab.x];
            const double dy = flt.x[3 * (size_t)ab.y + 1] - flt.x[3 * (size_t)ab.x + 1];
            const double dz = flt.x[3 * (size_t)ab.y + 2] - flt.x[3 * (size_t)ab.x + 2];
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            const double sr = flt.f * (flt.radius[ab.x] + flt.radius[ab.y]);
            if (!(r2 < sr * sr)) continue;
            atomicAdd(reinterpret_cast<unsigned long long *>(flt.nhit), 1ull);
        }
        int ra = ab.x, rb = ab.y;
        while (true) {
            ra = grp_find(parent, ra);
            rb = grp_find(parent, rb);
            if (ra == rb) break;
            const int hi = ra > rb ? ra : rb, lo = ra > rb ? rb : ra;
            if (atomicCAS(s.parent + hi, hi, lo) == hi) break;  // hi was still a root: now under the smaller root
        }
    }
}

__global__ void __launch_bounds__(kGrpThreads) nb_grp_compress_kernel(GroupScratch s, int *__restrict__ label, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= N) return;
    int r = i;
    while (true) { const int p = s.parent[r]; if (p == r) break; r = p; }
    label[i] = r;
    atomicAdd(s.size + r, 1);
}

// exclusive block scan of two ints per thread (blockDim.x == kGrpScanBlock); returns the block totals
__device__ __forceinline__ void grp_block_scan2(int &a, int &b, int &ta, int &tb, int *sm /* [2 * 32 + 2] */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int xa = __shfl_up_sync(0xffffffffu, ia, o), xb = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += xa; ib += xb; }
    }
    if (lane == 31) { sm[w] = ia; sm[32 + w] = ib; }
    __syncthreads();
    if (w == 0) {
        int wa = sm[lane], wb = sm[32 + lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int xa = __shfl_up_sync(0xffffffffu, wa, o), xb = __shfl_up_sync(0xffffffffu, wb, o);
            if (lane >= o) { wa += xa; wb += xb; }
        }
        if (lane == 31) { sm[64] = wa; sm[65] = wb; }
        sm[lane] = wa - sm[lane];        // exclusive warp offsets
        sm[32 + lane] = wb - sm[32 + lane];
    }
    __syncthreads();
    a = ia - a + sm[w];
    b = ib - b + sm[32 + w];
    ta = sm[64];
    tb = sm[65];
    __syncthreads();
}

// per-block totals of (leaders, members of listed groups) over kGrpScanBlock bodies
__global__ void __launch_bounds__(kGrpScanBlock) nb_grp_blocksum_kernel(GroupScratch s, const int *__restrict__ label, int N) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    const bool lead = i < N && label[i] == i && s.size[i] >= 2;
    int a = lead ? 1 : 0, b = lead ? s.size[i] : 0, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    if (threadIdx.x == 0) { s.bsum[2 * blockIdx.x] = ta; s.bsum[2 * blockIdx.x + 1] = tb; }
}

// one CTA: exclusive scan of the per-block totals in place; totals to gstat
__global__ void __launch_bounds__(kGrpScanBlock) nb_grp_topscan_kernel(GroupScratch s, int nblk, int *__restrict__ gstart,
                                                                      long long *__restrict__ gstat) {
    __shared__ int sm[66];
    int run_a = 0, run_b = 0;
    for (int base = 0; base < nblk; base += kGrpScanBlock) {
        const int k = base + threadIdx.x;
        int a = k < nblk ? s.bsum[2 * k] : 0, b = k < nblk ? s.bsum[2 * k + 1] : 0, ta, tb;
        grp_block_scan2(a, b, ta, tb, sm);
        if (k < nblk) { s.bsum[2 * k] = a + run_a; s.bsum[2 * k + 1] = b + run_b; }
        run_a += ta;
        run_b += tb;
    }
    if (threadIdx.x == 0) { gstat[0] = run_a; gstat[1] = run_b; gstart[run_a] = run_b; }
}

// group number and first slot of every leader; largest group; list of giant groups
__global__ void __launch_bounds__(kGrpScanBlock) nb_grp_offsets_kernel(GroupScratch s, const int *__restrict__ label, int N,
                                                                      int *__restrict__ gstart, long long *__restrict__ gstat) {
    __shared__ int sm[66];
    const int i = blockIdx.x * kGrpScanBlock + threadIdx.x;
    const bool lead = i < N && label[i] == i && s.size[i] >= 2;
    const int sz = lead ? s.size[i] : 0;
    int a = lead ? 1 : 0, b = sz, ta, tb;
    grp_block_scan2(a, b, ta, tb, sm);
    if (lead) {
        const int g = a + s.bsum[2 * blockIdx.x], start = b + s.bsum[2 * blockIdx.x + 1];
        gstart[g] = start;
        s.segstart[i] = start;
        s.cursor[i] = start;
        atomicMax(reinterpret_cast<unsigned long long *>(gstat + 2), (unsigned long long)sz);
        if (sz >= kGiant) s.giant[atomicAdd(s.ngiant, 1)] = i;
    }
}

// small groups: members in arrival order
__global__ void __launch_bounds__(kGrpThreads) nb_grp_scatter_kernel(GroupScratch s, const int *__restrict__ label, int N) {
    const int i = blockIdx.x * kGrpThreads + threadIdx.x;
    if (i >= N) return;
    const int L = label[i], sz = s.size[L];
    if (sz < 2 || sz >= kGiant) return;
    s.tmp[atomicAdd(s.cursor + L, 1)] = i;
}

// small groups: rank sort inside the segment (members ascending)
__global__ void __launch_bounds__(kGrpThreads) nb_grp_ranksort_kernel(GroupScratch s, const int *__restrict__ label,
                                                                     const long long *__restrict__ gstat,
                                                                     int *__restrict__ members) {
    const long long p = (long long)blockIdx.x * kGrpThreads + threadIdx.x;
    if (p >= gstat[1]) return;
    const int b = s.tmp[p];
    if (b < 0) return;  // slot of a giant group
    const int L = label[b], start = s.segstart[L], sz = s.size[L];
    int rank = 0;
    for (int q = start; q < start + sz; ++q) rank += (s.tmp[q] < b) ? 1 : 0;
    members[start + rank] = b;
}

// giant groups: one CTA per group compacts the indicator (label[i] == L) over all bodies in index order
__global__ void __launch_bounds__(kGrpScanBlock) nb_grp_giant_kernel(GroupScratch s, const int *__restrict__ label, int N,
                                                                    int *__restrict__ members) {
    __shared__ int sm[66];
    const int ng = *s.ngiant;
    for (int k = blockIdx.x; k < ng; k += gridDim.x) {
        const int L = s.giant[k];
        int run = s.segstart[L];
        for (int base = L; base < N; base += kGrpScanBlock) {  // no member precedes the leader
            const int i = base + threadIdx.x;
            const bool in = i < N && label[i] == L;
            int a = in ? 1 : 0, b = 0, ta, tb;
            grp_block_scan2(a, b, ta, tb, sm);
            (void)tb;
            if (in) members[run + a] = i;
            run += ta;
        }
    }
}

}  // namespace nbk
