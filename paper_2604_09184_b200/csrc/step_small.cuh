// step_small.cuh -- whole steps of the integrator in ONE cooperative launch, for small N (at N = 2048 a force
// evaluation is ~4 us of arithmetic and a step was five launches of 6-11 us each; the paper itself notes that GPUs lose at
// small N to kernel overhead).
//
// One persistent grid of 128-thread CTAs runs, per step, the four phases of the multi-launch path (nbkick.cu step_impl)
//     drift (first H_C half-shift + Kepler)  |  prep (second half-shift, Eq. 7, staging)  |  force tiles  |  slot sum + kick
// separated by grid-wide barriers: each phase needs a sum over ALL bodies of the previous one (total momentum for H_C,
// every staged j-record, every partial acceleration).  The phases execute the SAME device functions on the SAME virtual
// blocks as the stand-alone kernels -- a 256-body block of the O(N) kernels is taken by 128 threads, two bodies each, with
// the 256-leaf reduction tree reproduced -- so the results are bit-identical to the multi-launch path (tested), and the
// summation order stays fixed: deterministic, no fp64 atomics.
#pragma once
#include <cooperative_groups.h>

#include "body_kernels.cuh"
#include "force_tiles.cuh"

namespace nbk {

struct SmallStepParams {
    PrepParams pp;       // x, v, m, rcrit, jrec, ... (mv_in is set per phase)
    ForceParams fp;
    double *acc;         // [N,3]
    double *mvA, *mvB;   // momentum partials [ceil(N/256), 3]
    double mu, dt, hk, dtc;
    int nsteps;          // steps this launch runs
    int last_nhalf;      // half-kicks applied after the last evaluation (1: the run ends; 2: another launch follows)
    int iblocks, nsplit; // force geometry
    int nblk;            // 256-body blocks
};

// block-wide sum of three values per LEAF for 256 leaves held by 128 threads (leaf t and leaf t + 128 in thread t):
// the tree of block_sum3 (nb_common.cuh), level by level.  Every thread returns the totals.
__device__ __forceinline__ void small_sum3(const double (&a)[2], const double (&b)[2], const double (&c)[2], double &sa,
                                           double &sb, double &sc, double *sm /* [3 * 256] */) {
    const int t = threadIdx.x;
    sm[t] = a[0]; sm[t + 128] = a[1];
    sm[256 + t] = b[0]; sm[256 + t + 128] = b[1];
    sm[512 + t] = c[0]; sm[512 + t + 128] = c[1];
    __syncthreads();
#pragma unroll
    for (int s = 128; s > 0; s >>= 1) {
        if (t < s) {
            sm[t] += sm[t + s];
            sm[256 + t] += sm[256 + t + s];
            sm[512 + t] += sm[512 + t + s];
        }
        __syncthreads();
    }
    sa = sm[0]; sb = sm[256]; sc = sm[512];
    __syncthreads();
}

// reduce_partials3 (nb_common.cuh) for 256 leaves on 128 threads: leaf l adds blocks l, l + 256, ... in order
__device__ __forceinline__ void small_reduce_partials3(const double *__restrict__ part, const int nblk, double &sx, double &sy,
                                                       double &sz, double *sm) {
    double a[2] = {0.0, 0.0}, b[2] = {0.0, 0.0}, c[2] = {0.0, 0.0};
#pragma unroll
    for (int h = 0; h < 2; ++h)
        for (int k = threadIdx.x + 128 * h; k < nblk; k += 256) {
            a[h] += part[3 * k];
            b[h] += part[3 * k + 1];
            c[h] += part[3 * k + 2];
        }
    small_sum3(a, b, c, sx, sy, sz, sm);
}

template <int I, bool PAIRS>
__global__ void __launch_bounds__(kForceThreads, I == 4 ? 3 : 4) nb_step_small_kernel(const SmallStepParams q) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ __align__(128) JRec ring[kStages][kTileJ];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ __align__(8) uint64_t empty[kStages];
    double *sm = reinterpret_cast<double *>(&ring[0][0]);   // the O(N) phases reuse the ring as reduction scratch (6 KB)
    const int t = threadIdx.x;
    const int cover = max(q.pp.N, q.pp.Njpad);
    const int nprep = (cover + kBodyThreads - 1) / kBodyThreads;

    for (int step = 0; step < q.nsteps; ++step) {
        // ---- C(dt/2) A(dt): first half-shift + Kepler drift; momentum partials of the drifted velocities -> mvB
        {
            double sx, sy, sz;
            small_reduce_partials3(q.mvA, q.nblk, sx, sy, sz, sm);
            sx /= q.pp.M_star; sy /= q.pp.M_star; sz /= q.pp.M_star;
            for (int vb = blockIdx.x; vb < q.nblk; vb += gridDim.x) {
                double a[2], b[2], c[2];
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    drift_one(q.pp.x, const_cast<double *>(q.pp.v), q.pp.m, q.pp.N, q.mu, q.dt, true, q.dtc, sx, sy, sz, true,
                              q.pp.status, nullptr, vb * kBodyThreads + t + 128 * h, a[h], b[h], c[h]);
                double pa, pb, pc;
                small_sum3(a, b, c, pa, pb, pc, sm);
                if (t == 0) { q.mvB[3 * vb] = pa; q.mvB[3 * vb + 1] = pb; q.mvB[3 * vb + 2] = pc; }
            }
        }
        grid.sync();
        // ---- C(dt/2) folded into prep: second half-shift, Eq. 7, staging of the j-records
        {
            double sx, sy, sz;
            small_reduce_partials3(q.mvB, q.nblk, sx, sy, sz, sm);
            sx /= q.pp.M_star; sy /= q.pp.M_star; sz /= q.pp.M_star;
            PrepParams pp = q.pp;
            pp.mv_in = q.mvB;
            for (int vb = blockIdx.x; vb < nprep; vb += gridDim.x) {
                prep_one(pp, vb * kBodyThreads + t, sx, sy, sz);
                prep_one(pp, vb * kBodyThreads + t + 128, sx, sy, sz);
            }
        }
        grid.sync();
        // ---- force tiles: virtual CTA (i-block, j-split), exactly the stand-alone kernel's
        for (int w = blockIdx.x; w < q.iblocks * q.nsplit; w += gridDim.x) {
            // the ring was written through the generic proxy (reduction scratch) and is about to be written by TMA
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();   // nobody still reads the ring (scratch or the previous work item)
            force_tiles_cta<I, PAIRS, true>(q.fp, w % q.iblocks, w / q.iblocks, ring, full, empty);
            __syncthreads();
            if (t == 0) {
#pragma unroll
                for (int s = 0; s < kStages; ++s) {
                    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&full[s])) : "memory");
                    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&empty[s])) : "memory");
                }
            }
        }
        grid.sync();
        // ---- slot sum, B(dt/2) [+ B(dt/2) of the next step], momentum partials of the kicked velocities -> mvA
        {
            const int nhalf = (step + 1 < q.nsteps) ? 2 : q.last_nhalf;
            for (int vb = blockIdx.x; vb < q.nblk; vb += gridDim.x) {
                double a[2], b[2], c[2];
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    kickv_one(q.fp.part, q.nsplit, q.acc, const_cast<double *>(q.pp.v), q.pp.m, q.pp.N, q.hk, nhalf, true, nullptr,
                              vb * kBodyThreads + t + 128 * h, a[h], b[h], c[h]);
                double pa, pb, pc;
                small_sum3(a, b, c, pa, pb, pc, sm);
                if (t == 0) { q.mvA[3 * vb] = pa; q.mvA[3 * vb + 1] = pb; q.mvA[3 * vb + 2] = pc; }
            }
        }
        if (step + 1 < q.nsteps) grid.sync();
    }
}

}  // namespace nbk
