// encounter.cuh -- H_A with close encounters (Eq. 4: Kepler terms + pair terms weighted by
// [1 - K]; "a direct solver is needed which propagates the involved bodies through the close
// encounter phase ... must not necessarily be symplectic"; "finding independent close
// encounter groups and integrating them independently").
//
// One CTA per group (groups.cuh), one thread per member.  Equations of motion (weight on the force,
// DESIGN.md reading S3, so that kick + this = the full Newtonian pair force; rc held fixed):
//     dx_i/dt = v_i
//     dv_i/dt = -G M_star x_i / r_i^3 + sum_{j in group, j != i} G m_j [1 - W(r_ij; rc_ij)] (x_j - x_i) / r_ij^3
// Integrator (reading S19): Bulirsch-Stoer -- modified midpoint with 2, 4, ..., 16 substeps, polynomial
// extrapolation in h^2, at most 8 columns; column error = max over members of |dx|^2/|x|^2 and
// |dv|^2/max(|v|^2, mu/|x|), accepted at <= tol^2; accepted in <= 6 columns: h *= 1.3, in 8: h *= 0.55,
// rejected: h /= 2; the first trial step is the whole interval.  Every thread of the CTA takes the same
// decisions (the error is a CTA-wide maximum), so the control flow is uniform.
#pragma once
#include "kepler.cuh"  // rcp_fast, rsqrt_fast, sqrt_from_rsqrt (MUFU seed + one third-order correction, ~1 ulp)
#include "nb_common.cuh"

namespace nbk {

constexpr int kBsCols = 8;
constexpr int kMaxGroup = 1024;  // larger groups are left to the Kepler drift and counted (NB_MAX_GROUP)

// 1 - W(r; rc): the complement of the kick weight, formed directly (no cancellation near W = 1)
__device__ __forceinline__ double one_minus_weight(const double r, const double rc, const int kind) {
    if (!(r < rc)) return 0.0;
    const double t0 = r - 0.1 * rc;
    if (t0 <= 0.0) return 1.0;
    const double y = t0 * rcp_fast(0.9 * rc);
    if (y >= 1.0) return 0.0;
    const double z = 1.0 - y;
    return kind == 1 ? z * z * z * (1.0 + y * (3.0 + 6.0 * y)) : (z * z) * rcp_fast(2.0 * y * y - 2.0 * y + 1.0);
}

// Acceleration of a body at q = (x, y, z) whose critical radius has the two terms (my_hill, my_vel): star term plus
// the pair terms of the n members whose positions / G m / radius terms sit in the given (shared-memory) arrays;
// `self` is skipped.  Level radii rc_k = max(hill, vel / 2^k) (multilevel.cuh); the pair weight is the product over
// k < nlev of [1 - W(r; rc_k,ij)] -- nlev = 1 with vel = 0: Eq. 4 as printed, rc = hill.
// No IEEE divide or sqrt on the common path (latency is what a small group pays for).
__device__ __forceinline__ void enc_accel(const double qx, const double qy, const double qz, const double my_hill,
                                          const double my_vel, const int self, const int n, const double *__restrict__ px,
                                          const double *__restrict__ py, const double *__restrict__ pz,
                                          const double *__restrict__ sgm, const double *__restrict__ shill,
                                          const double *__restrict__ svel, const int nlev, const double mu, const int kind,
                                          double &ax, double &ay, double &az, const bool ghost = false) {
    const double r2 = (qx * qx + qy * qy) + qz * qz;
    const double ir = rsqrt_fast(r2);
    const double s = -mu * (ir * ir * ir);
    ax = s * qx; ay = s * qy; az = s * qz;
    if (ghost) return;   // absorbed by a collision (reading S26): takes no part in the encounter, feels only the star
    for (int j = 0; j < n; ++j) {
        if (j == self || sgm[j] == 0.0) continue;        // a massless member (semi-active mode) pulls on nobody
        const double dx = px[j] - qx, dy = py[j] - qy, dz = pz[j] - qz;
        const double d2 = (dx * dx + dy * dy) + dz * dz;
        const double hill = fmax(my_hill, shill[j]), vel = fmax(my_vel, svel[j]);
        const double rc0 = fmax(hill, vel);
        if (!(d2 < rc0 * rc0) || d2 == 0.0) continue;    // 1 - W_0 = 0 outside rc; coincident: no direction
        const double id = rsqrt_fast(d2);
        const double d = sqrt_from_rsqrt(d2, id);
        double w = one_minus_weight(d, rc0, kind), sc = 0.5;
        for (int k = 1; k < nlev && w != 0.0; ++k, sc *= 0.5) w *= one_minus_weight(d, fmax(hill, vel * sc), kind);
        if (w == 0.0) continue;
        const double tt = sgm[j] * w * (id * id * id);
        ax += tt * dx; ay += tt * dy; az += tt * dz;
    }
}

// 1 / ((n_c / n_{c-m})^2 - 1) of the Aitken-Neville extrapolation, n_k = 2k
__device__ __forceinline__ double bs_weight(const int c, const int mc) {
    const double ratio = (double)(2 * c) / (double)(2 * (c - mc));
    return 1.0 / (ratio * ratio - 1.0);
}

struct EncParams {
    double *x, *v;            // [N,3] in/out (members only)
    const double *m, *rcrit;  // [N]; rcrit: the critical radius, or its Hill term when rc_vel is given
    const double *rc_vel;     // [N] velocity term of Eq. 7 (multilevel.cuh: rc_k = max(rcrit, rc_vel / 2^k)) or nullptr
    int nlev;                 // levels whose [1 - W_k] multiply in the pair term (1: the plain hybrid scheme)
    const int *members, *gstart;
    const long long *gstat;   // [0] = number of groups
    long long *status;
    double mu, G, dt, tol;
    int kind;
    int min_size, max_size;   // this launch handles groups with min_size <= n <= max_size
    const int *gcore;         // [ngroups] active members per group (semi-active mode) or nullptr
    // collisions inside the solver (reading S26; all nullptr / 0: off).  Fully active case only.
    double *m_io, *radius;    // [N] in/out: masses (= m) and physical radii; an absorbed body ends with m = 0, R = 0
    int *absorbed_by;         // [N] out: body that holds an absorbed body (entries of the others are not written)
    double frad;              // radius inflation factor f
    unsigned long long *work; // [2] work counters of the small-group and the satellite kernel, zero at launch: the CTAs take the
                              // next problem when they are done with one (a few hard encounters take ~70 Bulirsch-Stoer steps,
                              // most take one or two: a fixed stride would leave the last CTAs with the hard ones)
};

__device__ __forceinline__ int enc_group_size(const EncParams &p, const long long g, const int n, bool &split);

// Collisions inside the direct solver (reading S26), called after every ACCEPTED
// Bulirsch-Stoer step by the n member threads of a group (t = member, act = t < n; a warp if WARP, else the whole CTA)
// with the members' state in shared memory: X*, V* positions / velocities, smm masses, sgm = G m, srad radii,
// sinto[k] = member that absorbed member k (-1: none; -2: absorbed in an earlier call by a body outside the group), slab scratch.  Contact iff r_ij < f (R_i + R_j), strict, fp64 on
// r^2 = (dx^2 + dy^2) + dz^2 without contraction (the test of nb_merge, reading S21); members linked by a chain of
// contacts merge into the one with the smallest index: m <- sum m_k, x <- sum m_k x_k / sum m_k, v likewise (index
// order, unfused), R <- cbrt(sum R_k^3); an absorbed member gets m = 0, R = 0 and the survivor's x, v, and from then on
// takes no part in the encounter (sinto != -1: it exerts nothing and feels only the star, enc_accel's `ghost`).  Returns (to every calling thread) whether anything merged; *nabs (thread 0's) counts.
// The common case -- nobody touches -- costs one pass of n cheap tests per thread.
template <bool WARP>
__device__ __forceinline__ bool enc_collide(double *X0, double *X1, double *X2, double *V0, double *V1, double *V2,
                                            double *smm, double *sgm, double *srad, int *sinto, int *slab, const int n,
                                            const int t, const bool act, const double G, const double frad, int &nabs) {
    auto sync = [&]() { if (WARP) __syncwarp(); else __syncthreads(); };
    auto any = [&](const bool b) -> bool { return WARP ? (__any_sync(0xffffffffu, b) != 0) : (__syncthreads_or(b ? 1 : 0) != 0); };
    auto eligible = [&](const int k) { return sinto[k] == -1 && !(smm[k] == 0.0 && srad[k] == 0.0); };
    auto touch = [&](const int i, const int j) {
        const double dx = X0[j] - X0[i], dy = X1[j] - X1[i], dz = X2[j] - X2[i];
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        const double sr = __dmul_rn(frad, __dadd_rn(srad[i], srad[j]));
        return r2 < __dmul_rn(sr, sr);
    };
    sync();
    const bool mine = act && eligible(t);
    int lab = t;
    bool hit = false;
    if (mine)
        for (int j = 0; j < n; ++j)
            if (j != t && eligible(j) && touch(t, j)) { hit = true; if (j < lab) lab = j; }
    if (!any(hit)) return false;
    // label propagation to the smallest index of every cluster (clusters are tiny; this path is rare)
    if (act) slab[t] = lab;
    while (true) {
        sync();
        int nl = lab;
        if (hit) {
            for (int j = 0; j < n; ++j)
                if (j != t && eligible(j) && touch(t, j) && slab[j] < nl) nl = slab[j];
            if (slab[nl] < nl) nl = slab[nl];
        }
        const bool changed = nl != lab;
        sync();
        if (changed) { lab = nl; slab[t] = nl; }
        if (!any(changed)) break;
    }
    sync();
    int mine_abs = 0;
    if (hit && lab == t) {   // this member is the survivor of its cluster: sums over the cluster in index order
        double mt = 0.0, mx0 = 0.0, mx1 = 0.0, mx2 = 0.0, mv0 = 0.0, mv1 = 0.0, mv2 = 0.0, vol = 0.0;
        for (int k = t; k < n; ++k) {
            if (slab[k] != t || !eligible(k)) continue;
            const double mk = smm[k], rk = srad[k];
            mt = __dadd_rn(mt, mk);
            mx0 = __dadd_rn(mx0, __dmul_rn(mk, X0[k])); mx1 = __dadd_rn(mx1, __dmul_rn(mk, X1[k])); mx2 = __dadd_rn(mx2, __dmul_rn(mk, X2[k]));
            mv0 = __dadd_rn(mv0, __dmul_rn(mk, V0[k])); mv1 = __dadd_rn(mv1, __dmul_rn(mk, V1[k])); mv2 = __dadd_rn(mv2, __dmul_rn(mk, V2[k]));
            vol = __dadd_rn(vol, __dmul_rn(__dmul_rn(rk, rk), rk));
        }
        if (mt > 0.0) {
            X0[t] = __ddiv_rn(mx0, mt); X1[t] = __ddiv_rn(mx1, mt); X2[t] = __ddiv_rn(mx2, mt);
            V0[t] = __ddiv_rn(mv0, mt); V1[t] = __ddiv_rn(mv1, mt); V2[t] = __ddiv_rn(mv2, mt);
        }
        smm[t] = mt; sgm[t] = __dmul_rn(G, mt); srad[t] = cbrt(vol);
        for (int k = t + 1; k < n; ++k) {
            if (slab[k] != t || !eligible(k)) continue;
            smm[k] = 0.0; sgm[k] = 0.0; srad[k] = 0.0; sinto[k] = t; ++mine_abs;
            X0[k] = X0[t]; X1[k] = X1[t]; X2[k] = X2[t]; V0[k] = V0[t]; V1[k] = V1[t]; V2[k] = V2[t];
        }
    }
    nabs += mine_abs;
    sync();
    return true;
}

// CTA-wide maximum of a non-negative double; every thread gets it.
template <int THREADS>
__device__ __forceinline__ double cta_max(double val, double *red /* [32] */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) val = fmax(val, __shfl_xor_sync(0xffffffffu, val, o));
    if (THREADS > 32) {
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        __syncthreads();
        if (lane == 0) red[w] = val;
        __syncthreads();
        double r = (lane < THREADS / 32) ? red[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r = fmax(r, __shfl_xor_sync(0xffffffffu, r, o));
        val = r;
    }
    return val;
}

template <int THREADS>
__global__ void __launch_bounds__(THREADS) nb_encounter_kernel(const EncParams p) {
    extern __shared__ double enc_sm[];  // px[T] py[T] pz[T] gm[T] rc[T] vel[T] red[32]; with collisions (enc_smem_bytes):
                                        // + vx[T] vy[T] vz[T] mm[T] rad[T] and int into[T] lab[T]
    double *px = enc_sm, *py = px + THREADS, *pz = py + THREADS, *sgm = pz + THREADS, *src = sgm + THREADS,
           *svel = src + THREADS, *red = svel + THREADS;
    double *vx = red + 32, *vy = vx + THREADS, *vz = vy + THREADS, *smm = vz + THREADS, *srad = smm + THREADS;
    int *sinto = reinterpret_cast<int *>(srad + THREADS), *slab = sinto + THREADS;
    const bool collide = p.radius != nullptr;
    const int t = threadIdx.x;
    const long long ngroups = p.gstat[0];
    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const int g0 = p.gstart[g];
        bool split;
        const int n = enc_group_size(p, g, p.gstart[g + 1] - g0, split);
        if (n < p.min_size) continue;
        if (n > p.max_size) {
            if (n > kMaxGroup && p.max_size == kMaxGroup && t == 0) status_add(p.status, ST_GROUP_SKIPPED, 1);
            continue;
        }
        const bool act = t < n;
        const int b = act ? p.members[g0 + t] : 0;
        double y[6] = {0, 0, 0, 0, 0, 0};
        __syncthreads();
        if (act) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { y[c] = p.x[3 * (size_t)b + c]; y[3 + c] = p.v[3 * (size_t)b + c]; }
            sgm[t] = p.G * p.m[b];
            src[t] = p.rcrit[b];
            svel[t] = p.rc_vel != nullptr ? p.rc_vel[b] : 0.0;
            if (collide) { smm[t] = p.m[b]; srad[t] = p.radius[b]; sinto[t] = p.absorbed_by[b] >= 0 ? -2 : -1; }
        }
        if (collide) {
            __syncthreads();
            if (act && sinto[t] == -2) {   // absorbed in an earlier call: follows its holder if that is a member of this group
                const int holder = p.absorbed_by[b];
                for (int q = 0; q < n; ++q) if (p.members[g0 + q] == holder) sinto[t] = q;
            }
        }
        int nabs = 0;
        const double my_rc = act ? src[t] : 0.0, my_vel = act ? svel[t] : 0.0;

        // acceleration of this thread's body at position (qx,qy,qz), all members' positions taken from shared memory
        auto rhs = [&](const double (&q)[6], double (&f)[6]) {
            __syncthreads();
            if (act) { px[t] = q[0]; py[t] = q[1]; pz[t] = q[2]; }
            __syncthreads();
            if (act) {
                double ax, ay, az;
                enc_accel(q[0], q[1], q[2], my_rc, my_vel, t, n, px, py, pz, sgm, src, svel, p.nlev, p.mu, p.kind, ax, ay, az,
                          collide && sinto[t] != -1);
                f[0] = q[3]; f[1] = q[4]; f[2] = q[5]; f[3] = ax; f[4] = ay; f[5] = az;
            }
        };

        double T[kBsCols][6];
        double f0[6], f[6], ym[6], yn[6], dif[6];
        double tcur = 0.0, h = p.dt;
        const double tol2 = p.tol * p.tol;
        bool failed = false;
        while (tcur != p.dt) {
            if (fabs(h) > fabs(p.dt - tcur)) h = p.dt - tcur;
            if (fabs(h) < 1e-14 * fabs(p.dt)) { failed = true; break; }
            rhs(y, f0);
            bool accepted = false;
            int cols = 0;
            for (int c = 1; c <= kBsCols && !accepted; ++c) {
                const int nsub = 2 * c;
                const double hs = h / nsub;
#pragma unroll
                for (int k = 0; k < 6; ++k) { ym[k] = y[k]; yn[k] = y[k] + hs * f0[k]; }
                for (int s = 2; s <= nsub; ++s) {
                    rhs(yn, f);
#pragma unroll
                    for (int k = 0; k < 6; ++k) { const double tmp = ym[k] + 2.0 * hs * f[k]; ym[k] = yn[k]; yn[k] = tmp; }
                }
                rhs(yn, f);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    double cur = 0.5 * (ym[k] + yn[k] + hs * f[k]);
                    const double last_diag = c >= 2 ? T[c - 2][k] : 0.0;
                    for (int mc = 1; mc < c; ++mc) {
                        const double old = T[mc - 1][k];
                        T[mc - 1][k] = cur;
                        cur = cur + (cur - old) * bs_weight(c, mc);
                    }
                    T[c - 1][k] = cur;
                    dif[k] = cur - last_diag;
                }
                if (c >= 2) {
                    double e2 = 0.0;
                    if (act) {
                        const double ex = (dif[0] * dif[0] + dif[1] * dif[1]) + dif[2] * dif[2];
                        const double ev = (dif[3] * dif[3] + dif[4] * dif[4]) + dif[5] * dif[5];
                        const double sx = (y[0] * y[0] + y[1] * y[1]) + y[2] * y[2];
                        double sv = (y[3] * y[3] + y[4] * y[4]) + y[5] * y[5];
                        const double vc2 = p.mu / sqrt(sx);
                        if (sv < vc2) sv = vc2;
                        e2 = fmax(ex / sx, ev / sv);
                        if (!(e2 == e2)) e2 = INFINITY;  // NaN never passes
                    }
                    e2 = cta_max<THREADS>(e2, red);
                    if (e2 <= tol2) { accepted = true; cols = c; }
                }
            }
            if (accepted) {
#pragma unroll
                for (int k = 0; k < 6; ++k) y[k] = T[cols - 1][k];
                tcur = (fabs(p.dt - (tcur + h)) <= 1e-15 * fabs(p.dt)) ? p.dt : tcur + h;
                if (cols <= 6) h *= 1.3; else if (cols == 8) h *= 0.55;
                if (collide) {   // contacts at the accepted state (CTA-uniform): the state goes through shared memory
                    __syncthreads();
                    if (act) { px[t] = y[0]; py[t] = y[1]; pz[t] = y[2]; vx[t] = y[3]; vy[t] = y[4]; vz[t] = y[5]; }
                    if (enc_collide<false>(px, py, pz, vx, vy, vz, smm, sgm, srad, sinto, slab, n, t, act, p.G, p.frad, nabs) && act) {
                        y[0] = px[t]; y[1] = py[t]; y[2] = pz[t]; y[3] = vx[t]; y[4] = vy[t]; y[5] = vz[t];
                    }
                }
            } else {
                h *= 0.5;
            }
        }
        if (failed) {
            if (t == 0) status_add(p.status, ST_BS_FAIL, 1);  // group left unchanged
        } else if (collide) {
            // an absorbed member ends on the body that holds it now (its survivor may have been absorbed later itself)
            __syncthreads();
            if (act) { px[t] = y[0]; py[t] = y[1]; pz[t] = y[2]; vx[t] = y[3]; vy[t] = y[4]; vz[t] = y[5]; }
            __syncthreads();
            if (act) {
                int s0 = t;
                while (sinto[s0] >= 0) s0 = sinto[s0];
                p.x[3 * (size_t)b] = px[s0]; p.x[3 * (size_t)b + 1] = py[s0]; p.x[3 * (size_t)b + 2] = pz[s0];
                p.v[3 * (size_t)b] = vx[s0]; p.v[3 * (size_t)b + 1] = vy[s0]; p.v[3 * (size_t)b + 2] = vz[s0];
                p.m_io[b] = smm[t]; p.radius[b] = srad[t];
                if (s0 != t) p.absorbed_by[b] = p.members[g0 + s0];
                if (nabs > 0) status_add(p.status, ST_ABSORBED, nabs);
            }
        } else if (act) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { p.x[3 * (size_t)b + c] = y[c]; p.v[3 * (size_t)b + c] = y[3 + c]; }
        }
    }
}

// dynamic shared memory of nb_encounter_kernel<T>
__host__ __device__ constexpr size_t enc_smem_bytes(int T, bool collide) {
    return (6 * (size_t)T + 32) * sizeof(double) + (collide ? 5 * (size_t)T * sizeof(double) + 2 * (size_t)T * sizeof(int) : 0);
}

// Groups of up to 32 members: latency is everything (a hard pair takes tens of serial Bulirsch-Stoer steps),
// so the 8 extrapolation columns of a trial step -- independent modified-midpoint integrations with 2, 4,
// ..., 16 substeps -- run CONCURRENTLY, one warp per column, lane = member; warp 0 then builds the tableau
// column by column exactly as the sequential algorithm does and accepts the first column that passes, so
// the result is the sequential algorithm's, bit for bit.  Critical path per step: 17 right-hand sides
// instead of up to 80.
// Plan of the direct solver for one pair list: per group the number of active members (gcore; the whole group when
// everybody is active) and per body whether the solver will move it (flag; nb_drift_kernel then leaves it alone).
// A group is taken if its effective size -- the core of a split semi-active group, else the whole group -- is at
// most kMaxGroup.  One warp per group.
__global__ void __launch_bounds__(256) nb_enc_plan_kernel(const int *__restrict__ members, const int *__restrict__ gstart,
                                                         const long long *__restrict__ gstat, const int n_active,
                                                         int *__restrict__ gcore, int *__restrict__ flag) {
    const int lane = threadIdx.x & 31;
    const long long ngroups = gstat[0];
    for (long long g = ((long long)blockIdx.x * 256 + threadIdx.x) >> 5; g < ngroups; g += ((long long)gridDim.x * 256) >> 5) {
        const int g0 = gstart[g], n = gstart[g + 1] - g0;
        int nc = 0;
        for (int base = 0; base < n; base += 32) {  // members ascend: the active ones come first
            const bool a = base + lane < n && members[g0 + base + lane] < n_active;
            const int c = __popc(__ballot_sync(0xffffffffu, a));
            nc += c;
            if (c < 32) break;
        }
        const bool split = nc <= 31 && nc < n;
        const int take = (split ? nc : n) <= kMaxGroup;
        if (lane == 0) gcore[g] = nc;
        // the flags start at 0 (memset by the host): a group the solver does not take -- the one giant group of a dense disk,
        // 65 000 members written by one warp: 1.3 ms -- has nothing to write
        if (take)
            for (int k = lane; k < n; k += 32) flag[members[g0 + k]] = 1;
    }
}

// One problem of up to 32 bodies, solved by the whole CTA (8 warps = 8 columns; lane = member, b = the lane's body).
// Lanes >= keep_from write their final state back (0: everybody; nc: only the test particle of a split group).
// NW = 8 warps: one per column.  NW = 4 (the multi-level scheme's innermost calls: thousands of easy problems, throughput-
// bound): always two passes, columns 1 .. 4 and, if needed, 5 .. 8 on the same four warps -- half the CTA, twice as many per SM.
template <int NW>
__device__ __forceinline__ void bs_small_problem(const EncParams &p, const int b, const int n, const int keep_from) {
    __shared__ double px[NW][32], py[NW][32], pz[NW][32];
    __shared__ double sgm[32], src[32], svel[32];
    __shared__ double col[kBsCols][6][32];   // T_{c,0} of every column
    __shared__ double ycur[6][32];
    __shared__ double ctrl_h, ctrl_t;
    __shared__ int ctrl_done;                // 0 running, 1 finished, 2 failed
    __shared__ double smm[32], srad[32];     // collisions inside the solver (p.radius != nullptr): masses, radii,
    __shared__ int sinto[32], slab[32], sbody[32];   // who absorbed whom, label scratch, body of every member
    const bool collide = p.radius != nullptr;
    int nabs = 0;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const double tol2 = p.tol * p.tol;
    const bool act = lane < n;
    __syncthreads();
    if (w == 0) {
        if (act) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { ycur[c][lane] = p.x[3 * (size_t)b + c]; ycur[3 + c][lane] = p.v[3 * (size_t)b + c]; }
            sgm[lane] = p.G * p.m[b];
            src[lane] = p.rcrit[b];
            svel[lane] = p.rc_vel != nullptr ? p.rc_vel[b] : 0.0;
            if (collide) { smm[lane] = p.m[b]; srad[lane] = p.radius[b]; sinto[lane] = p.absorbed_by[b] >= 0 ? -2 : -1; sbody[lane] = b; }
        }
        if (lane == 0) { ctrl_h = p.dt; ctrl_t = 0.0; ctrl_done = (p.dt == 0.0) ? 1 : 0; }
        if (collide) {
            // absorbed in an earlier call and still in the arrays: follows its holder if that is a member of this problem
            __syncwarp();
            if (act && sinto[lane] == -2) {
                const int holder = p.absorbed_by[b];
                for (int q = 0; q < n; ++q) if (sbody[q] == holder) sinto[lane] = q;
            }
        }
    }
    __syncthreads();
    const double my_rc = act ? src[lane] : 0.0, my_vel = act ? svel[lane] : 0.0;
    double T[kBsCols][6];                // warp 0: current row of the tableau
    // A trial step whose first few columns already pass does not need the long ones: the columns are computed in two
    // passes -- 1 .. first, then (only if none of them passed) first + 1 .. 8 -- with first = 4 for the first trial step
    // of the short intervals of the multi-level scheme (dt / 2^L: most problems are done in that one step, in 3 or 4
    // columns) and after a step that was accepted in at most 4 columns, else 8 (one pass).  The tableau is still built
    // column by column and the first column that passes is taken: the result is the sequential algorithm's; the critical
    // path of such a step falls from 17 to 9 right-hand sides.  Measured: config 3 with the Eq. 7 radius and 4 levels
    // 37.2 -> 30.0 ms per step; single-level runs 1 - 2 % (the step-size rule grows h until ~6 columns are needed, so
    // easy steps are rare there).
    __shared__ int ctrl_first, ctrl_more;
    if (threadIdx.x == 0) ctrl_first = (NW == 4 || p.nlev > 1) ? 4 : kBsCols;
    __syncthreads();
    while (true) {
        if (ctrl_done != 0) break;
        double h = ctrl_h;
        const double tcur = ctrl_t;
        if (fabs(h) > fabs(p.dt - tcur)) h = p.dt - tcur;
        const bool underflow = fabs(h) < 1e-14 * fabs(p.dt);
        const int first = ctrl_first;
        double y[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) y[k] = act ? ycur[k][lane] : 0.0;
        bool accepted = false;           // warp 0
        int cols = 0;
        for (int pass = 0; pass < 2; ++pass) {
            const int c_lo = pass == 0 ? 1 : first + 1, c_hi = pass == 0 ? first : kBsCols;
            if (c_lo > c_hi) break;                       // one pass held all eight columns
            if (pass == 1 && ctrl_more == 0) break;       // a column of the first pass was accepted (or the step size underflowed)
            const int c = NW == 4 ? w + 1 + 4 * pass : w + 1;   // this warp's column in this pass
            if (!underflow && c >= c_lo && c <= c_hi) {
                // column c: modified midpoint with 2c substeps
                auto rhs = [&](const double (&q)[6], double (&f)[6]) {
                    __syncwarp();
                    if (act) { px[w][lane] = q[0]; py[w][lane] = q[1]; pz[w][lane] = q[2]; }
                    __syncwarp();
                    if (act) {
                        double ax, ay, az;
                        enc_accel(q[0], q[1], q[2], my_rc, my_vel, lane, n, px[w], py[w], pz[w], sgm, src, svel, p.nlev, p.mu, p.kind, ax, ay, az,
                                  collide && sinto[lane] != -1);
                        f[0] = q[3]; f[1] = q[4]; f[2] = q[5]; f[3] = ax; f[4] = ay; f[5] = az;
                    }
                };
                const int nsub = 2 * c;
                const double hs = h / nsub;
                double f0[6] = {0, 0, 0, 0, 0, 0}, f[6] = {0, 0, 0, 0, 0, 0}, ym[6], yn[6];
                rhs(y, f0);
#pragma unroll
                for (int k = 0; k < 6; ++k) { ym[k] = y[k]; yn[k] = y[k] + hs * f0[k]; }
                for (int s = 2; s <= nsub; ++s) {
                    rhs(yn, f);
#pragma unroll
                    for (int k = 0; k < 6; ++k) { const double tmp = ym[k] + 2.0 * hs * f[k]; ym[k] = yn[k]; yn[k] = tmp; }
                }
                rhs(yn, f);
#pragma unroll
                for (int k = 0; k < 6; ++k) col[c - 1][k][lane] = 0.5 * (ym[k] + yn[k] + hs * f[k]);
            }
            __syncthreads();
            if (w == 0) {
                if (!underflow) {
#pragma unroll
                    for (int c = 1; c <= kBsCols; ++c) {   // (compile-time column numbers: the tableau stays in registers)
                        if (c < c_lo || c > c_hi || accepted) continue;
                        double dif[6];
#pragma unroll
                        for (int k = 0; k < 6; ++k) {
                            double cur = col[c - 1][k][lane];
                            const double last_diag = c >= 2 ? T[c - 2][k] : 0.0;
                            for (int mc = 1; mc < c; ++mc) {
                                const double old = T[mc - 1][k];
                                T[mc - 1][k] = cur;
                                cur = cur + (cur - old) * bs_weight(c, mc);
                            }
                            T[c - 1][k] = cur;
                            dif[k] = cur - last_diag;
                        }
                        if (c >= 2) {
                            double e2 = 0.0;
                            if (act) {
                                const double ex = (dif[0] * dif[0] + dif[1] * dif[1]) + dif[2] * dif[2];
                                const double ev = (dif[3] * dif[3] + dif[4] * dif[4]) + dif[5] * dif[5];
                                const double sx = (y[0] * y[0] + y[1] * y[1]) + y[2] * y[2];
                                double sv = (y[3] * y[3] + y[4] * y[4]) + y[5] * y[5];
                                const double vc2 = p.mu / sqrt(sx);
                                if (sv < vc2) sv = vc2;
                                e2 = fmax(ex / sx, ev / sv);
                                if (!(e2 == e2)) e2 = INFINITY;
                            }
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) e2 = fmax(e2, __shfl_xor_sync(0xffffffffu, e2, o));
                            if (e2 <= tol2) { accepted = true; cols = c; }
                        }
                    }
                }
                if (lane == 0) ctrl_more = (!accepted && !underflow) ? 1 : 0;
            }
            __syncthreads();
        }
        if (w == 0) {
            if (accepted && act) {
#pragma unroll
                for (int k = 0; k < 6; ++k) ycur[k][lane] = T[cols - 1][k];
            }
            if (collide && accepted)   // warp-uniform: contacts at the accepted state, clusters merge at once
                enc_collide<true>(ycur[0], ycur[1], ycur[2], ycur[3], ycur[4], ycur[5], smm, sgm, srad, sinto, slab, n, lane, act,
                                  p.G, p.frad, nabs);
            if (lane == 0) {
                if (underflow) {
                    ctrl_done = 2;
                } else if (accepted) {
                    const double tn = (fabs(p.dt - (tcur + h)) <= 1e-15 * fabs(p.dt)) ? p.dt : tcur + h;
                    ctrl_t = tn;
                    ctrl_h = cols <= 6 ? h * 1.3 : (cols == 8 ? h * 0.55 : h);
                    ctrl_first = (NW == 4 || cols <= 4) ? 4 : kBsCols;
                    if (tn == p.dt) ctrl_done = 1;
                } else {
                    ctrl_h = h * 0.5;
                    ctrl_first = NW == 4 ? 4 : kBsCols;
                }
            }
        }
        __syncthreads();
    }
    if (w == 0) {
        if (ctrl_done == 2) {
            if (lane == 0) status_add(p.status, ST_BS_FAIL, 1);  // group left unchanged
        } else if (act && lane >= keep_from) {
            int src = lane;
            if (collide) {
                // an absorbed member ends on the body that holds it now (its survivor may have been absorbed later itself)
                while (sinto[src] >= 0) src = sinto[src];
                p.m_io[b] = smm[lane]; p.radius[b] = srad[lane];
                if (src != lane) p.absorbed_by[b] = sbody[src];
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) { p.x[3 * (size_t)b + c] = ycur[c][src]; p.v[3 * (size_t)b + c] = ycur[3 + c][src]; }
            if (nabs > 0) status_add(p.status, ST_ABSORBED, nabs);
        }
    }

}

// effective size of group g: its core in a split semi-active group (gcore), else the whole group
__device__ __forceinline__ int enc_group_size(const EncParams &p, const long long g, const int n, bool &split) {
    split = false;
    if (p.gcore == nullptr) return n;
    const int nc = p.gcore[g];
    split = nc <= 31 && nc < n;
    return split ? nc : n;
}

// (two CTAs per SM: the collision code must not cost the second one -- 146 registers uncapped, measured 37.9 -> 52.1 ms per
// step on config 3 with 4 levels)
template <int NW>
__global__ void __launch_bounds__(32 * NW, 16 / NW) nb_encounter_small_kernel(const EncParams p) {
    __shared__ long long sh_next;
    const int lane = threadIdx.x & 31;
    const long long ngroups = p.gstat[0];
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) sh_next = (long long)atomicAdd(p.work, 1ull);
        __syncthreads();
        const long long g = sh_next;
        if (g >= ngroups) break;
        const int g0 = p.gstart[g];
        bool split;
        const int n = enc_group_size(p, g, p.gstart[g + 1] - g0, split);
        if (n < p.min_size || n > p.max_size) continue;
        bs_small_problem<NW>(p, lane < n ? p.members[g0 + lane] : 0, n, 0);
    }
}

// Semi-active mode: the test particles of split groups, one CTA per particle: {core + particle} from the initial
// state, only the particle is kept (reading S22).  Must run BEFORE the kernels that advance the cores.
// Thousands of easy problems: throughput-bound, so the register allocation is capped for 4 CTAs per SM (the
// latency-bound kernel above is faster uncapped).
__global__ void __launch_bounds__(32 * kBsCols, 4) nb_encounter_sat_kernel(const EncParams p) {
    __shared__ int sh_g;
    __shared__ long long sh_k;
    const int lane = threadIdx.x & 31;
    const long long ngroups = p.gstat[0], nslots = p.gstat[1];
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) sh_k = (long long)atomicAdd(p.work + 1, 1ull);
        __syncthreads();
        const long long k = sh_k;
        if (k >= nslots) break;
        if (threadIdx.x == 0) {  // group of member slot k: last g with gstart[g] <= k
            long long lo = 0, hi = ngroups - 1;
            while (lo < hi) { const long long mid = (lo + hi + 1) >> 1; if (p.gstart[mid] <= k) lo = mid; else hi = mid - 1; }
            sh_g = (int)lo;
        }
        __syncthreads();
        const long long g = sh_g;
        const int g0 = p.gstart[g];
        bool split;
        const int nc = enc_group_size(p, g, p.gstart[g + 1] - g0, split);
        if (!split || k < g0 + nc) continue;  // not a test particle of a split group
        const int b = lane < nc ? p.members[g0 + lane] : (lane == nc ? p.members[k] : 0);
        bs_small_problem<kBsCols>(p, b, nc + 1, nc);
    }
}

}  // namespace nbk
