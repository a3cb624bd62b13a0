// body_kernels.cuh -- the O(N) kernels around the force tiles: critical radius + j-record staging
// (a0), partial-sum reduce + velocity kick (a4), H_C shift (a5), Kepler drift (a6).
// One thread per body, kBodyThreads per CTA.  The total momentum needed by H_C travels between
// kernels as per-CTA partial sums that every consumer CTA re-reduces in a fixed order, so a step
// needs no separate reduction launch and stays bit-reproducible.
#pragma once
#include "kepler.cuh"
#include "nb_common.cuh"

namespace nbk {

// Eq. 7 with reading S5 for R_Hill.
__device__ __forceinline__ double critical_radius(const double x, const double y, const double z, const double vx,
                                                  const double vy, const double vz, const double m,
                                                  const double M_star, const double G, const double n1,
                                                  const double n2, const double absdt, double *hill_term = nullptr,
                                                  double *vel_term = nullptr) {
    const double r = sqrt(x * x + y * y + z * z);
    const double v2 = vx * vx + vy * vy + vz * vz;
    const double inva = 2.0 / r - v2 / (G * M_star);
    const double a = (inva > 0.0) ? 1.0 / inva : r;
    const double rh = a * cbrt(m / (3.0 * M_star));
    const double t1 = n1 * rh, t2 = n2 * absdt * sqrt(v2);
    if (hill_term != nullptr) { *hill_term = t1; *vel_term = t2; }   // multilevel.cuh: rc_k = max(t1, t2 / 2^k)
    return fmax(t1, t2);
}

struct PrepParams {
    double *x;              // [N,3]; written only when mv_in != nullptr (second H_C half-shift)
    const double *v;        // [N,3]; needed when update_rc
    const double *m;        // [N]
    double *rcrit;          // [N]; written when update_rc, read otherwise
    double *rc_hill, *rc_vel;  // [N] the two terms of Eq. 7 for the multi-level scheme (nullptr: not wanted); with caller's
                            // radii (update_rc = 0): hill = 0, vel = rcrit, i.e. rc_k = rcrit / 2^k
    JRec *jrec;             // [Njpad] one-sided kernel's records (nullptr: not staged)
    double2 *sxy, *szg;     // [2 Npad_sym] symmetric kernel's (x,y) and (z,Gm), doubled-block layout (nullptr: not staged)
    int *sthr;              // [2 Npad_sym] hi32(rcrit^2) + 1
    JRecDs *jds;            // [Njpad] double-single records of the one-sided mixed-precision kernel (nullptr: not staged)
    float4 *sa, *sb;        // [2 Npad_sym] double-single records of the Newton-III mixed-precision kernel (nullptr: not staged)
    int Npad_sym;
    const int *pos_of;      // [N] staged position of each body (sort_staging.cuh) or nullptr: position = index
    const double *mv_in;    // [nblk_in,3] momentum partials or nullptr
    unsigned long long *npairs;  // reset to 0 here (nullptr: skip)
    long long *status;
    double dtc;             // shift time (dt/2)
    double M_star, G, n1, n2, absdt;
    int nblk_in;
    int N, Nj, Njpad;
    int update_rc;
};

// a5 (second half) + a0 + staging for ONE body slot i (the grid covers max(N, Njpad, Npad_sym)): x += dtc * s; rcrit
// from the shifted state; JRec for j < Nj.  (sx, sy, sz) = total momentum / M_star (0 when there is no shift).
__device__ __forceinline__ void prep_one(const PrepParams &p, const int i, const double sx, const double sy, const double sz) {
    if (i == 0 && p.npairs != nullptr) *p.npairs = 0ull;
    // padding record: zero mass, far away => contributes exactly 0 and never votes for the slow path
    JRec r;
    r.x = kFarJ; r.y = kFarJ; r.z = kFarJ; r.gm = 0.0; r.c1 = 0.0; r.c2 = 0.0; r.rc2 = 0.0; r.rc = 0.0;
    if (i < p.N) {
        double x = p.x[3 * (size_t)i], y = p.x[3 * (size_t)i + 1], z = p.x[3 * (size_t)i + 2];
        if (p.mv_in != nullptr) {
            x = x + p.dtc * sx; y = y + p.dtc * sy; z = z + p.dtc * sz;
            p.x[3 * (size_t)i] = x; p.x[3 * (size_t)i + 1] = y; p.x[3 * (size_t)i + 2] = z;
        }
        const double m = p.m[i];
        double rc;
        double t1 = 0.0, t2;
        if (p.update_rc) {
            rc = critical_radius(x, y, z, p.v[3 * (size_t)i], p.v[3 * (size_t)i + 1], p.v[3 * (size_t)i + 2], m,
                                 p.M_star, p.G, p.n1, p.n2, p.absdt, &t1, &t2);
            p.rcrit[i] = rc;
        } else {
            rc = p.rcrit[i];
            t2 = rc;
        }
        if (p.rc_hill != nullptr) { p.rc_hill[i] = t1; p.rc_vel[i] = t2; }
        if (i < p.Nj) {
            const double gm = p.G * m;
            r.x = x; r.y = y; r.z = z; r.gm = gm;
            r.c1 = 1.5 * gm; r.c2 = 1.875 * gm; r.rc2 = rc * rc; r.rc = rc;
            if (!(isfinite(x) && isfinite(y) && isfinite(z) && isfinite(gm) && isfinite(rc) && rc >= 0.0))
                status_add(p.status, ST_NONFINITE, 1);
        }
    }
    if (p.jrec != nullptr && i < p.Njpad) p.jrec[i] = r;  // grid covers max(N, Njpad, Npad_sym)
    if (p.jds != nullptr && i < p.Njpad) p.jds[i] = make_jrecds(r.x, r.y, r.z, r.gm, r.rc2);
    if (p.sxy != nullptr && i < p.Npad_sym) {
        // symmetric kernel: every body is both an i- and a j-body; padding bodies get distinct far
        // positions (pad-pad distances stay huge and finite) and zero mass
        double sx_ = r.x, sy_ = r.y, sz_ = r.z;
        if (i >= p.N) { sx_ = kFarJ + 1.0e27 * (double)(i - p.N + 1); sy_ = kFarJ; sz_ = kFarJ; }
        const int pos = (p.pos_of != nullptr && i < p.N) ? p.pos_of[i] : i;   // padding bodies keep the tail positions
        const size_t en = (size_t)(pos >> 5) * 64 + (pos & 31);  // doubled-block layout (force_sym.cuh)
        const int thr = __double2hiint(r.rc2) + 1;
        p.sxy[en] = make_double2(sx_, sy_); p.sxy[en + 32] = make_double2(sx_, sy_);
        p.szg[en] = make_double2(sz_, r.gm); p.szg[en + 32] = make_double2(sz_, r.gm);
        p.sthr[en] = thr; p.sthr[en + 32] = thr;
        if (p.sa != nullptr) symds_stage(p.sa, p.sb, pos, sx_, sy_, sz_, r.gm, r.rc2);
    }
}

__global__ void __launch_bounds__(kBodyThreads) nb_prep_kernel(const PrepParams p) {
    __shared__ double sm[3 * kBodyThreads];
    double sx = 0.0, sy = 0.0, sz = 0.0;
    if (p.mv_in != nullptr) {
        reduce_partials3(p.mv_in, p.nblk_in, sx, sy, sz, sm);
        sx /= p.M_star; sy /= p.M_star; sz /= p.M_star;
    }
    prep_one(p, blockIdx.x * kBodyThreads + threadIdx.x, sx, sy, sz);
}

// standalone a0
__global__ void __launch_bounds__(kBodyThreads) nb_rcrit_kernel(const double *__restrict__ x, const double *__restrict__ v,
                                                               const double *__restrict__ m, double *__restrict__ rcrit,
                                                               int N, double M_star, double G, double n1, double n2,
                                                               double absdt) {
    const int i = blockIdx.x * kBodyThreads + threadIdx.x;
    if (i >= N) return;
    rcrit[i] = critical_radius(x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], v[3 * (size_t)i],
                               v[3 * (size_t)i + 1], v[3 * (size_t)i + 2], m[i], M_star, G, n1, n2, absdt);
}

// a4: acc_i = sum over j-splits (in split order) of the partial sums; v_i = v_i + hk*acc_i, applied
// nhalf times (the closing half-kick of one step and the opening half-kick of the next are two
// separate roundings, as in the step definition).  Optionally emits momentum partials of the new v.
// perm != nullptr: the partial sums are indexed by staged position (sort_staging.cuh); thread t then serves
// position t (coalesced slot reads) and writes the body perm[t] (the real bodies hold positions 0 .. N-1).
// xcols > 0 (Newton-III kernel with tail splitting, force_sym.cuh kSymSplit): column nsplit-1-c of the tile grid was cut
// into parts whose i sides sit in 3 extra slots, nsplit + 3 c + {0, 1, 2}, valid for the positions in front of that
// column, t < (nsplit-1-c) S; they are added after the regular slots, in order.
// the work of thread slot t (of N): returns the momentum contribution of the kicked body
__device__ __forceinline__ void kickv_one(const double *part, const int nsplit, double *acc, double *__restrict__ v,
                                          const double *__restrict__ m, const int N, const double hk, const int nhalf,
                                          const bool want_mv, const int *__restrict__ perm, const int t, double &px, double &py,
                                          double &pz, const int xcols = 0, const int S = 0) {
    px = 0.0; py = 0.0; pz = 0.0;
    const int i = (perm != nullptr && t < N) ? perm[t] : t;
    if (t < N && i < N) {
        double ax = 0.0, ay = 0.0, az = 0.0;
        // the loads of 8 slots are issued together (the sum is latency-bound otherwise: up to 140 slots at N = 65536);
        // the additions keep the slot order
        int s = 0;
        for (; s + 8 <= nsplit; s += 8) {
            double b[8][3];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const double *q = part + ((size_t)(s + u) * N + t) * 3;
                b[u][0] = q[0]; b[u][1] = q[1]; b[u][2] = q[2];
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) { ax += b[u][0]; ay += b[u][1]; az += b[u][2]; }
        }
        for (; s < nsplit; ++s) {
            const double *q = part + ((size_t)s * N + t) * 3;
            ax += q[0]; ay += q[1]; az += q[2];
        }
        for (int c = 0; c < xcols; ++c) {
            if (t >= (nsplit - 1 - c) * S) continue;
            for (int e = 0; e < 3; ++e) {
                const double *q = part + ((size_t)(nsplit + 3 * c + e) * N + t) * 3;
                ax += q[0]; ay += q[1]; az += q[2];
            }
        }
        acc[3 * (size_t)i] = ax; acc[3 * (size_t)i + 1] = ay; acc[3 * (size_t)i + 2] = az;
        double vx = v[3 * (size_t)i], vy = v[3 * (size_t)i + 1], vz = v[3 * (size_t)i + 2];
        for (int h = 0; h < nhalf; ++h) {
            vx = vx + hk * ax; vy = vy + hk * ay; vz = vz + hk * az;
        }
        if (nhalf > 0) { v[3 * (size_t)i] = vx; v[3 * (size_t)i + 1] = vy; v[3 * (size_t)i + 2] = vz; }
        if (want_mv) { const double mi = m[i]; px = mi * vx; py = mi * vy; pz = mi * vz; }
    }
}

__global__ void __launch_bounds__(kBodyThreads) nb_kickv_kernel(const double *part, int nsplit,
                                                               double *acc, double *__restrict__ v,
                                                               const double *__restrict__ m, int N, double hk,
                                                               int nhalf, double *__restrict__ mv_out,
                                                               const int *__restrict__ perm, int xcols, int S) {
    __shared__ double sm[3 * kBodyThreads];
    double px, py, pz;
    kickv_one(part, nsplit, acc, v, m, N, hk, nhalf, mv_out != nullptr, perm, blockIdx.x * kBodyThreads + threadIdx.x, px, py, pz, xcols, S);
    if (mv_out != nullptr) {
        block_sum3(px, py, pz, sm);
        if (threadIdx.x == 0) {
            mv_out[3 * blockIdx.x] = px; mv_out[3 * blockIdx.x + 1] = py; mv_out[3 * blockIdx.x + 2] = pz;
        }
    }
}

// Banded evaluation of the Newton-III kernel (force_sym.cuh SymParams): folds the partial sums of the band of tile
// columns col0 .. col0 + ncols - 1 into acc, in a fixed order -- the i sides part_i[b][N] (valid for the positions in
// front of column col0 + b), then, for the band's own bodies, the j sides part_j[A][ncols S], A = 0 .. own block.
// first != 0: acc starts from 0.  Thread t serves staged position t and writes body perm[t] (or t).
__global__ void __launch_bounds__(kBodyThreads) nb_bandsum_kernel(const double *__restrict__ part_i, const double *__restrict__ part_j,
                                                                 double *acc, int N, int S, int col0, int ncols, int first,
                                                                 const int *__restrict__ perm) {
    const int t = blockIdx.x * kBodyThreads + threadIdx.x;
    if (t >= N) return;
    const int i = perm != nullptr ? perm[t] : t;
    if (i >= N) return;
    double ax = 0.0, ay = 0.0, az = 0.0;
    if (!first) { ax = acc[3 * (size_t)i]; ay = acc[3 * (size_t)i + 1]; az = acc[3 * (size_t)i + 2]; }
    for (int b = 0; b < ncols; ++b) {
        if (t >= (long long)(col0 + b) * S) continue;
        const double *q = part_i + ((size_t)b * N + t) * 3;
        ax += q[0]; ay += q[1]; az += q[2];
    }
    const int X = t / S;
    if (X >= col0 && X < col0 + ncols) {
        const size_t stride = (size_t)ncols * S, off = (size_t)t - (size_t)col0 * S;
        for (int A = 0; A <= X; ++A) {
            const double *q = part_j + ((size_t)A * stride + off) * 3;
            ax += q[0]; ay += q[1]; az += q[2];
        }
    }
    acc[3 * (size_t)i] = ax; acc[3 * (size_t)i + 1] = ay; acc[3 * (size_t)i + 2] = az;
}

// momentum partials of the current v (standalone nb_shift)
__global__ void __launch_bounds__(kBodyThreads) nb_momentum_kernel(const double *__restrict__ v, const double *__restrict__ m,
                                                                  int N, double *__restrict__ mv_out) {
    __shared__ double sm[3 * kBodyThreads];
    const int i = blockIdx.x * kBodyThreads + threadIdx.x;
    double px = 0.0, py = 0.0, pz = 0.0;
    if (i < N) { const double mi = m[i]; px = mi * v[3 * (size_t)i]; py = mi * v[3 * (size_t)i + 1]; pz = mi * v[3 * (size_t)i + 2]; }
    block_sum3(px, py, pz, sm);
    if (threadIdx.x == 0) { mv_out[3 * blockIdx.x] = px; mv_out[3 * blockIdx.x + 1] = py; mv_out[3 * blockIdx.x + 2] = pz; }
}

// standalone a5: x += dtc * P / M_star
__global__ void __launch_bounds__(kBodyThreads) nb_shift_kernel(double *__restrict__ x, const double *__restrict__ mv_in,
                                                               int nblk_in, int N, double dtc, double M_star) {
    __shared__ double sm[3 * kBodyThreads];
    double sx, sy, sz;
    reduce_partials3(mv_in, nblk_in, sx, sy, sz, sm);
    sx /= M_star; sy /= M_star; sz /= M_star;
    const int i = blockIdx.x * kBodyThreads + threadIdx.x;
    if (i < N) {
        x[3 * (size_t)i] = x[3 * (size_t)i] + dtc * sx;
        x[3 * (size_t)i + 1] = x[3 * (size_t)i + 1] + dtc * sy;
        x[3 * (size_t)i + 2] = x[3 * (size_t)i + 2] + dtc * sz;
    }
}

// a5 (first half, optional) + a6: x += dtc*P/M_star, then the Kepler flow for dt; optionally emits the
// momentum partials of the drifted velocities for the second half-shift.  With enc_flag (nb_enc_plan_kernel) the
// bodies the direct solver will move are shifted but not drifted.
__device__ __forceinline__ void drift_one(double *__restrict__ x, double *__restrict__ v, const double *__restrict__ m,
                                          const int N, const double mu, const double dt, const bool shift, const double dtc,
                                          const double sx, const double sy, const double sz, const bool want_mv,
                                          long long *status, const int *__restrict__ enc_flag, const int i, double &px,
                                          double &py, double &pz) {
    px = 0.0; py = 0.0; pz = 0.0;
    if (i < N) {
        double X0 = x[3 * (size_t)i], X1 = x[3 * (size_t)i + 1], X2 = x[3 * (size_t)i + 2];
        double V0 = v[3 * (size_t)i], V1 = v[3 * (size_t)i + 1], V2 = v[3 * (size_t)i + 2];
        if (shift) { X0 = X0 + dtc * sx; X1 = X1 + dtc * sy; X2 = X2 + dtc * sz; }
        // bodies of the encounter groups the direct solver takes (encounter.cuh) are left to it
        const bool in_group = enc_flag != nullptr && enc_flag[i] != 0;
        if (!in_group && kepler_elliptic_fast(X0, X1, X2, V0, V1, V2, mu, dt) != 0) {
            // rare: unbound, nearly parabolic, or the fast iteration did not settle -> universal variables (state untouched so far)
            double X[3] = {X0, X1, X2}, V[3] = {V0, V1, V2};
            const int rcode = kepler_universal(X, V, mu, dt);
            if (rcode != 0) status_add(status, ST_KEPLER_FAIL, 1);
            X0 = X[0]; X1 = X[1]; X2 = X[2]; V0 = V[0]; V1 = V[1]; V2 = V[2];
        }
        x[3 * (size_t)i] = X0; x[3 * (size_t)i + 1] = X1; x[3 * (size_t)i + 2] = X2;
        v[3 * (size_t)i] = V0; v[3 * (size_t)i + 1] = V1; v[3 * (size_t)i + 2] = V2;
        if (want_mv) { const double mi = m[i]; px = mi * V0; py = mi * V1; pz = mi * V2; }
    }
}

__global__ void __launch_bounds__(kBodyThreads) nb_drift_kernel(double *__restrict__ x, double *__restrict__ v,
                                                               const double *__restrict__ m, int N, double mu, double dt,
                                                               const double *__restrict__ mv_in, int nblk_in,
                                                               double dtc, double M_star, double *__restrict__ mv_out,
                                                               long long *status, const int *__restrict__ enc_flag) {
    __shared__ double sm[3 * kBodyThreads];
    double sx = 0.0, sy = 0.0, sz = 0.0;
    if (mv_in != nullptr) {
        reduce_partials3(mv_in, nblk_in, sx, sy, sz, sm);
        sx /= M_star; sy /= M_star; sz /= M_star;
    }
    double px, py, pz;
    drift_one(x, v, m, N, mu, dt, mv_in != nullptr, dtc, sx, sy, sz, mv_out != nullptr, status, enc_flag,
              blockIdx.x * kBodyThreads + threadIdx.x, px, py, pz);
    if (mv_out != nullptr) {
        block_sum3(px, py, pz, sm);
        if (threadIdx.x == 0) { mv_out[3 * blockIdx.x] = px; mv_out[3 * blockIdx.x + 1] = py; mv_out[3 * blockIdx.x + 2] = pz; }
    }
}

// Velocity-dependent extra force by the implicit midpoint method (Eq. 8):
//     v' = v + dt a_f(r, (v + v')/2),   a_f = -gamma |u|^p u,  u = v - (1 - eta) sqrt(mu/R) e_phi   (reading S24: gas drag)
// solved per body by the fixed-point iteration w <- v + dt a_f(r, (v + w)/2) from w = v until the update is below
// tol max(|w|, |v_gas|) or max_iter iterations ("needs some iterations to converge"); non-convergence is counted.
__global__ void __launch_bounds__(kBodyThreads) nb_midpoint_drag_kernel(const double *__restrict__ x, double *__restrict__ v,
                                                                       int N, double mu, double dt, double gamma, int power,
                                                                       double eta, double tol, int max_iter, long long *status) {
    const int i = blockIdx.x * kBodyThreads + threadIdx.x;
    if (i >= N) return;
    const double x0 = x[3 * (size_t)i], x1 = x[3 * (size_t)i + 1];
    const double v0 = v[3 * (size_t)i], v1 = v[3 * (size_t)i + 1], v2 = v[3 * (size_t)i + 2];
    const double R2 = x0 * x0 + x1 * x1;
    double g0 = 0.0, g1 = 0.0, vgn = 0.0;
    if (R2 > 0.0) {
        const double R = sqrt(R2);
        const double vc = (1.0 - eta) * sqrt(mu / R);
        g0 = -vc * x1 / R; g1 = vc * x0 / R; vgn = fabs(vc);
    }
    double w0 = v0, w1 = v1, w2 = v2;
    bool converged = false;
#pragma unroll 1
    for (int it = 0; it < max_iter; ++it) {
        const double u0 = 0.5 * (v0 + w0) - g0, u1 = 0.5 * (v1 + w1) - g1, u2 = 0.5 * (v2 + w2);
        double f = gamma;
        if (power == 1) f = gamma * sqrt((u0 * u0 + u1 * u1) + u2 * u2);
        const double n0 = v0 + dt * (-f * u0), n1 = v1 + dt * (-f * u1), n2 = v2 + dt * (-f * u2);
        const double d = sqrt((n0 - w0) * (n0 - w0) + (n1 - w1) * (n1 - w1) + (n2 - w2) * (n2 - w2));
        const double nn = sqrt(n0 * n0 + n1 * n1 + n2 * n2);
        w0 = n0; w1 = n1; w2 = n2;
        if (d <= tol * fmax(nn, vgn)) { converged = true; break; }
    }
    if (!converged) status_add(status, ST_MIDPOINT_FAIL, 1);
    v[3 * (size_t)i] = w0; v[3 * (size_t)i + 1] = w1; v[3 * (size_t)i + 2] = w2;
}

// fp64 FMA-rate microbenchmark: 8 independent chains per thread, register only.  The FMAs read TWO
// distinct vector-register pairs (c = p*p + c): a DFMA reading three distinct pairs issues every 3
// clocks instead of 2 on sm_100 (register-file read ports; profiles/r1_fp64_pipe_microbench.md), so
// the three-operand form would understate the pipe's peak by a third.
__global__ void __launch_bounds__(256) nb_fp64_peak_kernel(double *out, long long iters, const double *src) {
    double c[8], p[8];
    const double tid = threadIdx.x * 1e-9;
#pragma unroll
    for (int r = 0; r < 8; ++r) { c[r] = tid + r; p[r] = src[r] + tid; }
#pragma unroll 1
    for (long long k = 0; k < iters; ++k) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int r = 0; r < 8; ++r) c[r] = __fma_rn(p[r], p[r], c[r]);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < 8; ++r) s += c[r];
    if (s == 123.456) out[0] = s;  // keeps the chains alive; practically never true
}

}  // namespace nbk
