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
#include "nb_common.cuh"

namespace nbk {

constexpr int kBsCols = 8;
constexpr int kMaxGroup = 1024;  // larger groups are left to the Kepler drift and counted (NB_MAX_GROUP)

__device__ __forceinline__ double one_minus_changeover(const double r, const double rc, const int kind) {
    if (!(r < rc)) return 0.0;
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 1.0;
    if (y >= 1.0) return 0.0;
    const double z = 1.0 - y;
    if (kind == 1) return z * z * z * (1.0 + y * (3.0 + 6.0 * y));
    return (z * z) / (2.0 * y * y - 2.0 * y + 1.0);
}

struct EncParams {
    double *x, *v;            // [N,3] in/out (members only)
    const double *m, *rcrit;  // [N]
    const int *members, *gstart;
    const long long *gstat;   // [0] = number of groups
    long long *status;
    double mu, G, dt, tol;
    int kind;
    int min_size, max_size;   // this launch handles groups with min_size <= n <= max_size
};

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
    extern __shared__ double enc_sm[];  // px[T] py[T] pz[T] gm[T] rc[T] red[32]
    double *px = enc_sm, *py = px + THREADS, *pz = py + THREADS, *sgm = pz + THREADS, *src = sgm + THREADS,
           *red = src + THREADS;
    const int t = threadIdx.x;
    const long long ngroups = p.gstat[0];
    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const int g0 = p.gstart[g], n = p.gstart[g + 1] - g0;
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
        }
        const double my_rc = act ? src[t] : 0.0;

        // acceleration of this thread's body at position (qx,qy,qz), all members' positions taken from shared memory
        auto rhs = [&](const double (&q)[6], double (&f)[6]) {
            __syncthreads();
            if (act) { px[t] = q[0]; py[t] = q[1]; pz[t] = q[2]; }
            __syncthreads();
            if (act) {
                const double r2 = (q[0] * q[0] + q[1] * q[1]) + q[2] * q[2];
                const double s = -p.mu / (r2 * sqrt(r2));
                double ax = s * q[0], ay = s * q[1], az = s * q[2];
                for (int j = 0; j < n; ++j) {
                    if (j == t) continue;
                    const double dx = px[j] - q[0], dy = py[j] - q[1], dz = pz[j] - q[2];
                    const double d2 = (dx * dx + dy * dy) + dz * dz;
                    if (d2 == 0.0) continue;
                    const double d = sqrt(d2);
                    const double w = one_minus_changeover(d, fmax(my_rc, src[j]), p.kind);
                    if (w == 0.0) continue;
                    const double tt = sgm[j] * w / (d2 * d);
                    ax += tt * dx; ay += tt * dy; az += tt * dz;
                }
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
                        const double ratio = (double)nsub / (double)(2 * (c - mc));
                        const double old = T[mc - 1][k];
                        T[mc - 1][k] = cur;
                        cur = cur + (cur - old) / (ratio * ratio - 1.0);
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
            } else {
                h *= 0.5;
            }
        }
        if (failed) {
            if (t == 0) status_add(p.status, ST_BS_FAIL, 1);  // group left unchanged
        } else if (act) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { p.x[3 * (size_t)b + c] = y[c]; p.v[3 * (size_t)b + c] = y[3 + c]; }
        }
    }
}

}  // namespace nbk
