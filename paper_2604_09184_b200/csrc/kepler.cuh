// kepler.cuh -- H_A without encounters: per-body Kepler flow about mu = G M_star with Gauss' f and g
// functions ("a Keplerian orbit can be solved analytically"; Eq. 4 first sum;
// PAPER.md:98; the f/g form is fixed by BASELINE.json:north_star; solver details: DESIGN.md S15).
#pragma once
#include "nb_common.cuh"

namespace nbk {

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kEps = 2.220446049250313e-16;


// ---- fast path of the bound-orbit solver -------------------------------------------------------
// Same equations as kepler_elliptic below (differenced Kepler equation, Gauss f and g), arranged
// for the FP64 pipe: no IEEE divide or sqrt (MUFU seeds + one third-order correction, ~1 ulp), ONE
// library sincos -- of the half angle dE/2, which gives sin dE = 2SC and 1 - cos dE = 2S^2 without
// cancellation -- and Halley steps whose trigonometric update is a rotation of (S, C) by the small
// correction.  Anything unusual (not bound, no convergence in 8 steps, non-finite) returns nonzero
// with the state untouched, and the caller falls back to the bracketed solver.

__device__ __forceinline__ double rcp_fast(const double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));  // MUFU.RCP64H, ~2^-20
    const double e = __fma_rn(-x, y, 1.0);
    return __fma_rn(y, __fma_rn(e, e, e), y);               // y (1 + e + e^2): ~2^-60
}
// 1/sqrt(x) to ~2^-60 for normal x > 0
__device__ __forceinline__ double rsqrt_fast(const double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));  // MUFU.RSQ64H, ~2^-20
    const double e = __fma_rn(-x, y * y, 1.0);
    return __fma_rn(y * e, __fma_rn(e, 0.375, 0.5), y);       // y (1 + e/2 + 3 e^2/8)
}
// sqrt(x) from y = 1/sqrt(x): one Markstein correction
__device__ __forceinline__ double sqrt_from_rsqrt(const double x, const double y) {
    const double s = x * y;
    return __fma_rn(__fma_rn(-s, s, x), 0.5 * y, s);
}

// Returns 0 ok (x, v advanced), nonzero: not handled here (state untouched).
__device__ __forceinline__ int kepler_elliptic_fast(double &x0, double &x1, double &x2, double &v0, double &v1,
                                                    double &v2, const double mu, const double h) {
    const double rr = __fma_rn(x2, x2, __fma_rn(x1, x1, x0 * x0));
    const double vv = __fma_rn(v2, v2, __fma_rn(v1, v1, v0 * v0));
    const double u = __fma_rn(x2, v2, __fma_rn(x1, v1, x0 * v0));
    if (!(rr > 1e-200 && rr < 1e200)) return 2;
    const double ir0 = rsqrt_fast(rr);
    const double r0 = sqrt_from_rsqrt(rr, ir0);
    const double imu = rcp_fast(mu);
    const double alpha = __fma_rn(-vv, imu, 2.0 * ir0);  // 1/a
    if (!(alpha > 1e-100 && alpha < 1e100)) return 2;
    const double a = rcp_fast(alpha);
    const double t = mu * alpha;
    const double irt = rsqrt_fast(t);                    // 1/sqrt(mu/a)
    const double n = alpha * sqrt_from_rsqrt(t, irt);    // sqrt(mu/a^3)
    const double inv_n = a * irt;
    const double sma = mu * irt;                         // sqrt(mu a)
    const double ec = __fma_rn(-r0, alpha, 1.0);
    const double es = u * (irt * alpha);                 // u / sqrt(mu a)
    double dM = n * h;
    dM = __fma_rn(-kTwoPi, rint(dM * (1.0 / kTwoPi)), dM);
    double dE = dM, S, C;
    sincos(0.5 * dE, &S, &C);
    const double omec = 1.0 - ec;
    bool converged = false;
#pragma unroll 1
    for (int it = 0; it < 8; ++it) {
        const double sd = 2.0 * S * C, cd = 2.0 * S * S;  // sin dE, 1 - cos dE
        const double F = __fma_rn(es, cd, __fma_rn(-ec, sd, dE - dM));
        const double Fp = __fma_rn(es, sd, __fma_rn(ec, cd, omec));          // r/a > 0
        const double Fpp = __fma_rn(es, 1.0 - cd, ec * sd);
        const double iFp = rcp_fast(Fp);
        const double dN = -F * iFp;                                          // Newton
        const double delta = __fma_rn(-dN, 0.5 * dN * Fpp * iFp, dN);        // Halley, expanded to first order
        if (!(fabs(delta) < 1.0)) return 1;                                  // wild step or NaN: leave it to the bracketed solver
        dE += delta;
        const double hh = 0.5 * delta;
        if (fabs(hh) <= 0.05) {
            // rotate (S, C) by hh: Taylor series, next terms hh^11/11! and hh^12/12! < 1e-22
            const double h2 = hh * hh;
            const double sh = hh * __fma_rn(h2, __fma_rn(h2, __fma_rn(h2, __fma_rn(h2, 1.0 / 362880.0, -1.0 / 5040.0), 1.0 / 120.0), -1.0 / 6.0), 1.0);
            const double chm1 = h2 * __fma_rn(h2, __fma_rn(h2, __fma_rn(h2, __fma_rn(h2, -1.0 / 3628800.0, 1.0 / 40320.0), -1.0 / 720.0), 1.0 / 24.0), -0.5);
            const double Sn = __fma_rn(C, sh, __fma_rn(S, chm1, S));
            const double Cn = __fma_rn(-S, sh, __fma_rn(C, chm1, C));
            S = Sn; C = Cn;
        } else {
            sincos(0.5 * dE, &S, &C);
        }
        // cubic convergence: once |delta| < 2e-7 the next correction is below 1e-18 even for e = 0.9
        if (fabs(delta) <= 2e-7 * fmax(1.0, fabs(dE))) { converged = true; break; }
    }
    if (!converged) return 1;
    const double sd = 2.0 * S * C, cd = 2.0 * S * S;
    const double Fp = __fma_rn(es, sd, __fma_rn(ec, cd, omec));  // r/a
    const double iFp = rcp_fast(Fp);
    const double ir = iFp * alpha;                               // 1/r
    const double f = __fma_rn(-(a * ir0), cd, 1.0);
    const double g = __fma_rn(r0 * alpha, sd, es * cd) * inv_n;
    const double fd = -sma * sd * ir * ir0;
    const double gd = __fma_rn(-iFp, cd, 1.0);
    if (!(isfinite(f) && isfinite(g) && isfinite(fd) && isfinite(gd))) return 1;
    const double n0 = __fma_rn(f, x0, g * v0), n1 = __fma_rn(f, x1, g * v1), n2 = __fma_rn(f, x2, g * v2);
    const double w0 = __fma_rn(fd, x0, gd * v0), w1 = __fma_rn(fd, x1, gd * v1), w2 = __fma_rn(fd, x2, gd * v2);
    x0 = n0; x1 = n1; x2 = n2;
    v0 = w0; v1 = w1; v2 = w2;
    return 0;
}

// Bound orbit (alpha = 2/r0 - v^2/mu > 0), differenced eccentric anomaly dE:
//   F(dE) = dE - ec sin dE + es (1 - cos dE) - dM = 0,  F' = r/a > 0
// Newton from dE = dM, kept inside a shrinking bracket [dM - 3e, dM + 3e] by bisection.
// Returns 0 ok, 1 not converged (state untouched), 2 not elliptic (state untouched).
__device__ __noinline__ int kepler_elliptic(double (&x)[3], double (&v)[3], const double mu, const double h) {
    const double r0 = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const double u = x[0] * v[0] + x[1] * v[1] + x[2] * v[2];
    const double alpha = 2.0 / r0 - v2 / mu;
    if (!(alpha > 0.0)) return 2;
    const double a = 1.0 / alpha;
    const double n = sqrt(mu / (a * a * a));
    const double ec = 1.0 - r0 / a;
    const double sma = sqrt(mu * a);
    const double es = u / sma;
    const double e = sqrt(ec * ec + es * es);
    double dM = n * h;
    dM = dM - kTwoPi * rint(dM / kTwoPi);
    double lo = dM - 3.0 * e, hi = dM + 3.0 * e;
    double dE = dM;
    bool converged = false;
    for (int it = 0; it < 64; ++it) {
        double sn, cs;
        sincos(dE, &sn, &cs);
        const double F = dE - ec * sn + es * (1.0 - cs) - dM;
        const double Fp = 1.0 - ec * cs + es * sn;
        if (F > 0.0) hi = dE; else lo = dE;
        double nxt = dE - F / Fp;
        if (!(nxt > lo && nxt < hi)) nxt = 0.5 * (lo + hi);
        const double delta = nxt - dE;
        dE = nxt;
        if (fabs(delta) <= kEps * fmax(1.0, fabs(dE))) { converged = true; break; }
    }
    if (!converged) return 1;
    const double sh = sin(0.5 * dE);
    const double c = 2.0 * sh * sh;  // 1 - cos dE without cancellation
    const double s = sin(dE);
    const double r = a * (1.0 - ec * (1.0 - c) + es * s);
    const double f = 1.0 - (a / r0) * c;
    const double g = ((r0 / a) * s + es * c) / n;
    const double fd = -sma * s / (r * r0);
    const double gd = 1.0 - (a / r) * c;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double xn = f * x[k] + g * v[k];
        const double vn = fd * x[k] + gd * v[k];
        x[k] = xn;
        v[k] = vn;
    }
    return 0;
}

// Stumpff functions c0..c3(z): quarter the argument until |z| <= 0.1, Taylor series, then the
// duplication formulas back up.
__device__ __forceinline__ void stumpff(double z, double &c0, double &c1, double &c2, double &c3) {
    int nq = 0;
    while (fabs(z) > 0.1) { z *= 0.25; ++nq; }
    double a2 = 0.5, a3 = 1.0 / 6.0, t2 = a2, t3 = a3;
#pragma unroll 1
    for (int k = 1; k < 12; ++k) {
        t2 *= -z / ((2.0 * k + 1.0) * (2.0 * k + 2.0));
        t3 *= -z / ((2.0 * k + 2.0) * (2.0 * k + 3.0));
        a2 += t2;
        a3 += t3;
    }
    double C2 = a2, C3 = a3, C1 = 1.0 - z * C3, C0 = 1.0 - z * C2;
    for (; nq > 0; --nq) {
        C3 = 0.25 * (C2 + C0 * C3);
        C2 = 0.5 * C1 * C1;
        C1 = C0 * C1;
        C0 = 2.0 * C0 * C0 - 1.0;
    }
    c0 = C0; c1 = C1; c2 = C2; c3 = C3;
}

// Any conic, universal variable s with G_k(s) = s^k c_k(beta s^2), beta = 2 mu/r0 - v^2:
//   h = r0 G1 + u G2 + mu G3   (dh/ds = r > 0),  r = r0 G0 + u G1 + mu G2,
//   f = 1 - (mu/r0) G2, g = h - mu G3, fdot = -(mu/(r r0)) G1, gdot = 1 - (mu/r) G2.
// Newton from s = h/r0 with an expanding bracket + bisection.  Returns 0 ok, 1 not converged.
__device__ __noinline__ int kepler_universal(double (&x)[3], double (&v)[3], const double mu, const double h) {
    const double r0 = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const double u = x[0] * v[0] + x[1] * v[1] + x[2] * v[2];
    const double beta = 2.0 * mu / r0 - v2;
    double s = h / r0;
    double lo = -INFINITY, hi = INFINITY;
    double c0, c1, c2, c3;
    bool converged = false;
#pragma unroll 1
    for (int it = 0; it < 200; ++it) {
        stumpff(beta * s * s, c0, c1, c2, c3);
        const double G1 = s * c1, G2 = s * s * c2, G3 = s * s * s * c3;
        const double F = r0 * G1 + u * G2 + mu * G3 - h;
        const double r = r0 * c0 + u * G1 + mu * G2;
        if (F > 0.0) hi = s; else lo = s;
        double nxt = s - F / r;
        if (!(nxt > lo && nxt < hi)) {
            if (isinf(lo)) nxt = (hi == 0.0) ? -1.0 : hi - 2.0 * fabs(hi) - 1e-3;
            else if (isinf(hi)) nxt = (lo == 0.0) ? 1.0 : lo + 2.0 * fabs(lo) + 1e-3;
            else nxt = 0.5 * (lo + hi);
        }
        const double delta = nxt - s;
        s = nxt;
        if (fabs(delta) <= kEps * fmax(fabs(s), fabs(h / r0))) { converged = true; break; }
    }
    if (!converged) return 1;
    stumpff(beta * s * s, c0, c1, c2, c3);
    const double G1 = s * c1, G2 = s * s * c2, G3 = s * s * s * c3;
    const double r = r0 * c0 + u * G1 + mu * G2;
    const double f = 1.0 - (mu / r0) * G2;
    const double g = h - mu * G3;
    const double fd = -(mu / (r * r0)) * G1;
    const double gd = 1.0 - (mu / r) * G2;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double xn = f * x[k] + g * v[k];
        const double vn = fd * x[k] + gd * v[k];
        x[k] = xn;
        v[k] = vn;
    }
    return 0;
}

}  // namespace nbk
