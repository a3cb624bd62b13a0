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
// correction.  Anything unusual (not bound or nearly parabolic, no convergence in 8 steps, non-finite)
// returns nonzero with the state untouched, and the caller falls back to the universal-variable solver
// below (a different formulation and a different iteration; the oracle's solvers are a third pair).

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
    if (!(alpha * r0 >= 0.05 && alpha < 1e100)) return 2;  // unbound or near-parabolic (r0/a < 0.05): universal variables
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

// ---- fall-back for everything the fast path declines: universal variables, Laguerre-Conway ------
// Any conic (bound, parabolic, hyperbolic), one formulation.  With beta = 2 mu/r0 - v^2, u = x.v and the
// universal functions G_k(s) = s^k c_k(beta s^2) (c_k: Stumpff functions), Kepler's equation reads
//     F(s) = r0 G1 + u G2 + mu G3 - h = 0,   F' = r = r0 G0 + u G1 + mu G2 > 0,   F'' = u G0 + (mu - beta r0) G1,
// and   f = 1 - (mu/r0) G2,  g = h - mu G3,  fdot = -(mu/(r r0)) G1,  gdot = 1 - (mu/r) G2.
// The Stumpff functions come from their closed forms (circular functions for z > 1, hyperbolic ones for
// z < -1, the power series in between), the root from Laguerre's iteration of order 5 (Conway's choice
// for Kepler's equation: cubically convergent near the root and, unlike Newton, not fooled by the
// exponential growth of F on a hyperbola or by the flat stretches of F near the pericentre of an
// eccentric orbit), started at s = h/r0 clipped to the large-s asymptote of a hyperbola.  An overflow
// (far beyond the root) halves s.  If 40 iterations do not settle, the interval [0, s_hi] is bisected
// (F is monotone, F(0) = -h).  Returns 0 ok, 1 not converged / non-finite input (state untouched).
__device__ __forceinline__ void stumpff_closed(const double z, double &c0, double &c1, double &c2, double &c3) {
    if (fabs(z) <= 1.0) {
        // c2 = sum_k (-z)^k / (2k+2)!,  c3 = sum_k (-z)^k / (2k+3)!;  k <= 10: next term < 1/24! ~ 2e-24
        const double w = -z;
        constexpr double k2[11] = {1.0 / 2.0, 1.0 / 24.0, 1.0 / 720.0, 1.0 / 40320.0, 1.0 / 3628800.0, 1.0 / 479001600.0, 1.0 / 87178291200.0, 1.0 / 20922789888000.0, 1.0 / 6402373705728000.0, 1.0 / 2432902008176640000.0, 1.0 / 1124000727777607680000.0};
        constexpr double k3[11] = {1.0 / 6.0, 1.0 / 120.0, 1.0 / 5040.0, 1.0 / 362880.0, 1.0 / 39916800.0, 1.0 / 6227020800.0, 1.0 / 1307674368000.0, 1.0 / 355687428096000.0, 1.0 / 121645100408832000.0, 1.0 / 51090942171709440000.0, 1.0 / 25852016738884976640000.0};
        double a2 = k2[10], a3 = k3[10];
#pragma unroll
        for (int k = 9; k >= 0; --k) { a2 = __fma_rn(a2, w, k2[k]); a3 = __fma_rn(a3, w, k3[k]); }  // Horner
        c2 = a2; c3 = a3;
        c1 = __fma_rn(-z, a3, 1.0);
        c0 = __fma_rn(-z, a2, 1.0);
    } else if (z > 0.0) {
        const double q = sqrt(z);
        double sn, cs, sh, ch;
        sincos(q, &sn, &cs);
        sincos(0.5 * q, &sh, &ch);
        c0 = cs; c1 = sn / q; c2 = 2.0 * sh * sh / z; c3 = (q - sn) / (z * q);
    } else {
        const double q = sqrt(-z);
        const double sh = sinh(q), hh = sinh(0.5 * q);
        c0 = cosh(q); c1 = sh / q; c2 = 2.0 * hh * hh / (-z); c3 = (sh - q) / ((-z) * q);
    }
}

__device__ __noinline__ int kepler_universal(double (&x)[3], double (&v)[3], const double mu, const double h) {
    const double r0 = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const double u = x[0] * v[0] + x[1] * v[1] + x[2] * v[2];
    const double beta = 2.0 * mu / r0 - v2;
    if (!(isfinite(beta) && isfinite(u) && r0 > 0.0 && isfinite(h))) return 1;
    if (h == 0.0) return 0;
    double s = h / r0;
    if (beta < 0.0) {
        // hyperbola: for large k|s| (k = sqrt(-beta)) F ~ mu sinh(k s)/k^3, so the root is near asinh(k^3 h/mu)/k
        const double k = sqrt(-beta);
        const double cap = 1.5 * asinh(k * k * k * fabs(h) / mu) / k + 1.0 / k;
        if (fabs(s) > cap) s = copysign(cap, h);
    }
    const double scale = fabs(h / r0);
    double c0, c1, c2, c3, G1 = 0.0, G2 = 0.0, G3 = 0.0, r = r0;
    bool converged = false;
    double prev = INFINITY;
#pragma unroll 1
    for (int it = 0; it < 40; ++it) {
        stumpff_closed(beta * s * s, c0, c1, c2, c3);
        G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
        const double F = r0 * G1 + u * G2 + mu * G3 - h;
        r = r0 * c0 + u * G1 + mu * G2;
        const double Fpp = u * c0 + (mu - beta * r0) * G1;
        if (!(isfinite(F) && isfinite(r) && isfinite(Fpp))) { s *= 0.5; prev = INFINITY; continue; }
        if (F == 0.0) { converged = true; break; }
        const double disc = fabs(16.0 * r * r - 20.0 * F * Fpp);
        const double den = r + copysign(sqrt(disc), r);
        const double ds = -5.0 * F / den;
        if (!isfinite(ds)) { s *= 0.5; prev = INFINITY; continue; }
        s += ds;
        const double tol = kEps * fmax(fabs(s), scale);
        // settled: the step is at rounding level, or it stopped shrinking while already tiny
        if (fabs(ds) <= 2.0 * tol || (fabs(ds) >= prev && prev <= 512.0 * tol)) { converged = true; break; }
        prev = fabs(ds);
    }
    if (!converged) {
        // last resort: bisection on the monotone F between 0 and an end found by doubling
        double lo = 0.0, hi = (h > 0.0) ? fmax(fabs(s), scale) : -fmax(fabs(s), scale);
        auto Fof = [&](const double ss) {
            stumpff_closed(beta * ss * ss, c0, c1, c2, c3);
            const double val = r0 * (ss * c1) + u * (ss * ss * c2) + mu * (ss * ss * ss * c3) - h;
            return isfinite(val) ? val : copysign(INFINITY, ss);
        };
        int guard = 0;
        while (Fof(hi) * h < 0.0 && ++guard < 64) hi *= 2.0;   // F(hi) must have the sign of h
        if (guard >= 64) return 1;
#pragma unroll 1
        for (int it = 0; it < 200; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (mid == lo || mid == hi) break;
            if (Fof(mid) * h < 0.0) lo = mid; else hi = mid;
        }
        s = 0.5 * (lo + hi);
    }
    stumpff_closed(beta * s * s, c0, c1, c2, c3);
    G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
    r = r0 * c0 + u * G1 + mu * G2;
    const double f = 1.0 - (mu / r0) * G2;
    const double g = h - mu * G3;
    const double fd = -(mu / (r * r0)) * G1;
    const double gd = 1.0 - (mu / r) * G2;
    if (!(isfinite(f) && isfinite(g) && isfinite(fd) && isfinite(gd))) return 1;
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
