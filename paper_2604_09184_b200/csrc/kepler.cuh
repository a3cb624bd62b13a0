// kepler.cuh -- H_A without encounters: per-body Kepler flow about mu = G M_star with Gauss' f and g
// functions ("a Keplerian orbit can be solved analytically"; Eq. 4 first sum;
// PAPER.md:98; the f/g form is fixed by BASELINE.json:north_star; solver details: DESIGN.md S15).
#pragma once
#include "nb_common.cuh"

namespace nbk {

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kEps = 2.220446049250313e-16;

// Bound orbit (alpha = 2/r0 - v^2/mu > 0), differenced eccentric anomaly dE:
//   F(dE) = dE - ec sin dE + es (1 - cos dE) - dM = 0,  F' = r/a > 0
// Newton from dE = dM, kept inside a shrinking bracket [dM - 3e, dM + 3e] by bisection.
// Returns 0 ok, 1 not converged (state untouched), 2 not elliptic (state untouched).
__device__ __forceinline__ int kepler_elliptic(double (&x)[3], double (&v)[3], const double mu, const double h) {
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
