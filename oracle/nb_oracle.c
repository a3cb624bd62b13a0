/*
 * nb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of the hot path of the hybrid symplectic
 * integrator in Grimm & Stadel (arxiv 2604.09184; /root/reference/PAPER.md):
 *   - changeover weight W            PAPER.md:94            (shape: DESIGN.md reading S2)
 *   - critical radius                PAPER.md:94-96, Eq. 7  (R_Hill: reading S5)
 *   - H_B kick, O(N^2)               PAPER.md:86 Eq. 5, 98  (force weighting: readings S1, S3)
 *   - close-encounter pair list      PAPER.md:94, 98, 106   (r_crit,ij = max: reading S4)
 *   - H_C shift                      PAPER.md:91-92 Eq. 6
 *   - H_A Kepler drift, Gauss f,g    PAPER.md:64, 98        (solver: reading S15)
 *   - step  B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2)           PAPER.md:80 Eq. 3 (order: S6, S17)
 *   - diagnostics E, L               PAPER.md:84-92 Eq. 4-6 (K terms cancel in H_A + H_B)
 *   - independent encounter groups   PAPER.md:106           (connected components of the pair graph)
 *   - collisions inside the direct solver  PAPER.md:98, 130, 168  (reading S26; "parity unpinned" against the paper)
 *
 * It is the definition written out: explicit loops in the paper's index order, no blocking,
 * no fusion, no FMA contraction (build with -ffp-contract=off).  All inputs and outputs are
 * fp64.  O(N) sums are Neumaier-compensated, and the O(N^2) acceleration sum carries its terms
 * in `long double` before one final rounding to fp64, so that the whole 1e-12 error budget
 * belongs to the CUDA path.  HOST DEPENDENCE: this relies on x86-64, where `long double` is the
 * x87 80-bit format (64-bit significand); oracle_long_double_digits() reports LDBL_MANT_DIG and
 * a test requires >= 64 -- on a host whose long double is plain fp64 the oracle would still be
 * the definition, only with its own rounding (~sqrt(N) eps) inside the tolerance it arbitrates.
 * It is an extended-precision checker, not a tuned CPU kernel: its interactions/s understate
 * what a vectorised fp64 CPU code would do by several times.  Decisions that produce integers
 * (the pair test r^2 < rc^2) are taken in plain fp64.  OpenMP parallelises over the OUTER body
 * index i only; every per-body sum runs sequentially in j order.
 *
 * It shares no code, header, table or helper with paper_2604_09184_b200/ (the CUDA path) and
 * neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): every exported function is pinned by closed
 * forms, invariants or brute force; the SHAPE of W between its end points, the max() rule for
 * r_crit,ij and force-vs-potential weighting are "parity unpinned" against the paper (the
 * paper gives no formula for them) -- see DESIGN.md.
 */
#include <float.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.141592653589793238462643383279502884

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* significand bits of the type the O(N^2) sum is carried in (64 on x86-64: x87 extended) */
int oracle_long_double_digits(void) { return LDBL_MANT_DIG; }

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Neumaier's compensated summation: (sum, comp) += t. */
static inline void neumaier_add(double *sum, double *comp, double t) {
    double s = *sum + t;
    if (fabs(*sum) >= fabs(t)) *comp += (*sum - s) + t;
    else                       *comp += (t - s) + *sum;
    *sum = s;
}

/* ------------------------------------------------------------------------------------------
 * Changeover / kick weight W(r; rc)  -- PAPER.md:94 "smooth changeover function ranging from
 * 0 to 1"; the changeover "starts to act" at the critical radius.  Reading S1: W = 1 far
 * (r >= rc), W = 0 close (r <= 0.1 rc).  Reading S2: between, with y = (r-0.1rc)/(0.9rc),
 *   kind 0: K_C(y) = y^2 / (2y^2 - 2y + 1)       (form of the hybrid scheme the paper cites [9])
 *   kind 1: 10y^3 - 15y^4 + 6y^5                 (quintic smoothstep, alternative)
 * ------------------------------------------------------------------------------------------ */
double oracle_changeover(double r, double rc, int kind) {
    if (!(r < rc)) return 1.0;            /* r >= rc; also rc == 0 */
    double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    if (kind == 1) return y * y * y * (10.0 + y * (-15.0 + 6.0 * y));
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
}

/* ------------------------------------------------------------------------------------------
 * Critical radius, Eq. 7:  rc_i = max(n1 R_Hill,i , n2 dt v_i),  n1 = 3, n2 = 0.4.
 * Reading S5: R_Hill,i = a_i (m_i / (3 M_star))^(1/3), a_i from vis-viva with the stored
 * (barycentric) velocity, 1/a = 2/r - v^2/(G M_star); if 1/a <= 0 use a_i = r_i.
 * |dt| is used so that a backward step sees the same radius.
 * ------------------------------------------------------------------------------------------ */
void oracle_rcrit(const double *x, const double *v, const double *m, double M_star, int64_t N,
                  double dt, double G, double n1, double n2, double *rcrit) {
    for (int64_t i = 0; i < N; ++i) {
        double xi = x[3 * i], yi = x[3 * i + 1], zi = x[3 * i + 2];
        double vx = v[3 * i], vy = v[3 * i + 1], vz = v[3 * i + 2];
        double r = sqrt((xi * xi + yi * yi) + zi * zi);
        double v2 = (vx * vx + vy * vy) + vz * vz;
        double inva = 2.0 / r - v2 / (G * M_star);
        double a = (inva > 0.0) ? 1.0 / inva : r;
        double rh = a * cbrt(m[i] / (3.0 * M_star));
        double t1 = n1 * rh;
        double t2 = n2 * fabs(dt) * sqrt(v2);
        rcrit[i] = (t1 > t2) ? t1 : t2;
    }
}

/* ------------------------------------------------------------------------------------------
 * H_B accelerations (Eq. 5; "H_B describes the N^2 mutual
 * gravitational force terms"; BASELINE.json:north_star):
 *     a_i = sum_{j != i, j < n_active} G m_j W(r_ij; rc_ij) (x_j - x_i) / r_ij^3
 * rc_ij = max(rc_i, rc_j) (S4).  The weight multiplies the force (S3).  r_ij^2 is formed as
 * (dx*dx + dy*dy) + dz*dz.  S10: the self term is skipped; W = 0 contributes exactly 0 (so a
 * coincident pair with rc_ij > 0 never forms 0 * inf); a coincident pair with rc_ij == 0 is
 * counted in *n_singular and contributes 0.
 * Semi-active mode (north_star; not in the paper): j runs over the first n_active bodies only.
 * rows == NULL: all i = 0..N-1 (acc is [N,3]); otherwise only the listed rows (acc is [nrows,3]).
 * abs_sum (optional, same shape as acc): sum_j |term| per component, for the conditioning-aware
 * error report.
 * ------------------------------------------------------------------------------------------ */
static long double changeover_ext(long double r, long double rc, int kind) {
    if (!(r < rc)) return 1.0L;
    long double y = (r - 0.1L * rc) / (0.9L * rc);
    if (y <= 0.0L) return 0.0L;
    if (y >= 1.0L) return 1.0L;
    if (kind == 1) return y * y * y * (10.0L + y * (-15.0L + 6.0L * y));
    return (y * y) / (2.0L * y * y - 2.0L * y + 1.0L);
}

void oracle_accel(const double *x, const double *m, const double *rcrit, int64_t N,
                  int64_t n_active, double G, int kind, const int64_t *rows, int64_t nrows,
                  double *acc, double *abs_sum, int64_t *n_singular) {
    /* Every term and the three running sums are carried in the host's extended precision
       (x87 long double, 64-bit significand) and rounded to fp64 once at the end, so that the
       oracle's own rounding is far below the 1e-12 per-component tolerance it arbitrates. */
    int64_t nr = rows ? nrows : N;
    int64_t nsing = 0;
    if (n_active <= 0 || n_active > N) n_active = N;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : nsing)
    for (int64_t k = 0; k < nr; ++k) {
        int64_t i = rows ? rows[k] : k;
        long double xi = x[3 * i], yi = x[3 * i + 1], zi = x[3 * i + 2];
        long double rci = rcrit ? rcrit[i] : 0.0;
        long double sx = 0, sy = 0, sz = 0;
        long double bx = 0, by = 0, bz = 0;
        for (int64_t j = 0; j < n_active; ++j) {
            if (j == i) continue;
            long double dx = x[3 * j] - xi, dy = x[3 * j + 1] - yi, dz = x[3 * j + 2] - zi;
            long double r2 = (dx * dx + dy * dy) + dz * dz;
            long double rcj = rcrit ? rcrit[j] : 0.0;
            long double rc = (rci > rcj) ? rci : rcj;
            long double r = sqrtl(r2);
            long double W = changeover_ext(r, rc, kind);
            if (W == 0.0L) continue;
            if (r2 == 0.0L) { nsing++; continue; }   /* only reachable with rc == 0 */
            long double f = (long double)G * m[j] * W / (r2 * r);
            long double tx = f * dx, ty = f * dy, tz = f * dz;
            sx += tx; sy += ty; sz += tz;
            bx += fabsl(tx); by += fabsl(ty); bz += fabsl(tz);
        }
        acc[3 * k] = (double)sx; acc[3 * k + 1] = (double)sy; acc[3 * k + 2] = (double)sz;
        if (abs_sum) { abs_sum[3 * k] = (double)bx; abs_sum[3 * k + 1] = (double)by; abs_sum[3 * k + 2] = (double)bz; }
    }
    if (n_singular) *n_singular = nsing;
}

/* Kick: acc <- a(x); v_i += dt * a_i. */
void oracle_kick(const double *x, double *v, const double *m, int64_t N, int64_t n_active,
                 double dt, const double *rcrit, double G, int kind, double *acc) {
    oracle_accel(x, m, rcrit, N, n_active, G, kind, NULL, 0, acc, NULL, NULL);
    for (int64_t i = 0; i < 3 * N; ++i) v[i] = v[i] + dt * acc[i];
}

/* ------------------------------------------------------------------------------------------
 * Close-encounter pairs ("critical radius describes the separation distance ...
 * when the changeover starts to act"): every unordered {i,j} with
 * r_ij < rc_ij = max(rc_i, rc_j), emitted once as (min,max) (S11, S12).  Semi-active: at
 * least one member must be active (index < n_active) (S13).
 * The north_star tolerance clause ("pairs within 1e-12 relative of the r_crit threshold ...
 * listed separately") is applied in r^2 (tol2 = 2e-12):
 *    sure        r^2 <  rc^2 (1 - tol2)
 *    borderline  |r^2/rc^2 - 1| <= tol2
 * rows == NULL: all pairs.  rows != NULL: pairs incident to the listed bodies (each (min,max)
 * may then appear once per listed member; the caller de-duplicates).
 * Output order is unspecified (the caller sorts).  Counts keep counting past the capacities.
 * ------------------------------------------------------------------------------------------ */
void oracle_pairs(const double *x, const double *rcrit, int64_t N, int64_t n_active,
                  double tol2, const int64_t *rows, int64_t nrows,
                  int32_t *sure, int64_t cap_sure, int64_t *n_sure,
                  int32_t *border, int64_t cap_border, int64_t *n_border) {
    int64_t ns = 0, nb = 0;
    if (n_active <= 0 || n_active > N) n_active = N;
    int64_t nr = rows ? nrows : n_active;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < nr; ++k) {
        int64_t i = rows ? rows[k] : k;
        double xi = x[3 * i], yi = x[3 * i + 1], zi = x[3 * i + 2];
        double rci = rcrit[i];
        /* full list: j > i (i is active since i < n_active);
           row list : all j != i with at least one of (i,j) active */
        int64_t j0 = rows ? 0 : i + 1;
        int64_t j1 = (rows && i >= n_active) ? n_active : N;
        for (int64_t j = j0; j < j1; ++j) {
            if (j == i) continue;
            double dx = x[3 * j] - xi, dy = x[3 * j + 1] - yi, dz = x[3 * j + 2] - zi;
            double r2 = (dx * dx + dy * dy) + dz * dz;
            double rcj = rcrit[j];
            double rc = (rci > rcj) ? rci : rcj;
            double rc2 = rc * rc;
            int is_sure = r2 < rc2 * (1.0 - tol2);
            int is_border = !is_sure && (fabs(r2 / rc2 - 1.0) <= tol2);
            if (!is_sure && !is_border) continue;
            int32_t lo = (int32_t)(i < j ? i : j), hi = (int32_t)(i < j ? j : i);
#pragma omp critical(oracle_pairs_append)
            {
                if (is_sure) {
                    if (ns < cap_sure) { sure[2 * ns] = lo; sure[2 * ns + 1] = hi; }
                    ns++;
                } else {
                    if (nb < cap_border) { border[2 * nb] = lo; border[2 * nb + 1] = hi; }
                    nb++;
                }
            }
        }
    }
    *n_sure = ns;
    *n_border = nb;
}

/* ------------------------------------------------------------------------------------------
 * H_C (Eq. 6): H_C = (sum p_i)^2 / (2 m_0)  =>  every heliocentric position
 * moves by  dt * (sum_i m_i v_i) / M_star.  Sum in index order, compensated.
 * ------------------------------------------------------------------------------------------ */
void oracle_shift(double *x, const double *v, const double *m, double M_star, int64_t N,
                  double dt) {
    double s[3] = {0, 0, 0}, c[3] = {0, 0, 0};
    for (int64_t i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) neumaier_add(&s[k], &c[k], m[i] * v[3 * i + k]);
    for (int k = 0; k < 3; ++k) s[k] = (s[k] + c[k]) / M_star;
    for (int64_t i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) x[3 * i + k] = x[3 * i + k] + dt * s[k];
}

/* ------------------------------------------------------------------------------------------
 * H_A without encounters: Kepler flow about mu = G M_star ("a Keplerian orbit can
 * be solved analytically"; Eq. 4 first sum), advanced with Gauss'
 * f and g functions (BASELINE.json:north_star).
 *
 * Elliptic solver (alpha = 2/r0 - v^2/mu with alpha r0 >= 0.05), in the differenced eccentric anomaly dE:
 *   a = 1/alpha, n = sqrt(mu/a^3), ec = 1 - r0/a, es = (x.v)/sqrt(mu a),
 *   dM = n h reduced to (-pi, pi],
 *   F(dE) = dE - ec sin dE + es (1 - cos dE) - dM = 0,   F' = r/a > 0   (unique root),
 *   Newton from dE = dM safeguarded by bisection on [dM - 3e, dM + 3e],
 *   c = 2 sin^2(dE/2), s = sin dE, r = a (1 - ec (1 - c) + es s),
 *   f = 1 - (a/r0) c,  g = [(r0/a) s + es c]/n,  fdot = -sqrt(mu a) s/(r r0),  gdot = 1 - (a/r) c.
 * The elliptic elements lose their meaning as the orbit approaches a parabola (a -> inf: ec -> 1, n h -> 0, and
 * for alpha = O(eps) by rounding alone the formulas return garbage without noticing -- found by the pin against
 * numerical integration, tests/test_oracle_pins.py): this solver takes only orbits with r0/a >= 0.05 (every
 * bound orbit with e <= 0.95 at any phase); the rest goes to the universal-variable solver, which is uniformly
 * accurate across the parabola (reading S15).
 * Returns 0 on convergence, 1 if 64 iterations did not reach the fixed point (state then
 * left unchanged), 2 if not handled here: unbound or near-parabolic (state unchanged).
 * ------------------------------------------------------------------------------------------ */
int oracle_kepler_elliptic(double *x, double *v, double mu, double h) {
    double r0 = sqrt((x[0] * x[0] + x[1] * x[1]) + x[2] * x[2]);
    double v2 = (v[0] * v[0] + v[1] * v[1]) + v[2] * v[2];
    double u = (x[0] * v[0] + x[1] * v[1]) + x[2] * v[2];
    double alpha = 2.0 / r0 - v2 / mu;
    if (!(alpha * r0 >= 0.05)) return 2;   /* unbound or near-parabolic (r0/a < 0.05): universal variables */
    double a = 1.0 / alpha;
    double n = sqrt(mu / (a * a * a));
    double ec = 1.0 - r0 / a;
    double es = u / sqrt(mu * a);
    double e = sqrt(ec * ec + es * es);
    double dM = n * h;
    dM = dM - 2.0 * ORACLE_PI * nearbyint(dM / (2.0 * ORACLE_PI));
    double lo = dM - 3.0 * e, hi = dM + 3.0 * e;
    double dE = dM;
    int converged = 0;
    for (int it = 0; it < 64; ++it) {
        double sn = sin(dE), cs = cos(dE);
        double F = dE - ec * sn + es * (1.0 - cs) - dM;
        double Fp = 1.0 - ec * cs + es * sn;
        if (F > 0.0) hi = dE; else lo = dE;
        double step = F / Fp;
        double nxt = dE - step;
        if (!(nxt > lo && nxt < hi)) nxt = 0.5 * (lo + hi);   /* bisection safeguard */
        double delta = nxt - dE;
        dE = nxt;
        if (fabs(delta) <= 2.220446049250313e-16 * fmax(1.0, fabs(dE))) { converged = 1; break; }
    }
    if (!converged) return 1;
    double sh = sin(0.5 * dE);
    double c = 2.0 * sh * sh;
    double s = sin(dE);
    double r = a * (1.0 - ec * (1.0 - c) + es * s);
    double f = 1.0 - (a / r0) * c;
    double g = ((r0 / a) * s + es * c) / n;
    double fd = -sqrt(mu * a) * s / (r * r0);
    double gd = 1.0 - (a / r) * c;
    for (int k = 0; k < 3; ++k) {
        double xn = f * x[k] + g * v[k];
        double vn = fd * x[k] + gd * v[k];
        x[k] = xn; v[k] = vn;
    }
    return 0;
}

/* Stumpff functions c0..c3 of z (Danby's argument-quartering + series + duplication). */
static void stumpff(double z, double *c0, double *c1, double *c2, double *c3) {
    int nq = 0;
    if (!isfinite(z)) { *c0 = *c1 = *c2 = *c3 = NAN; return; }   /* the caller treats it as "beyond the root" */
    while (fabs(z) > 0.1) { z *= 0.25; nq++; }
    /* series: c2 = sum (-z)^k/(2k+2)!, c3 = sum (-z)^k/(2k+3)! */
    double a2 = 1.0 / 2.0, a3 = 1.0 / 6.0, t2 = a2, t3 = a3;
    for (int k = 1; k < 12; ++k) {
        t2 *= -z / ((2.0 * k + 1.0) * (2.0 * k + 2.0));
        t3 *= -z / ((2.0 * k + 2.0) * (2.0 * k + 3.0));
        a2 += t2; a3 += t3;
    }
    double C2 = a2, C3 = a3, C1 = 1.0 - z * C3, C0 = 1.0 - z * C2;
    for (; nq > 0; --nq) {
        C3 = 0.25 * (C2 + C0 * C3);
        C2 = 0.5 * C1 * C1;
        C1 = C0 * C1;
        C0 = 2.0 * C0 * C0 - 1.0;
    }
    *c0 = C0; *c1 = C1; *c2 = C2; *c3 = C3;
}

/* Universal-variable solver (any conic; second, independent route -- also the fallback when
 * alpha <= 0, S15).  With beta = 2 mu/r0 - v^2, G_k(s) = s^k c_k(beta s^2), u = x.v:
 *    h = r0 G1 + u G2 + mu G3            (universal Kepler equation, dF/ds = r > 0)
 *    r = r0 G0 + u G1 + mu G2
 *    f = 1 - (mu/r0) G2, g = h - mu G3, fdot = -(mu/(r r0)) G1, gdot = 1 - (mu/r) G2.
 * F(s) = r0 G1 + u G2 + mu G3 - h is strictly increasing with F(0) = -h, so the root lies on the
 * side of sign(h): the bracket starts as [0, +inf) or (-inf, 0].  Newton from s = h/r0, safeguarded
 * the textbook way: a Newton step is taken only if it stays inside the bracket AND is at most half
 * the previous step; otherwise the bracket is expanded (while one end is infinite) or bisected.  On
 * a strongly hyperbolic orbit F grows like exp(sqrt(-beta) s): plain Newton from far beyond the root
 * creeps by 1/sqrt(-beta) per step, the half-step rule sends those iterations to bisection.  A
 * non-finite F or r (overflow far beyond the root) counts as "beyond the root".
 * Returns 0 ok, 1 not converged (state unchanged). */
int oracle_kepler_universal(double *x, double *v, double mu, double h) {
    double r0 = sqrt((x[0] * x[0] + x[1] * x[1]) + x[2] * x[2]);
    double v2 = (v[0] * v[0] + v[1] * v[1]) + v[2] * v[2];
    double u = (x[0] * v[0] + x[1] * v[1]) + x[2] * v[2];
    double beta = 2.0 * mu / r0 - v2;
    double s = h / r0;
    double lo = (h > 0.0) ? 0.0 : -INFINITY, hi = (h < 0.0) ? 0.0 : INFINITY;
    double c0, c1, c2, c3, G0 = 1, G1 = 0, G2 = 0, G3 = 0, r = r0;
    double prev = INFINITY;                       /* size of the previous step */
    int converged = 0;
    if (h == 0.0) return 0;
    for (int it = 0; it < 300; ++it) {
        stumpff(beta * s * s, &c0, &c1, &c2, &c3);
        G0 = c0; G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
        double F = r0 * G1 + u * G2 + mu * G3 - h;
        r = r0 * G0 + u * G1 + mu * G2;
        if (!isfinite(F) || !isfinite(r)) { F = (s > 0.0) ? INFINITY : -INFINITY; r = NAN; }
        if (F == 0.0) { converged = 1; break; }
        if (F > 0.0) hi = s; else lo = s;
        const double scale = 2.220446049250313e-16 * fmax(fabs(s), fabs(h / r0));
        double nxt = s - F / r;                    /* Newton */
        if (fabs(nxt - s) <= scale) { s = nxt; converged = 1; break; }   /* F is monotone: s is the root to rounding */
        if (!(nxt > lo && nxt < hi) || 2.0 * fabs(nxt - s) > prev) {
            if (isinf(lo)) nxt = hi - 2.0 * fabs(hi) - 1e-3;
            else if (isinf(hi)) nxt = lo + 2.0 * fabs(lo) + 1e-3;
            else nxt = 0.5 * (lo + hi);
        }
        prev = fabs(nxt - s);
        if (prev <= scale) { s = nxt; converged = 1; break; }            /* the bracket has collapsed */
        s = nxt;
    }
    if (!converged) return 1;
    stumpff(beta * s * s, &c0, &c1, &c2, &c3);
    G0 = c0; G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
    r = r0 * G0 + u * G1 + mu * G2;
    double f = 1.0 - (mu / r0) * G2;
    double g = h - mu * G3;
    double fd = -(mu / (r * r0)) * G1;
    double gd = 1.0 - (mu / r) * G2;
    if (!(isfinite(f) && isfinite(g) && isfinite(fd) && isfinite(gd))) return 1;
    for (int k = 0; k < 3; ++k) {
        double xn = f * x[k] + g * v[k];
        double vn = fd * x[k] + gd * v[k];
        x[k] = xn; v[k] = vn;
    }
    return 0;
}

/* Drift every body: elliptic solver when bound, universal variables otherwise (S15).
 * solver: 0 = as described, 1 = force the universal solver for every body (cross-check).
 * Returns the number of bodies that failed to converge (left unchanged). */
int64_t oracle_drift_kepler(double *x, double *v, double M_star, int64_t N, double dt, double G,
                            int solver) {
    double mu = G * M_star;
    int64_t nfail = 0;
#pragma omp parallel for schedule(static) reduction(+ : nfail)
    for (int64_t i = 0; i < N; ++i) {
        int rcode = 2;
        if (solver == 0) rcode = oracle_kepler_elliptic(x + 3 * i, v + 3 * i, mu, dt);
        if (rcode == 2) rcode = oracle_kepler_universal(x + 3 * i, v + 3 * i, mu, dt);
        if (rcode != 0) nfail++;
    }
    return nfail;
}

/* ------------------------------------------------------------------------------------------
 * One run of nsteps steps (Eq. 3; order S6: B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2)).
 * S17: r_crit is recomputed from the current (x, v) immediately before every force
 * evaluation (skipped when n1 == n2 == 0: the caller's rcrit is used unchanged); the closing
 * half-kick of step n and the opening half-kick of step n+1 share that evaluation.
 * On return acc / rcrit are those of the last evaluation (at the final positions).
 * Returns the number of Kepler non-convergences.
 * ------------------------------------------------------------------------------------------ */
int64_t oracle_step(double *x, double *v, const double *m, double M_star, int64_t N,
                    int64_t n_active, double dt, double G, double n1, double n2, int kind,
                    double *rcrit, double *acc, int64_t nsteps) {
    int64_t nfail = 0;
    int update_rc = !(n1 == 0.0 && n2 == 0.0);
    if (update_rc) oracle_rcrit(x, v, m, M_star, N, dt, G, n1, n2, rcrit);
    oracle_accel(x, m, rcrit, N, n_active, G, kind, NULL, 0, acc, NULL, NULL);
    for (int64_t st = 0; st < nsteps; ++st) {
        for (int64_t i = 0; i < 3 * N; ++i) v[i] = v[i] + (0.5 * dt) * acc[i];
        oracle_shift(x, v, m, M_star, N, 0.5 * dt);
        nfail += oracle_drift_kepler(x, v, M_star, N, dt, G, 0);
        oracle_shift(x, v, m, M_star, N, 0.5 * dt);
        if (update_rc) oracle_rcrit(x, v, m, M_star, N, dt, G, n1, n2, rcrit);
        oracle_accel(x, m, rcrit, N, n_active, G, kind, NULL, 0, acc, NULL, NULL);
        for (int64_t i = 0; i < 3 * N; ++i) v[i] = v[i] + (0.5 * dt) * acc[i];
    }
    return nfail;
}

/* ------------------------------------------------------------------------------------------
 * Diagnostics.  E = H_A + H_B + H_C with the K terms cancelling (Eq. 4-6):
 *   E = sum 1/2 m_i v_i^2 + |sum m_i v_i|^2/(2 M_star) - sum G M_star m_i/r_i
 *       - sum_{i<j} G m_i m_j / r_ij
 * L = sum m_i x_i cross v_i.   out = {E, Lx, Ly, Lz, T_bodies, T_star, U_star, U_mutual}.
 * Bodies with m == 0 contribute nothing.
 * ------------------------------------------------------------------------------------------ */
void oracle_diagnostics(const double *x, const double *v, const double *m, double M_star,
                        int64_t N, double G, double *out) {
    double T = 0, Tc = 0, Us = 0, Usc = 0;
    double p[3] = {0, 0, 0}, pc[3] = {0, 0, 0}, L[3] = {0, 0, 0}, Lc[3] = {0, 0, 0};
    for (int64_t i = 0; i < N; ++i) {
        const double *xi = x + 3 * i, *vi = v + 3 * i;
        double v2 = (vi[0] * vi[0] + vi[1] * vi[1]) + vi[2] * vi[2];
        double r = sqrt((xi[0] * xi[0] + xi[1] * xi[1]) + xi[2] * xi[2]);
        neumaier_add(&T, &Tc, 0.5 * m[i] * v2);
        if (m[i] != 0.0) neumaier_add(&Us, &Usc, -G * M_star * m[i] / r);
        for (int k = 0; k < 3; ++k) neumaier_add(&p[k], &pc[k], m[i] * vi[k]);
        neumaier_add(&L[0], &Lc[0], m[i] * (xi[1] * vi[2] - xi[2] * vi[1]));
        neumaier_add(&L[1], &Lc[1], m[i] * (xi[2] * vi[0] - xi[0] * vi[2]));
        neumaier_add(&L[2], &Lc[2], m[i] * (xi[0] * vi[1] - xi[1] * vi[0]));
    }
    /* mutual potential: one compensated row sum per i (parallel over i), rows added in index order */
    double *row = (double *)calloc((size_t)(N > 0 ? N : 1), sizeof(double));
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        if (m[i] == 0.0) continue;
        double si = 0, ci = 0;
        for (int64_t j = i + 1; j < N; ++j) {
            if (m[j] == 0.0) continue;
            double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1],
                   dz = x[3 * j + 2] - x[3 * i + 2];
            double r = sqrt((dx * dx + dy * dy) + dz * dz);
            neumaier_add(&si, &ci, -G * m[i] * m[j] / r);
        }
        row[i] = si + ci;
    }
    double Um = 0, Umc = 0;
    for (int64_t i = 0; i < N; ++i) neumaier_add(&Um, &Umc, row[i]);
    free(row);
    double px = p[0] + pc[0], py = p[1] + pc[1], pz = p[2] + pc[2];
    double Ts = ((px * px + py * py) + pz * pz) / (2.0 * M_star);
    out[4] = T + Tc; out[5] = Ts; out[6] = Us + Usc; out[7] = Um + Umc;
    out[0] = ((out[4] + out[5]) + out[6]) + out[7];
    out[1] = L[0] + Lc[0]; out[2] = L[1] + Lc[1]; out[3] = L[2] + Lc[2];
}


/* ---------------------------------------------------------------------------------------------
 * Independent close-encounter groups ("finding independent close encounter groups
 * and integrating them independently"; the direct solver "propagates the involved
 * bodies through the close encounter phase").  Two bodies belong to the same group when a chain of
 * close-encounter pairs connects them: the groups are the connected components of the undirected
 * graph (bodies, pairs).  This is the textbook statement: breadth-first search from every not yet
 * visited body, taken in index order, over adjacency lists.
 *
 *   pairs  [npairs,2] int32 (any order inside a pair, duplicates allowed)
 *   label  [N]  out: smallest body index of the body's group (a body without pairs: itself)
 *   members[N]  out: the bodies of all groups with >= 2 members, group after group, groups ordered by
 *               label, members ascending inside a group; the tail is filled with -1
 *   gstart [N/2 + 2] out: members[gstart[g] .. gstart[g+1]) is group g; entries past ngroups+1: -1
 *   gstat  [4]  out: number of groups (>= 2 members), number of member bodies, largest group,
 *               number of pairs read
 * Returns 0, or -1 if a pair holds an index outside [0, N) or i == j.
 */
static int cmp_i32(const void *a, const void *b) {
    const int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

int oracle_groups(const int32_t *pairs, int64_t npairs, int64_t N, int32_t *label, int32_t *members,
                  int32_t *gstart, int64_t *gstat) {
    int64_t *deg = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
    for (int64_t k = 0; k < npairs; ++k) {
        const int64_t a = pairs[2 * k], b = pairs[2 * k + 1];
        if (a < 0 || b < 0 || a >= N || b >= N || a == b) { free(deg); return -1; }
        deg[a + 1]++; deg[b + 1]++;
    }
    for (int64_t i = 0; i < N; ++i) deg[i + 1] += deg[i];              /* CSR offsets */
    int32_t *adj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(2 * npairs + 1));
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N + 1));
    memcpy(fill, deg, sizeof(int64_t) * (size_t)(N + 1));
    for (int64_t k = 0; k < npairs; ++k) {
        const int32_t a = pairs[2 * k], b = pairs[2 * k + 1];
        adj[fill[a]++] = b; adj[fill[b]++] = a;
    }
    int32_t *queue = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N + 1));
    for (int64_t i = 0; i < N; ++i) { label[i] = -1; members[i] = -1; }
    for (int64_t g = 0; g < N / 2 + 2; ++g) gstart[g] = -1;
    int64_t ngroups = 0, nmembers = 0, largest = 0;
    for (int64_t i = 0; i < N; ++i) {
        if (label[i] >= 0) continue;
        label[i] = (int32_t)i;                    /* i is the smallest index of a new group */
        if (deg[i + 1] == deg[i]) continue;       /* no pairs: a group of one, not listed */
        int64_t head = 0, tail = 0;
        queue[tail++] = (int32_t)i;
        while (head < tail) {
            const int32_t a = queue[head++];
            for (int64_t e = deg[a]; e < deg[a + 1]; ++e) {
                const int32_t b = adj[e];
                if (label[b] < 0) { label[b] = (int32_t)i; queue[tail++] = b; }
            }
        }
        qsort(queue, (size_t)tail, sizeof(int32_t), cmp_i32);
        gstart[ngroups] = (int32_t)nmembers;
        for (int64_t k = 0; k < tail; ++k) members[nmembers + k] = queue[k];
        nmembers += tail;
        ngroups++;
        if (tail > largest) largest = tail;
    }
    gstart[ngroups] = (int32_t)nmembers;
    gstat[0] = ngroups; gstat[1] = nmembers; gstat[2] = largest; gstat[3] = npairs;
    free(deg); free(adj); free(fill); free(queue);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Close-encounter propagation of one group (Eq. 4: H_A = Kepler terms + the pair terms
 * weighted by [1 - K]; "when there is a close encounter, a direct solver is needed which
 * propagates the involved bodies through the close encounter phase ... must not necessarily be
 * symplectic"; groups are integrated independently).
 *
 * Equations of motion of the n members of a group under H_A (democratic coordinates; the weight
 * multiplies the force, reading S3, so that kick + this = the full Newtonian pair force):
 *     dx_i/dt = v_i
 *     dv_i/dt = - G M_star x_i / r_i^3 + sum_{j in group, j != i} G m_j [1 - W(r_ij; rc_ij)] (x_j - x_i) / r_ij^3
 * with W the kick weight of oracle_changeover and rc_ij = max(rc_i, rc_j) (S4), rc held fixed.
 *
 * Integrator (the paper prescribes none; reading S19): Bulirsch-Stoer -- Gragg's modified
 * midpoint rule with 2, 4, ..., 16 substeps, polynomial (Aitken-Neville) extrapolation in h^2, at
 * most 8 columns.  Error of a column = max over members of |dx|^2/|x|^2 and |dv|^2/max(|v|^2, mu/|x|)
 * between the last two diagonal entries (x, v at the start of the step), accepted when <= tol^2.  Step control: accepted in <= 6 columns: next
 * h = 1.3 h; in 8 columns: next h = 0.55 h; not accepted after 8 columns: retry with h/2.  The first
 * trial step is the whole interval.  Returns the number of accepted steps, or -1 if h underflows.
 * --------------------------------------------------------------------------------------------- */
static double one_minus_changeover(double r, double rc, int kind) {
    if (!(r < rc)) return 0.0;
    double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 1.0;
    if (y >= 1.0) return 0.0;
    double z = 1.0 - y;
    if (kind == 1) return z * z * z * (1.0 + y * (3.0 + 6.0 * y));   /* 1 - (10y^3 - 15y^4 + 6y^5) */
    return (z * z) / (2.0 * y * y - 2.0 * y + 1.0);                    /* 1 - y^2/(2y^2 - 2y + 1)   */
}

/* y = (x[3n], v[3n]) -> f = (v, a).  rc holds nlev critical radii per member, level-major (rc[k*n + i]); the pair
 * term carries the product over the levels k = 0 .. nlev-1 of [1 - W(r; rc_k,ij)]: nlev = 1 is Eq. 4 as printed, nlev > 1
 * is the innermost Hamiltonian of the multi-level scheme (oracle_level_kick below). */
static void group_rhs(const double *y, double *f, int n, const double *gm, const double *rc, int nlev, double mu, int kind,
                      const int32_t *into /* NULL, or: members with into[i] != -1 were absorbed (reading S26): star term only */) {
    const double *x = y, *v = y + 3 * n;
    for (int i = 0; i < n; ++i) {
        double r2 = (x[3 * i] * x[3 * i] + x[3 * i + 1] * x[3 * i + 1]) + x[3 * i + 2] * x[3 * i + 2];
        double s = -mu / (r2 * sqrt(r2));
        double ax = s * x[3 * i], ay = s * x[3 * i + 1], az = s * x[3 * i + 2];
        for (int j = 0; j < n; ++j) {
            if (j == i || (into != NULL && into[i] != -1)) continue;
            double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1], dz = x[3 * j + 2] - x[3 * i + 2];
            double d2 = (dx * dx + dy * dy) + dz * dz;
            if (d2 == 0.0) continue;                       /* coincident: no direction, contributes nothing */
            double d = sqrt(d2);
            double w = 1.0;
            for (int k = 0; k < nlev && w != 0.0; ++k) {
                double rcij = rc[k * n + i] > rc[k * n + j] ? rc[k * n + i] : rc[k * n + j];
                w = w * one_minus_changeover(d, rcij, kind);
            }
            if (w == 0.0) continue;
            double t = gm[j] * w / (d2 * d);
            ax += t * dx; ay += t * dy; az += t * dz;
        }
        f[3 * i] = v[3 * i]; f[3 * i + 1] = v[3 * i + 1]; f[3 * i + 2] = v[3 * i + 2];
        f[3 * n + 3 * i] = ax; f[3 * n + 3 * i + 1] = ay; f[3 * n + 3 * i + 2] = az;
    }
}

/* The right-hand side above for one group, exported so that the tests can pin the [1 - W] pair term
 * directly (it must equal (1 - oracle_changeover) G m_j / r^2, and kick + encounter = Newton). */
void oracle_encounter_rhs(const double *y, int n, const double *gm, const double *rc, int nlev, double mu, int kind, double *f) {
    group_rhs(y, f, n, gm, rc, nlev, mu, kind, NULL);
}

#define BS_COLS 8

/* Collisions inside the direct solver ("N-body simulations often treat collisions as perfect mergers";
 * PAPER.md:168 radii inflated by a constant factor f; PAPER.md:98 the solver "propagates the involved bodies through the
 * close encounter phase" -- which is where bodies touch).  DESIGN.md reading S26: after every ACCEPTED Bulirsch-Stoer step
 * the members are tested pairwise for contact, r_ij < f (R_i + R_j) (strict, fp64 on r^2 = (dx^2 + dy^2) + dz^2, the test
 * of reading S21); members linked by a chain of contacts merge at once by the rule of S21 -- into the one with the
 * smallest index: m <- sum m_k, x <- sum m_k x_k / sum m_k, v <- sum m_k v_k / sum m_k (index order, unfused),
 * R <- cbrt(sum R_k^3).  The survivor goes on with the group (its critical radius is held, like every rc, through the
 * step); an absorbed member keeps m = 0, R = 0 (it exerts nothing and is never tested again), is put on the survivor and
 * from then on takes no part in the encounter: it exerts nothing and feels only the star (were it left to feel the pair
 * terms it would be a massless particle at zero distance from its survivor, with another critical radius: a singular
 * encounter); when the group's integration ends it is put on the body that holds it then (x, v equal), so that the perfect merging at the step boundary (oracle.merge / nb_merge) removes it when the arrays are
 * compacted.  into[k] = member that absorbed member k (-1: none).  Returns the number of members absorbed by this test. */
static int group_collide(double *y, int n, double *mm, double *gm, double *rad, double G, double f, int32_t *into) {
    double *x = y, *v = y + 3 * n;
    int *parent = (int *)malloc(sizeof(int) * (size_t)n);
    int nabs = 0, any = 0;
    for (int i = 0; i < n; ++i) parent[i] = i;
    for (int i = 0; i < n; ++i) {
        if (into[i] != -1 || (mm[i] == 0.0 && rad[i] == 0.0)) continue;
        for (int j = i + 1; j < n; ++j) {
            if (into[j] != -1 || (mm[j] == 0.0 && rad[j] == 0.0)) continue;
            double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1], dz = x[3 * j + 2] - x[3 * i + 2];
            double r2 = (dx * dx + dy * dy) + dz * dz;
            double sr = f * (rad[i] + rad[j]);
            if (r2 < sr * sr) {
                int a = i, b = j;
                while (parent[a] != a) a = parent[a];
                while (parent[b] != b) b = parent[b];
                if (a < b) parent[b] = a; else if (b < a) parent[a] = b;   /* the smaller index is the root */
                any = 1;
            }
        }
    }
    if (any) {
        for (int s0 = 0; s0 < n; ++s0) {
            if (parent[s0] != s0) continue;
            double mt = 0.0, mx[3] = {0, 0, 0}, mv[3] = {0, 0, 0}, vol = 0.0;
            int cnt = 0;
            for (int k = s0; k < n; ++k) {                      /* members of the cluster in index order */
                int r = k;
                while (parent[r] != r) r = parent[r];
                if (r != s0) continue;
                mt = mt + mm[k];
                for (int c = 0; c < 3; ++c) { mx[c] = mx[c] + mm[k] * x[3 * k + c]; mv[c] = mv[c] + mm[k] * v[3 * k + c]; }
                vol = vol + rad[k] * rad[k] * rad[k];
                ++cnt;
            }
            if (cnt < 2) continue;
            if (mt > 0.0)
                for (int c = 0; c < 3; ++c) { x[3 * s0 + c] = mx[c] / mt; v[3 * s0 + c] = mv[c] / mt; }
            mm[s0] = mt; gm[s0] = G * mt; rad[s0] = cbrt(vol);
            for (int k = s0 + 1; k < n; ++k) {
                int r = k;
                while (parent[r] != r) r = parent[r];
                if (r != s0) continue;
                mm[k] = 0.0; gm[k] = 0.0; rad[k] = 0.0; into[k] = s0; ++nabs;
                for (int c = 0; c < 3; ++c) { x[3 * k + c] = x[3 * s0 + c]; v[3 * k + c] = v[3 * s0 + c]; }
            }
        }
    }
    free(parent);
    return nabs;
}

static int64_t encounter_group_core(double *y, int n, double *gm, const double *rc, int nlev, double mu, int kind,
                                    double dt, double tol, double *mm, double *rad, double G, double frad, int32_t *into,
                                    int64_t *absorbed);

int64_t oracle_encounter_group(double *y, int n, const double *gm, const double *rc, int nlev, double mu, int kind,
                               double dt, double tol) {
    /* without radii: gm is only read */
    return encounter_group_core(y, n, (double *)gm, rc, nlev, mu, kind, dt, tol, NULL, NULL, 0.0, 0.0, NULL, NULL);
}

/* mm != NULL: collisions on (reading S26); mm, gm, rad [n] in/out, into [n] out */
static int64_t encounter_group_core(double *y, int n, double *gm, const double *rc, int nlev, double mu, int kind,
                                    double dt, double tol, double *mm, double *rad, double G, double frad, int32_t *into,
                                    int64_t *absorbed) {
    const int dim = 6 * n;
    double *buf = (double *)malloc(sizeof(double) * (size_t)dim * (5 + BS_COLS));
    double *f = buf, *ym = buf + dim, *yn = buf + 2 * dim, *tmp = buf + 3 * dim, *f0 = buf + 4 * dim;
    double *T = buf + 5 * dim;                             /* T[c*dim + k]: current row of the tableau */
    double t = 0.0, h = dt;
    int64_t steps = 0;
    const double tol2 = tol * tol;
    while (t != dt) {
        if (fabs(h) > fabs(dt - t)) h = dt - t;
        if (fabs(h) < 1e-14 * fabs(dt)) { free(buf); return -1; }
        group_rhs(y, f0, n, gm, rc, nlev, mu, kind, into);
        int accepted = 0, cols = 0;
        for (int c = 1; c <= BS_COLS && !accepted; ++c) {
            const int nsub = 2 * c;
            const double hs = h / nsub;
            for (int k = 0; k < dim; ++k) { ym[k] = y[k]; yn[k] = y[k] + hs * f0[k]; }
            for (int s = 2; s <= nsub; ++s) {
                group_rhs(yn, f, n, gm, rc, nlev, mu, kind, into);
                for (int k = 0; k < dim; ++k) { tmp[k] = ym[k] + 2.0 * hs * f[k]; ym[k] = yn[k]; yn[k] = tmp[k]; }
            }
            group_rhs(yn, f, n, gm, rc, nlev, mu, kind, into);
            /* new tableau row: tmp[] runs along the row, T[] holds the previous row */
            double err2 = 0.0;
            for (int k = 0; k < dim; ++k) {
                double cur = 0.5 * (ym[k] + yn[k] + hs * f[k]);     /* T_{c,0} */
                double last_diag = c >= 2 ? T[(c - 2) * dim + k] : 0.0;  /* T_{c-1,c-2} */
                for (int mcol = 1; mcol < c; ++mcol) {
                    double ratio = (double)nsub / (double)(2 * (c - mcol));
                    double old = T[(mcol - 1) * dim + k];               /* T_{c-1,mcol-1} */
                    T[(mcol - 1) * dim + k] = cur;                      /* becomes T_{c,mcol-1} */
                    cur = cur + (cur - old) / (ratio * ratio - 1.0);    /* T_{c,mcol} */
                }
                T[(c - 1) * dim + k] = cur;                             /* T_{c,c-1}: the diagonal */
                tmp[k] = cur - last_diag;
            }
            if (c >= 2) {
                for (int i = 0; i < n; ++i) {
                    const double *dx = tmp + 3 * i, *dv = tmp + 3 * n + 3 * i;
                    const double *xx = y + 3 * i, *vv = y + 3 * n + 3 * i;
                    double ex = (dx[0] * dx[0] + dx[1] * dx[1]) + dx[2] * dx[2];
                    double ev = (dv[0] * dv[0] + dv[1] * dv[1]) + dv[2] * dv[2];
                    /* scales: heliocentric distance^2; speed^2, not below the circular speed^2 mu/r */
                    double sx = (xx[0] * xx[0] + xx[1] * xx[1]) + xx[2] * xx[2];
                    double sv = (vv[0] * vv[0] + vv[1] * vv[1]) + vv[2] * vv[2];
                    double vc2 = mu / sqrt(sx);
                    if (sv < vc2) sv = vc2;
                    if (ex > err2 * sx) err2 = ex / sx;
                    if (ev > err2 * sv) err2 = ev / sv;
                }
                if (err2 <= tol2) { accepted = 1; cols = c; }
            }
        }
        if (accepted) {
            for (int k = 0; k < dim; ++k) y[k] = T[(cols - 1) * dim + k];
            t = (fabs(dt - (t + h)) <= 1e-15 * fabs(dt)) ? dt : t + h;
            steps++;
            if (mm != NULL) *absorbed += group_collide(y, n, mm, gm, rad, G, frad, into);
            if (cols <= 6) h *= 1.3; else if (cols == 8) h *= 0.55;
        } else {
            h *= 0.5;
        }
    }
    if (mm != NULL) {
        /* absorbed members end on the body that holds them now (a survivor may have been absorbed later itself) */
        for (int k = 0; k < n; ++k) {
            if (into[k] < 0) continue;
            int s0 = into[k];
            while (into[s0] >= 0) s0 = into[s0];
            for (int c = 0; c < 3; ++c) { y[3 * k + c] = y[3 * s0 + c]; y[3 * n + 3 * k + c] = y[3 * n + 3 * s0 + c]; }
        }
    }
    free(buf);
    return steps;
}


/* All listed groups of at most max_group members (members / gstart / ngroups as oracle_groups writes
 * them), one after the other; x, v of the members are advanced in place by dt under H_A with
 * encounters, every other body is left alone.  stats = {groups integrated, groups skipped because they
 * exceed max_group, groups whose step size underflowed (left unchanged), accepted steps in total}. */
void oracle_encounter(double *x, double *v, const double *m, const double *rcrit, int64_t nlev, int64_t N, double M_star,
                      double G, double dt, int kind, double tol, const int32_t *members, const int32_t *gstart,
                      int64_t ngroups, int64_t max_group, int64_t *stats) {
    /* rcrit: [nlev][N] critical radii, level-major (nlev = 1: the plain hybrid scheme) */
    stats[0] = stats[1] = stats[2] = stats[3] = 0;
    for (int64_t g = 0; g < ngroups; ++g) {
        const int n = gstart[g + 1] - gstart[g];
        if (n > max_group) { stats[1]++; continue; }
        double *y = (double *)malloc(sizeof(double) * (size_t)((7 + nlev) * n));
        double *gm = y + 6 * n, *rc = y + 7 * n;
        for (int k = 0; k < n; ++k) {
            const int32_t b = members[gstart[g] + k];
            for (int c = 0; c < 3; ++c) { y[3 * k + c] = x[3 * (int64_t)b + c]; y[3 * n + 3 * k + c] = v[3 * (int64_t)b + c]; }
            gm[k] = G * m[b];
            for (int64_t l = 0; l < nlev; ++l) rc[l * n + k] = rcrit[l * N + b];
        }
        const int64_t st = oracle_encounter_group(y, n, gm, rc, (int)nlev, G * M_star, kind, dt, tol);
        if (st < 0) { stats[2]++; free(y); continue; }
        for (int k = 0; k < n; ++k) {
            const int32_t b = members[gstart[g] + k];
            for (int c = 0; c < 3; ++c) { x[3 * (int64_t)b + c] = y[3 * k + c]; v[3 * (int64_t)b + c] = y[3 * n + 3 * k + c]; }
        }
        stats[0]++; stats[3] += st;
        free(y);
    }
}

/* oracle_encounter with collisions examined inside the solver (reading S26, group_collide above; fully active case):
 * m, radius [N] in/out, absorbed_by [N] in/out (body that holds an absorbed body at the end of the call, -1 for
 * everybody else; bodies marked by earlier calls stay out of the encounter, as absorbed members do: group_collide).  stats[4] = bodies absorbed. */
void oracle_encounter_collide(double *x, double *v, double *m, double *radius, const double *rcrit, int64_t nlev, int64_t N,
                              double M_star, double G, double dt, int kind, double tol, double f, const int32_t *members,
                              const int32_t *gstart, int64_t ngroups, int64_t max_group, int32_t *absorbed_by, int64_t *stats) {
    stats[0] = stats[1] = stats[2] = stats[3] = stats[4] = 0;
    for (int64_t g = 0; g < ngroups; ++g) {
        const int n = gstart[g + 1] - gstart[g];
        if (n > max_group) { stats[1]++; continue; }
        double *y = (double *)malloc(sizeof(double) * (size_t)((9 + nlev) * n));
        double *gm = y + 6 * n, *mm = y + 7 * n, *rad = y + 8 * n, *rc = y + 9 * n;
        int32_t *into = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
        for (int k = 0; k < n; ++k) {
            const int32_t b = members[gstart[g] + k];
            for (int c = 0; c < 3; ++c) { y[3 * k + c] = x[3 * (int64_t)b + c]; y[3 * n + 3 * k + c] = v[3 * (int64_t)b + c]; }
            mm[k] = m[b]; gm[k] = G * m[b]; rad[k] = radius[b]; into[k] = -1;
            if (absorbed_by[b] >= 0) {
                /* absorbed in an earlier call and not yet removed from the arrays: still takes no part; it follows its
                 * holder if that is a member of this group (-2: it is not) */
                into[k] = -2;
                for (int q = 0; q < n; ++q) if (members[gstart[g] + q] == absorbed_by[b]) into[k] = q;
            }
            for (int64_t l = 0; l < nlev; ++l) rc[l * n + k] = rcrit[l * N + b];
        }
        int64_t nabs = 0;
        const int64_t st = encounter_group_core(y, n, gm, rc, (int)nlev, G * M_star, kind, dt, tol, mm, rad, G, f, into, &nabs);
        if (st < 0) { stats[2]++; free(y); free(into); continue; }   /* step size underflow: the group is left unchanged */
        for (int k = 0; k < n; ++k) {
            const int32_t b = members[gstart[g] + k];
            for (int c = 0; c < 3; ++c) { x[3 * (int64_t)b + c] = y[3 * k + c]; v[3 * (int64_t)b + c] = y[3 * n + 3 * k + c]; }
            m[b] = mm[k]; radius[b] = rad[k];
            if (into[k] >= 0) {
                int s0 = into[k];
                while (into[s0] >= 0) s0 = into[s0];
                absorbed_by[b] = members[gstart[g] + s0];
            }
        }
        stats[0]++; stats[3] += st; stats[4] += nabs;
        free(y); free(into);
    }
}

/* Semi-active mode (the first n_active bodies exert force, the others only feel it; BASELINE.json:north_star,
 * DESIGN.md readings S13, S22).  A test particle pulls on nobody, so inside a group the active members (the
 * "core"; the first members of the group, since members ascend) move exactly as if the test particles were not
 * there, and the test particles are mutually independent.  A group that has test particles is therefore
 * split: the core is integrated alone, and every test particle s is integrated together with the core
 * (core + s, from the same initial state), of which only s is kept.  split_max_core < 0 (the definition): every
 * such group is split; split_max_core >= 0: only groups whose core has at most that many members are split, the
 * others are treated as one problem, as in oracle_encounter (an implementation may stop splitting at some core
 * size; the two treatments agree to the Bulirsch-Stoer tolerance, not bit for bit).
 * max_group bounds the core (split groups) or the group (unsplit ones).
 * stats = {groups integrated, groups skipped, sub-integrations whose step size underflowed (body/core left
 * unchanged), accepted steps in total}. */
void oracle_encounter_split(double *x, double *v, const double *m, const double *rcrit, int64_t N, int64_t n_active,
                            double M_star, double G, double dt, int kind, double tol, const int32_t *members,
                            const int32_t *gstart, int64_t ngroups, int64_t max_group, int64_t split_max_core,
                            int64_t *stats) {
    (void)N;
    stats[0] = stats[1] = stats[2] = stats[3] = 0;
    for (int64_t g = 0; g < ngroups; ++g) {
        const int g0 = gstart[g], n = gstart[g + 1] - g0;
        int nc = 0;
        while (nc < n && members[g0 + nc] < n_active) ++nc;
        const int split = (nc < n && (split_max_core < 0 || nc <= split_max_core));
        if ((split ? nc : n) > max_group) { stats[1]++; continue; }
        const int nn = split ? nc + 1 : n;                   /* size of the largest sub-problem */
        double *y = (double *)malloc(sizeof(double) * (size_t)(8 * nn));
        double *gm = y + 6 * nn, *rc = y + 7 * nn;
        double *x0 = (double *)malloc(sizeof(double) * (size_t)(6 * n)), *v0 = x0 + 3 * n;
        for (int k = 0; k < n; ++k)
            for (int c = 0; c < 3; ++c) { x0[3 * k + c] = x[3 * (int64_t)members[g0 + k] + c]; v0[3 * k + c] = v[3 * (int64_t)members[g0 + k] + c]; }
        const int nsub = split ? 1 + (n - nc) : 1;          /* sub-problem 0: the core (or the whole group) */
        for (int sub = 0; sub < nsub; ++sub) {
            const int nb = split ? (sub == 0 ? nc : nc + 1) : n;
            for (int k = 0; k < nb; ++k) {
                const int src = (split && k == nc) ? nc + sub - 1 : k;   /* the satellite of this sub-problem */
                const int32_t b = members[g0 + src];
                for (int c = 0; c < 3; ++c) { y[3 * k + c] = x0[3 * src + c]; y[3 * nb + 3 * k + c] = v0[3 * src + c]; }
                gm[k] = G * m[b]; rc[k] = rcrit[b];
            }
            const int64_t st = oracle_encounter_group(y, nb, gm, rc, 1, G * M_star, kind, dt, tol);
            if (st < 0) { stats[2]++; continue; }
            stats[3] += st;
            const int first = (split && sub > 0) ? nc : 0;   /* a satellite sub-problem keeps only the satellite */
            for (int k = first; k < nb; ++k) {
                const int src = (split && k == nc) ? nc + sub - 1 : k;
                const int32_t b = members[g0 + src];
                for (int c = 0; c < 3; ++c) { x[3 * (int64_t)b + c] = y[3 * k + c]; v[3 * (int64_t)b + c] = y[3 * nb + 3 * k + c]; }
            }
        }
        stats[0]++;
        free(y); free(x0);
    }
}


/* ---------------------------------------------------------------------------------------------
 * Multi-level changeover ("introducing higher-level changeover functions ... to not switch from the
 * symplectic integrator directly to the direct integrator but to introduce intermediate phases, where the symplectic
 * integrator reduces the time step level by level for the affected bodies.  Only the last level is then performed with
 * the inner direct integrator.  Every level needs again a smooth changeover function").  DESIGN.md reading S23: the
 * hybrid split of PAPER.md:84-86 (Eq. 4, 5) is applied again to H_A, level after level.  With W_k(r) = W(r; rc_k,ij) the
 * kick weight of level k (critical radii rc_k = Eq. 7 evaluated with the level's time step dt / 2^k) and
 *     Omega_l(r) = prod_{k=0..l} [1 - W_k(r)]        (what is left of a pair force after levels 0 .. l took their share)
 * the level-(l+1) kick Hamiltonian carries the pair force weighted by Omega_l W_{l+1} and the level-(l+1) "H_A" the
 * pair force weighted by Omega_{l+1}; at every r:  W_0 + Omega_0 W_1 + ... + Omega_{L-1} W_L + Omega_L = 1.
 *
 * oracle_level_kick: v_i += h * sum_{j : {i,j} in pairs} G m_j Omega_level(r_ij) W_{level+1}(r_ij) (x_j - x_i)/r_ij^3
 * for the listed pairs only (the pairs in a close encounter at this level; for every other pair Omega_level = 0 at the
 * moment the list was made).  rcl: [nlev][N] level-major, nlev >= level + 2.  The pair terms of a body are summed in the
 * order of the list, the sum is applied with one rounding (as in oracle_kick).  A massless body pulls on nobody.
 * --------------------------------------------------------------------------------------------- */
void oracle_level_kick(const double *x, double *v, const double *m, int64_t N, double G, int kind, const int32_t *pairs,
                       int64_t npairs, const double *rcl, int64_t level, double h) {
    double *acc = (double *)calloc((size_t)(3 * N > 0 ? 3 * N : 1), sizeof(double));
    for (int64_t p = 0; p < npairs; ++p) {
        const int64_t i = pairs[2 * p], j = pairs[2 * p + 1];
        const double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1], dz = x[3 * j + 2] - x[3 * i + 2];
        const double r2 = (dx * dx + dy * dy) + dz * dz;
        if (r2 == 0.0) continue;
        const double r = sqrt(r2);
        double w = 1.0;
        for (int64_t k = 0; k <= level && w != 0.0; ++k) {
            const double rck = rcl[k * N + i] > rcl[k * N + j] ? rcl[k * N + i] : rcl[k * N + j];
            w = w * one_minus_changeover(r, rck, kind);
        }
        if (w == 0.0) continue;
        const double rcn = rcl[(level + 1) * N + i] > rcl[(level + 1) * N + j] ? rcl[(level + 1) * N + i] : rcl[(level + 1) * N + j];
        w = w * oracle_changeover(r, rcn, kind);
        if (w == 0.0) continue;
        const double f = w / (r2 * r);
        const double fi = G * m[j] * f, fj = G * m[i] * f;
        acc[3 * i] += fi * dx; acc[3 * i + 1] += fi * dy; acc[3 * i + 2] += fi * dz;
        acc[3 * j] -= fj * dx; acc[3 * j + 1] -= fj * dy; acc[3 * j + 2] -= fj * dz;
    }
    for (int64_t k = 0; k < 3 * N; ++k) v[k] = v[k] + h * acc[k];
    free(acc);
}

/* ---------------------------------------------------------------------------------------------
 * Velocity-dependent extra forces by the implicit midpoint method (Eq. 8):
 *     v^{t+dt} = v^t + dt * a_f( r^t, (v^t + v^{t+dt}) / 2 )
 * "The implicit midpoint method needs some iterations to converge and is applied in between of the basic
 * symplectic operations."  The paper refers to its source [21] for the forces themselves; ONE
 * simple force stands in for them here (reading S24): drag against a gas disk on circular orbits,
 *     a_f(r, v) = - gamma |u|^p u,   u = v - v_gas(r),   v_gas = (1 - eta) sqrt(mu / R) e_phi,
 * R = sqrt(x^2 + y^2) the cylindrical radius, e_phi = (-y, x, 0)/R, p = 0 (linear) or 1 (quadratic).
 * Eq. 8 is solved per body by the fixed-point iteration w <- v + dt a_f(r, (v + w)/2), started at w = v, until
 * |w_new - w| <= tol * max(|w_new|, |v_gas|) or max_iter iterations.  v is replaced by w.
 * Returns the number of bodies that did not converge (their last iterate is kept); *iters_max = most iterations used.
 * --------------------------------------------------------------------------------------------- */
static void drag_accel(const double *x, const double *vm, double mu, double gamma, int power, double eta, double *a,
                       double *vgas_norm) {
    double R2 = x[0] * x[0] + x[1] * x[1];
    double vg[3] = {0.0, 0.0, 0.0};
    if (R2 > 0.0) {
        double R = sqrt(R2);
        double vc = (1.0 - eta) * sqrt(mu / R);
        vg[0] = -vc * x[1] / R; vg[1] = vc * x[0] / R;
        *vgas_norm = fabs(vc);
    } else {
        *vgas_norm = 0.0;
    }
    double u[3] = {vm[0] - vg[0], vm[1] - vg[1], vm[2] - vg[2]};
    double f = gamma;
    if (power == 1) f = gamma * sqrt((u[0] * u[0] + u[1] * u[1]) + u[2] * u[2]);
    for (int k = 0; k < 3; ++k) a[k] = -f * u[k];
}

int64_t oracle_midpoint_drag(const double *x, double *v, int64_t N, double mu, double dt, double gamma, int power,
                             double eta, double tol, int64_t max_iter, int64_t *iters_max) {
    int64_t nfail = 0, imax = 0;
    for (int64_t i = 0; i < N; ++i) {
        const double *xi = x + 3 * i;
        double v0[3] = {v[3 * i], v[3 * i + 1], v[3 * i + 2]};
        double w[3] = {v0[0], v0[1], v0[2]};
        int converged = 0;
        int64_t it = 0;
        for (it = 1; it <= max_iter; ++it) {
            double vm[3], a[3], vgn, wn[3];
            for (int k = 0; k < 3; ++k) vm[k] = 0.5 * (v0[k] + w[k]);
            drag_accel(xi, vm, mu, gamma, power, eta, a, &vgn);
            for (int k = 0; k < 3; ++k) wn[k] = v0[k] + dt * a[k];
            double d2 = 0.0, n2 = 0.0;
            for (int k = 0; k < 3; ++k) { d2 += (wn[k] - w[k]) * (wn[k] - w[k]); n2 += wn[k] * wn[k]; }
            double scale = sqrt(n2) > vgn ? sqrt(n2) : vgn;
            for (int k = 0; k < 3; ++k) w[k] = wn[k];
            if (sqrt(d2) <= tol * scale) { converged = 1; break; }
        }
        if (!converged) { nfail++; it = max_iter; }
        if (it > imax) imax = it;
        for (int k = 0; k < 3; ++k) v[3 * i + k] = w[k];
    }
    if (iters_max) *iters_max = imax;
    return nfail;
}

/* The step of oracle_step with the extra force applied "in between of the basic symplectic operations"
 * (PAPER.md:116), reading S24: D(dt/2) B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) D(dt/2) with D the implicit-midpoint
 * velocity update above.  Force evaluations, r_crit and their sharing between steps exactly as in oracle_step (the
 * evaluation at a step boundary sees the velocities before the closing half-kick and before D).
 * Returns Kepler non-convergences + midpoint non-convergences. */
int64_t oracle_step_drag(double *x, double *v, const double *m, double M_star, int64_t N, int64_t n_active, double dt,
                         double G, double n1, double n2, int kind, double *rcrit, double *acc, int64_t nsteps,
                         double gamma, int power, double eta, double tol, int64_t max_iter) {
    int64_t nfail = 0;
    int update_rc = !(n1 == 0.0 && n2 == 0.0);
    if (update_rc) oracle_rcrit(x, v, m, M_star, N, dt, G, n1, n2, rcrit);
    oracle_accel(x, m, rcrit, N, n_active, G, kind, NULL, 0, acc, NULL, NULL);
    for (int64_t st = 0; st < nsteps; ++st) {
        nfail += oracle_midpoint_drag(x, v, N, G * M_star, 0.5 * dt, gamma, power, eta, tol, max_iter, NULL);
        for (int64_t i = 0; i < 3 * N; ++i) v[i] = v[i] + (0.5 * dt) * acc[i];
        oracle_shift(x, v, m, M_star, N, 0.5 * dt);
        nfail += oracle_drift_kepler(x, v, M_star, N, dt, G, 0);
        oracle_shift(x, v, m, M_star, N, 0.5 * dt);
        if (update_rc) oracle_rcrit(x, v, m, M_star, N, dt, G, n1, n2, rcrit);
        oracle_accel(x, m, rcrit, N, n_active, G, kind, NULL, 0, acc, NULL, NULL);
        for (int64_t i = 0; i < 3 * N; ++i) v[i] = v[i] + (0.5 * dt) * acc[i];
        nfail += oracle_midpoint_drag(x, v, N, G * M_star, 0.5 * dt, gamma, power, eta, tol, max_iter, NULL);
    }
    return nfail;
}
