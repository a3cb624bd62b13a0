/*
 * nbkick.h -- C ABI of libnbkick.so: the data-parallel hot path of the hybrid symplectic
 * planet-formation integrator of Grimm & Stadel (arxiv 2604.09184; cited as PAPER.md:<line>),
 * hand-written CUDA for NVIDIA B200 (sm_100a).  One GPU, no sharding, no CPU fallback.
 *
 * State ("democratic coordinates"): heliocentric positions x[N,3], barycentric
 * velocities v[N,3], masses m[N] of the N non-star bodies; the star (mass M_star) sits at the
 * origin and is not in the arrays.  Everything is fp64, contiguous, row-major.  Pair indices
 * are int32.  Units are the caller's; G is set with nb_configure (default: Gaussian k^2 in
 * AU, day, solar mass).
 *
 * Pointers.  Every array argument of the nb_* calls below is a DEVICE pointer unless the
 * function name ends in _host (those take HOST pointers and copy in and out themselves).
 * Ownership: the caller owns every buffer, including the scratch workspace handed over with
 * nb_configure; the library allocates no device memory in the device-pointer calls.  (The
 * _host calls keep one private, lazily grown device arena, released by nb_release.)
 *
 * Asynchrony.  Device-pointer calls enqueue work on the configured CUDA stream and return
 * without synchronising; results are ordered on that stream.  _host calls and nb_status
 * synchronise the stream before they return.
 *
 * Errors.  Every int-returning call returns NB_OK (0) or a negative NB_E_* code for
 * conditions detectable on the host at call time; nb_last_error() then holds a message.
 * Conditions only the device can see (pair list overflow, Kepler non-convergence,
 * non-finite input, coincident bodies) are counted lazily and read with nb_status.
 *
 * Semi-active mode (BASELINE.json:north_star; not in the paper): with n_active = A < N the
 * first A bodies are fully interacting and the remaining N-A "feel but do not exert" force:
 * the j-sum runs over j < A only, and a pair is listed only if at least one member is active.
 */
#ifndef NBKICK_H
#define NBKICK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NB_OK 0
#define NB_E_NULL (-1)      /* a required pointer is NULL */
#define NB_E_BADN (-2)      /* N <= 0 or N > 2^31 - 1 */
#define NB_E_BADARG (-3)    /* non-finite dt, M_star <= 0, n_active > N, nsteps < 0, bad config value */
#define NB_E_WORKSPACE (-4) /* no workspace configured or it is smaller than nb_workspace_bytes(N) */
#define NB_E_CUDA (-5)      /* a CUDA runtime call failed (message in nb_last_error) */

/* Changeover shapes for the transition 0.1 r_crit < r < r_crit (PAPER.md:94 says only
 * "smooth changeover function ranging from 0 to 1"; reading S2). */
#define NB_CHANGEOVER_RATIONAL 0 /* y^2 / (2y^2 - 2y + 1), y = (r - 0.1 rc) / (0.9 rc) */
#define NB_CHANGEOVER_QUINTIC 1  /* 10y^3 - 15y^4 + 6y^5 */

/* The O(N^2) sum has two kernels that compute the same accelerations and the same pair list
 * (summation order, hence the last bits, differ):
 *   NB_FORCE_TILES      one-sided: every ordered interaction (i,j) is evaluated for body i;
 *                       any n_active, any N.
 *   NB_FORCE_SYMMETRIC  Newton's third law: every unordered pair is evaluated once and its r^-3
 *                       serves both bodies (two thirds of the fp64 instructions); fully active case
 *                       only -- with n_active < N the call falls back to NB_FORCE_TILES.
 *   NB_FORCE_AUTO       symmetric when fully active and N >= 4096, else tiles. */
/* Arithmetic of the O(N^2) sum (PAPER.md:160 contrasts FP32 and FP64 runs):
 *   NB_PRECISION_F64    everything in fp64 (default; the north_star's 1e-12 tolerance applies)
 *   NB_PRECISION_MIXED  pairs out of reach of every critical radius are evaluated in fp32; pairs within reach, the
 *                       changeover weight, the pair test and the pair list stay in fp64 and are identical to the fp64
 *                       kernel's.  Tolerance: DESIGN.md reading S25 (~1e-7 relative, typically).  Two kernels:
 *                       fully active, N >= 4096 (or NB_FORCE_SYMMETRIC): the Newton-III
 *                       kernel on double-single positions -- differences fl(fl(xjh - xih) + fl(xjl - xil)), r^2, r^-3,
 *                       products and the sums over one visit of a 32-body block all on the FP32 pipe, fp64 from there on;
 *                       otherwise (semi-active, NB_FORCE_TILES): the one-sided kernel with the same double-single
 *                       arithmetic, summed in fp32 per 128-body tile and in fp64 across tiles -- when it holds 2 or 4
 *                       i-bodies per thread; with one (small N: latency-bound launches, where fp32 does not pay) the
 *                       fp64 kernel runs, which meets the tolerance trivially.
 *                       Units: r^-3 and G m r^-3 of the far pairs must lie in the fp32 range (1e-38 .. 1e38): they do in
 *                       AU / day / solar mass (the defaults) and in any units of that kind; they do not in cgs (r^-3 ~
 *                       1e-42).  Pairs closer than 1e-15 length units always take the fp64 pass. */
#define NB_PRECISION_F64 0
#define NB_PRECISION_MIXED 1
#define NB_SORT_AUTO 0
#define NB_SORT_ON 1
#define NB_SORT_OFF 2
#define NB_FORCE_AUTO 0
#define NB_FORCE_TILES 1
#define NB_FORCE_SYMMETRIC 2

/* Process-wide settings.  nb_default_config fills the defaults named below. */
typedef struct nb_config {
    void *stream;            /* cudaStream_t the calls enqueue on; NULL = legacy default stream */
    void *workspace;         /* DEVICE scratch owned by the caller, 256-byte aligned */
    size_t workspace_bytes;  /* its size; must be >= nb_workspace_bytes(N) of every call */
    int64_t pair_capacity;   /* rows of the caller's pairs[cap,2] buffer (default 0) */
    int64_t n_active;        /* semi-active: number of force-exerting bodies; 0 = all N */
    double G;                /* gravitational constant (default 0.01720209895^2) */
    double n1;               /* Eq. 7 safety factor on R_Hill (default 3) */
    double n2;               /* Eq. 7 safety factor on dt*v   (default 0.4) */
    int changeover_kind;     /* NB_CHANGEOVER_* (default rational) */
    int i_per_thread;        /* tuning: i-bodies held in registers per thread, 0 = auto (1,2,4) */
    int j_splits;            /* tuning: number of j-chunks the force grid is split into, 0 = auto */
    int use_graph;           /* nb_step: replay one captured CUDA graph per step (default 1) */
    int reuse_acc;           /* nb_step: acc (and rcrit, pairs) already hold the evaluation at the current x,
                                as left by the previous nb_step/nb_kick(dt=0) call on this state: skip the
                                evaluation at t0, so a run stepped in chunks costs one evaluation per step
                                (default 0) */
    int time_force;          /* bracket every force-tile launch with CUDA events (nb_force_time); implies
                                no graph replay (default 0) */
    int force_kernel;        /* NB_FORCE_AUTO (default), NB_FORCE_TILES, NB_FORCE_SYMMETRIC (see below) */
    int sym_block;           /* tuning: super-block size S of the symmetric kernel (128, 256, 512, 1024, 2048), 0 = auto */
    int resolve_encounters;  /* nb_step: 1 = the members of the encounter groups of each step's pair list are
                                propagated through A(dt) by the direct solver (nb_encounter) instead of the Kepler
                                drift; needs pairs != NULL (default 0: pure Kepler drift) */
    double bs_tol;           /* relative tolerance of the direct solver's Bulirsch-Stoer steps (default 1e-12) */
    double radius_factor;    /* nb_merge: factor f by which the physical radii are inflated (default 1) */
    int sort_staging;        /* tuning (symmetric kernel): NB_SORT_ON stages the bodies sorted by azimuth, so that super-tiles whose
                                arcs cannot hold an encounter pair skip the test (results keep the caller's indexing);
                                NB_SORT_AUTO (default): on for N >= 32768; NB_SORT_OFF */
    int levels;              /* nb_step with resolve_encounters, nb_encounter_levels: number L of intermediate changeover
                                levels (0 .. 8, default 0 = the plain hybrid scheme).  Level l = 1 .. L runs
                                with the time step dt / 2^l and the critical radii of Eq. 7 for that time step; only what
                                is still in a close encounter at level L reaches the direct solver.  Needs workspace for
                                two adjacency slots per row of the pair list (nb_workspace_bytes accounts for it). */
    double drag_gamma;       /* nb_midpoint_drag, nb_step: coefficient of the extra force a_f = -gamma |u|^p u (
                                reading S24); 0 (default) = no extra force, nb_step is the plain step */
    double drag_eta;         /* u = v - (1 - eta) sqrt(G M_star / R) e_phi: gas on circular orbits, slower by the fraction eta */
    int drag_power;          /* p: 0 linear drag (default), 1 quadratic drag */
    int midpoint_iters;      /* Eq. 8 fixed-point iterations at most (default 50) */
    double midpoint_tol;     /* stop when the update is below tol * max(|v|, |v_gas|) (default 1e-14) */
    int precision;           /* NB_PRECISION_F64 (default) or NB_PRECISION_MIXED (see above) */
    int64_t slot_bytes_max;  /* tuning (symmetric kernel): cap of the partial-acceleration slots in the workspace; 0 (default) =
                                4 GiB.  A grid whose slots (24 N^2 / S bytes) would pass it is evaluated in bands of tile
                                columns, one launch and one fold into acc per band (same results to rounding order) */
    double *collide_radius;  /* nb_step with resolve_encounters: DEVICE double[N] in/out, physical radii; non-NULL switches on the
                                collisions inside the direct solver (nb_encounter_collide; reading S26),
                                inflated by radius_factor.  The step then CHANGES m (the caller's array, although nb_step
                                takes it as const) and the radii: an absorbed body stays in the arrays with m = 0, R = 0
                                on the body that holds it until nb_merge compacts them.  Fully active case; with levels > 0 the
                                innermost solver examines the collisions and the level kicks that follow use the merged masses.
                                Default NULL: off */
    int32_t *collide_absorbed_by; /* with collide_radius: DEVICE int32[N] in/out, -1 or the body that holds an absorbed body
                                (initialise with -1; required) */
} nb_config;

void nb_default_config(nb_config *cfg);
/* Copies *cfg; validates G > 0, n1,n2 >= 0 and finite, pair_capacity >= 0, n_active >= 0.
 * The configuration is ONE per process (calls are serialised by a mutex): two simulations in one process re-issue
 * nb_configure between their calls, and share the one cached CUDA graph of an interior step (it is re-captured
 * whenever the pointers, sizes or tuning of the call differ from the cached ones). */
int nb_configure(const nb_config *cfg);
/* Bytes of scratch the device-pointer calls need for N bodies under the current tuning (the force
 * kernels' partial sums dominate: 24 N x slots, never more than slot_bytes_max: beyond it the symmetric kernel's tile
 * grid is evaluated in bands).  The O(N) calls need only its head: nb_rcrit none,
 * nb_drift_kepler the first 512 bytes (status words), nb_shift 512 + 2 x roundup256(24 ceil(N/256)) bytes. */
size_t nb_workspace_bytes(int64_t N);

/*
 * a0 -- critical radius, Eq. 7:  rcrit_i = max(n1 R_Hill,i , n2 |dt| |v_i|),
 * R_Hill,i = a_i (m_i / (3 M_star))^(1/3), a_i from vis-viva 1/a = 2/r - v^2/(G M_star) with the
 * stored velocity (a_i = r_i if 1/a <= 0)  [DESIGN.md reading S5].
 * x,v: [N,3] in; m: [N] in; rcrit: [N] out.
 */
int nb_rcrit(const double *x, const double *v, const double *m, double M_star, int64_t N, double dt,
             double *rcrit);

/*
 * a1-a4 -- H_B kick (Eq. 5; "H_B describes the N^2 mutual gravitational
 * force terms"; BASELINE.json:north_star):
 *     acc_i = sum_{j != i, j < n_active} G m_j W(r_ij; rc_ij) (x_j - x_i) / r_ij^3 ,
 *     v_i  += dt * acc_i                                  (dt = 0: accelerations and pairs only)
 * W = kick weight = 1 for r >= rc_ij, 0 for r <= 0.1 rc_ij, changeover_kind between (readings
 * S1-S3); rc_ij = max(rcrit_i, rcrit_j) (S4).  From the same tiles: every unordered pair with
 * r_ij < rc_ij (strict, decided in fp64 on r^2 < rc^2) is appended once as (min,max) to pairs
 * (PAPER.md:94, 98, 106), in unspecified order.
 *   x [N,3] in; v [N,3] in/out; m [N] in; rcrit [N] in, or NULL => computed internally by a0 from
 *   (x, v, m, M_star, dt) with the configured n1, n2 into workspace scratch (M_star is used for
 *   nothing else: H_B has no star term); acc [N,3] out; pairs [pair_capacity,2] int32 out or NULL
 *   (=> detection skipped); npairs: device int64[1] out, total number of pairs found -- it keeps
 *   counting past pair_capacity, only the first pair_capacity rows are written (required iff
 *   pairs != NULL).
 */
int nb_kick(const double *x, double *v, const double *m, double M_star, int64_t N, double dt,
            const double *rcrit, double *acc, int32_t *pairs, int64_t *npairs);

/*
 * nb_kick for callers that cannot allocate device memory (code under CUDA stream capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same operation (Eq. 5, 94, 98 -- see nb_kick), the same kernels
 * and launch geometry, but the scratch comes from a static device array of NB_STATIC_SCRATCH_BYTES (8 MiB) inside the
 * library instead of the workspace of nb_configure, which this call neither needs nor touches.  Every GPU that loads
 * the library holds those 8 MiB until the process exits.  The call itself allocates nothing: no cudaMalloc, cudaFree,
 * event or stream creation -- kernel launches, one 512-byte cudaMemsetAsync and at most one 64-byte device-to-device
 * cudaMemcpyAsync on the configured stream.
 *   Limit: nb_workspace_bytes(N) (for the current configuration) must not exceed NB_STATIC_SCRATCH_BYTES -- N up to
 *   about 4700 with the default configuration (N = 4096: 6.0 MB); beyond that the call returns NB_E_WORKSPACE and
 *   nb_last_error() names both sizes.  Use nb_kick with a caller-owned workspace for larger N.
 *   Arguments as nb_kick (all DEVICE pointers), plus status8: device int64[8] out or NULL -- the device-side
 *   condition counters of THIS call (layout of nb_status; they live in the static array, so nb_status does not
 *   see them).
 *   Sharing: all calls, from every stream and thread, use the one array of the current device.  It keeps the last
 *   call's contents; the call clears what must start at zero (the counters) and overwrites the rest before reading
 *   it.  Calls that OVERLAP on the GPU (different streams, or a captured graph replayed concurrently with another
 *   call) race on it: order them.
 * nb_kick_static_setup resolves the array's device address for the CURRENT device (cudaGetSymbolAddress, once per
 * device); nb_kick_static does the same on its first call per device, so calling it is only needed by callers who
 * want that out of the way beforehand (before beginning a stream capture, say).
 */
#define NB_STATIC_SCRATCH_BYTES (8u << 20)
int nb_kick_static_setup(void);
int nb_kick_static(const double *x, double *v, const double *m, double M_star, int64_t N, double dt,
                   const double *rcrit, double *acc, int32_t *pairs, int64_t *npairs, int64_t *status8);

/*
 * a5 -- H_C (Eq. 6): x_i += dt * (sum_k m_k v_k) / M_star for every body.
 * The sum is a fixed-shape tree reduction (deterministic, run-to-run reproducible).
 */
int nb_shift(double *x, const double *v, const double *m, double M_star, int64_t N, double dt);

/*
 * a6 -- H_A without encounters ("a Keplerian orbit can be solved analytically";
 * PAPER.md:84 Eq. 4 first sum): every body follows the Kepler flow about
 * mu = G M_star for dt, advanced with Gauss' f and g functions (BASELINE.json:north_star).
 * Bound orbits: Newton on the differenced Kepler equation; otherwise universal variables
 * (reading S15).  A body whose solver does not converge is left unchanged and counted.
 * x, v: [N,3] in/out.
 */
int nb_drift_kepler(double *x, double *v, double M_star, int64_t N, double dt);

/*
 * Velocity-dependent extra forces by the implicit midpoint method (Eq. 8:
 *     v^{t+dt} = v^t + dt a_f(r^t, (v^t + v^{t+dt})/2) ,
 * "needs some iterations to converge and is applied in between of the basic symplectic operations").  The paper
 * defers the forces themselves to its source; ONE simple force stands in (reading S24): drag against a gas
 * disk on circular orbits, a_f = -drag_gamma |u|^p u, u = v - (1 - drag_eta) sqrt(G M_star / R) e_phi, R the
 * cylindrical radius, p = drag_power.  Per body: fixed-point iteration from v until the update is below
 * midpoint_tol max(|v|, |v_gas|), at most midpoint_iters times; bodies that did not converge keep their last iterate
 * and are counted in nb_status[6].  x [N,3] in; v [N,3] in/out.  Needs the first 512 bytes of the workspace.
 * With drag_gamma > 0 nb_step applies this update for dt/2 before the opening and after the closing half-kick of every
 * step: D(dt/2) B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) D(dt/2).
 */
int nb_midpoint_drag(const double *x, double *v, double M_star, int64_t N, double dt);

/*
 * a7 -- nsteps steps of B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) (Eq. 3; order: reading
 * S6) with the adjacent half-kicks of consecutive steps sharing one force evaluation: one O(N^2)
 * evaluation per step plus one at the start.  rcrit is recomputed by a0 from the current (x, v)
 * immediately before every force evaluation (S17) unless n1 == n2 == 0, in which case the
 * caller's rcrit is used unchanged.  On return acc, rcrit, pairs, npairs are those of the last
 * evaluation (at the final positions).  nsteps = 0: one evaluation, no motion.
 *   x, v [N,3] in/out; m [N] in; rcrit [N] in/out; acc [N,3] out; pairs/npairs as in nb_kick.
 */
int nb_step(double *x, double *v, const double *m, double M_star, int64_t N, double dt, double *rcrit,
            double *acc, int32_t *pairs, int64_t *npairs, int64_t nsteps);

/*
 * Independent close-encounter groups ("finding independent close encounter groups and
 * integrating them independently"): the connected components of the graph whose edges
 * are the rows of a pair list as written by nb_kick / nb_step.  Integer work, every output unique
 * (bit-reproducible):
 *   pairs   [pair_capacity,2] int32 in; npairs: device int64[1] in -- min(*npairs, pair_capacity) rows
 *           are read (order inside a row and duplicates do not matter; a row with an index outside
 *           [0,N) or i == j is skipped and counted in nb_status[2])
 *   label   [N] int32 out: smallest body index of the body's group (a body without pairs: itself)
 *   members [N] int32 out: the bodies of all groups with >= 2 members, group after group, groups
 *           ordered by label, members ascending inside a group; the tail is -1
 *   gstart  [N/2 + 2] int32 out: members[gstart[g] .. gstart[g+1]) is group g; entries past the last: -1
 *   gstat   device int64[4] out: groups (>= 2 members), member bodies, largest group, pair rows read
 * Needs the first 512 + 2 x roundup256(24 ceil(N/256)) + 5 x roundup256(4 N) + ~8 N/1024 + 768 bytes of
 * the workspace (always inside nb_workspace_bytes(N)).
 */
int nb_groups(const int32_t *pairs, const int64_t *npairs, int64_t N, int32_t *label, int32_t *members,
              int32_t *gstart, int64_t *gstat);

/*
 * H_A with close encounters (Eq. 4: Kepler terms plus the pair terms weighted by [1 - K];
 * PAPER.md:98 "a direct solver is needed which propagates the involved bodies through the close
 * encounter phase"; PAPER.md:106 groups are integrated independently).  The members of every listed
 * group (members / gstart / gstat as nb_groups writes them) are advanced by dt under
 *     dx_i/dt = v_i,
 *     dv_i/dt = -G M_star x_i/r_i^3 + sum_{j in group, j != i} G m_j [1 - W(r_ij; rc_ij)] (x_j - x_i)/r_ij^3
 * (W, rc_ij as in nb_kick, rcrit held fixed; weight on the force: reading S3) with a Bulirsch-Stoer
 * integrator of relative tolerance bs_tol (reading S19: the paper prescribes no method); every other body
 * is left alone.  Groups of more than NB_MAX_GROUP members are left alone as well and counted in
 * nb_status[4] (the regime for which the paper proposes multi-level changeovers); a group
 * whose step size underflows is left unchanged and counted in nb_status[5].
 * Semi-active mode (n_active < N; reading S22): a test particle pulls on nobody, so a group with at most 31 active
 * members is split -- its active core is integrated alone and every test particle together with the core, of
 * which only the particle is kept; NB_MAX_GROUP then bounds the core, not the group (an embryo may carry
 * thousands of test particles).  Groups with a larger core are treated as one problem.
 * x, v [N,3] in/out; m, rcrit [N] in.  Needs the same head of the workspace as nb_groups.
 */
#define NB_MAX_GROUP 1024
int nb_encounter(double *x, double *v, const double *m, const double *rcrit, double M_star, int64_t N,
                 double dt, const int32_t *members, const int32_t *gstart, const int64_t *gstat);

/*
 * nb_encounter with collisions examined INSIDE the direct solver (the solver "propagates the involved
 * bodies through the close encounter phase" -- which is where bodies touch; PAPER.md:130 perfect mergers
 * radii inflated by radius_factor; reading S26).  After every ACCEPTED Bulirsch-Stoer step of a group its
 * members are tested pairwise for contact, r_ij < f (R_i + R_j) (strict, fp64 on r^2, the test of nb_merge); members
 * linked by a chain of contacts merge at once by the rule of nb_merge -- into the one with the smallest index:
 * m <- sum m_k, x <- sum m_k x_k / sum m_k, v likewise (index order), R <- cbrt(sum R_k^3).  The survivor goes on
 * with the group (critical radii are held through the step); an absorbed body gets m = 0, R = 0, is never tested
 * again and takes no part in the encounter any more -- it exerts nothing and feels only the star (left to feel the
 * pair terms it would be a massless particle at zero distance from its survivor: a singular encounter) -- and ends the
 * call ON the body that holds it (same x, v), so that nb_merge at the step boundary removes it when it compacts the
 * arrays (or the caller does, from absorbed_by).
 *   x, v [N,3] in/out; m, radius [N] in/out; rcrit [N] in; members / gstart / gstat as nb_encounter;
 *   absorbed_by [N] int32 in/out: -1, or for an absorbed body the body that holds it.  Initialise with -1; a body
 *   marked by an earlier call (and not yet removed from the arrays) stays out of the encounter in the same way and
 *   follows its holder.  Entries of bodies that are not absorbed are not written.  Absorbed bodies are counted in nb_status[7].  Fully active case only
 *   (NB_E_BADARG with 0 < n_active < N).  A group whose step size underflows is left unchanged, merges included.
 */
int nb_encounter_collide(double *x, double *v, double *m, double *radius, const double *rcrit, double M_star, int64_t N,
                         double dt, const int32_t *members, const int32_t *gstart, const int64_t *gstat,
                         int32_t *absorbed_by);

/*
 * Multi-level changeover ("introducing higher-level changeover functions ... to not switch from the
 * symplectic integrator directly to the direct integrator but to introduce intermediate phases, where the symplectic
 * integrator reduces the time step level by level for the affected bodies.  Only the last level is then performed with
 * the inner direct integrator.  Every level needs again a smooth changeover function"; reading S23).
 * H_A over dt for the bodies of a pair list with L = levels intermediate levels: with rc_k,i = max(rc_hill_i,
 * rc_vel_i / 2^k) (the two terms of Eq. 7; the velocity term shrinks with the level's time step dt / 2^k),
 * W_k = W(r; max(rc_k,i, rc_k,j)) and Omega_l = prod_{k <= l} [1 - W_k],
 *     advance(l, tau):  l == L: the direct solver of nb_encounter over tau for the groups of P_L, pair weight Omega_L
 *                       else twice, h = tau/2:  P_{l+1} = pairs of P_l with r < rc_{l+1} now (strict, fp64 on r^2)
 *                                               v_i += (h/2) sum_{j: {i,j} in P_l} G m_j Omega_l W_{l+1} (x_j - x_i)/r^3
 *                                               bodies of P_l in no pair of P_{l+1}: Kepler drift h;  advance(l + 1, h)
 *                                               the same kick again
 * starting with advance(0, dt) on P_0 = the given list.  At every r the weights W_0 (nb_kick), Omega_{l-1} W_l (level
 * kicks) and Omega_L (direct solver) sum to 1.  Bodies in no listed pair are left alone; groups of P_L beyond
 * NB_MAX_GROUP take the Kepler drift over tau and are counted in nb_status[4] (once per visit).  Sums run over a body's
 * partners in ascending index order: bit-reproducible.  Fully active case only.
 *   x, v [N,3] in/out; m, rc_hill, rc_vel [N] in; pairs / npairs in (device, as in nb_groups).
 * Needs the head of the workspace up to and including the multi-level area (inside nb_workspace_bytes(N)).
 */
int nb_encounter_levels(double *x, double *v, const double *m, const double *rc_hill, const double *rc_vel, double M_star,
                        int64_t N, double dt, const int32_t *pairs, const int64_t *npairs);

/*
 * Perfect merging ("N-body simulations often treat collisions as perfect mergers";
 * PAPER.md:168 radii inflated by a constant factor f = radius_factor; reading S21).  For every
 * row (i, j) of the pair list (as nb_kick / nb_step wrote it for the CURRENT positions) the bodies collide
 * iff r_ij < f (R_i + R_j) (strict, fp64 on r^2).  Bodies linked by a chain of collisions merge into the one
 * with the smallest index: m <- sum m_k, x <- sum m_k x_k / sum m_k, v <- sum m_k v_k / sum m_k (members
 * in index order; mass and momentum conserved), R <- cbrt(sum R_k^3); if all masses are zero the survivor
 * keeps its x, v.  The other members are removed and x, v, m, radius are compacted in index order (stable:
 * a semi-active ordering survives); rows past the new N are undefined.
 *   x, v [N,3], m, radius [N] in/out; pairs / npairs in (device, as in nb_groups);
 *   survivor_of [N] int32 out: index (before compaction) of the body each body ended up in (itself if untouched);
 *   mstat device int64[4] out: new N, colliding pair rows, bodies removed, new n_active (alive among the
 *   first n_active; = new N when n_active is 0).
 * acc, rcrit and the pair list refer to the old indexing afterwards: re-evaluate (nb_kick / nb_step with
 * reuse_acc = 0) with the new N, and re-issue nb_configure if n_active changed.  Needs nb_workspace_bytes(N).
 */
int nb_merge(double *x, double *v, double *m, double *radius, int64_t N, const int32_t *pairs,
             const int64_t *npairs, int32_t *survivor_of, int64_t *mstat);

/*
 * Host-buffer forms of nb_kick and nb_step: same semantics, every pointer is a HOST pointer
 * (pairs has room for pair_capacity rows; npairs is a host int64).  Inputs are copied to the
 * library's private device arena, the device path above runs, outputs are copied back, the
 * stream is synchronised.  rcrit may be NULL in nb_kick_host (as in nb_kick) and in
 * nb_step_host (then it is neither read nor returned; needs n1 or n2 > 0).
 */
int nb_kick_host(const double *x, double *v, const double *m, double M_star, int64_t N, double dt,
                 const double *rcrit, double *acc, int32_t *pairs, int64_t *npairs);
int nb_step_host(double *x, double *v, const double *m, double M_star, int64_t N, double dt,
                 double *rcrit, double *acc, int32_t *pairs, int64_t *npairs, int64_t nsteps);

/*
 * Lazy device-side conditions accumulated since the last nb_status_reset; synchronises the
 * stream.  flags (host int64[8]):
 *   [0] pairs dropped because the list was full (sum over evaluations)
 *   [1] Kepler solver non-convergences (body left unchanged)
 *   [2] non-finite positions / masses / radii seen while staging j-bodies; invalid rows of a pair list
 *   [3] coincident bodies (r_ij == 0, i != j) that contributed nothing
 *   [4] encounter groups larger than NB_MAX_GROUP, left to the Kepler drift
 *   [5] encounter groups whose Bulirsch-Stoer step size underflowed (left unchanged)
 *   [6] bodies whose implicit-midpoint iteration (Eq. 8) did not converge
 *   [7] bodies absorbed by a collision inside the direct solver (nb_encounter_collide)
 */
int nb_status(int64_t *flags);
int nb_status_reset(void);

/* Milliseconds the most recent force-tile kernel of nb_kick / nb_step(nsteps=0) took, timed with
 * CUDA events on the configured stream (synchronises).  Negative if none was recorded. */
double nb_last_force_ms(void);
/* Sum over the force-tile launches recorded since the last nb_force_time_reset (time_force = 1):
 * *launches and *total_ms (CUDA events on the configured stream; synchronises).  At most 4096
 * launches are kept between resets; later ones are not recorded. */
int nb_force_time(int64_t *launches, double *total_ms);
int nb_force_time_reset(void);
/* Launch geometry the force kernel would use for (N, n_active): out[0] = i-bodies per thread,
 * out[1] = i-blocks, out[2] = j-splits, out[3] = threads per CTA, out[4] = j-tile length
 * (one-sided kernel) or minus the super-block size S (symmetric kernel; out[1] = out[2] = super-blocks). */
int nb_force_geometry(int64_t N, int64_t *out5);

/*
 * Measurement aid: runs a register-only chain of independent fp64 FMAs on every SM and returns
 * the achieved rate in *tflops (2 flops per FMA), the roofline denominator for the kick.
 * Synchronises.  iters = FMAs per chain step; 0 = default.
 * Unlike the calls of the path this one allocates: a small result buffer (cudaMalloc / cudaFree inside the call).
 */
int nb_fp64_peak(int64_t iters, double *tflops, double *ms);

/* Frees the private arena, cached graphs and events. */
void nb_release(void);

const char *nb_last_error(void);
const char *nb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NBKICK_H */
