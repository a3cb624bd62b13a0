// nbkick.cu -- host side of libnbkick.so: the C ABI declared in include/nbkick.h.
// Argument validation, workspace carving, launch geometry, the step driver (a7) with CUDA-graph
// replay, the host-buffer entry points and the measurement aids.  All arithmetic of the method runs
// in the kernels of force_tiles.cuh / body_kernels.cuh; nothing here computes on the CPU.
#include "../../include/nbkick.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "body_kernels.cuh"
#include "encounter.cuh"
#include "force_mixed.cuh"
#include "force_sym.cuh"
#include "force_symds.cuh"
#include "force_tiles.cuh"
#include "groups.cuh"
#include "merge.cuh"
#include "multilevel.cuh"
#include "step_small.cuh"

namespace {

using namespace nbk;

std::mutex g_mu;
nb_config g_cfg = {nullptr, nullptr, 0, 0, 0, 0.01720209895 * 0.01720209895, 3.0, 0.4, 0, 0, 0, 1, 0, 0, 0, 0, 0, 1e-12, 1.0, 0, 0, 0.0, 0.0, 0, 50, 1e-14, 0};
char g_err[512] = "";
int g_sm_count = 0;
cudaEvent_t g_ev0 = nullptr, g_ev1 = nullptr;
bool g_force_timed = false;
constexpr int kMaxTimed = 4096;
cudaEvent_t g_tev[2 * kMaxTimed];
int g_tev_created = 0, g_tev_used = 0;

// private arena of the _host entry points
void *g_arena = nullptr;
size_t g_arena_bytes = 0;

// cached CUDA graph of one interior step of nb_step
struct StepKey {
    const void *x, *v, *m, *rcrit, *acc, *pairs, *npairs, *ws, *stream, *radius, *absorbed_by;
    int64_t N, n_active, cap;
    double dt, M_star, G, n1, n2, bs_tol, drag_gamma, drag_eta, midpoint_tol;
    int kind, ipt, jsplit, enc, levels, drag_power, midpoint_iters, band;
    size_t ws_bytes;
};
StepKey g_graph_key;
cudaGraphExec_t g_graph_exec = nullptr;

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define NB_CUDA(call)                                                                                   \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) return fail(NB_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

inline size_t align_up(size_t a, size_t b) { return (a + b - 1) / b * b; }
// Graph capture needs a capturable stream; the legacy default stream (what torch hands out unless the
// caller made its own) is not.  Graph replay then runs on a private stream ordered against the
// caller's stream with events, so the calls stay stream-ordered as include/nbkick.h promises.
cudaStream_t g_own_stream = nullptr;
cudaEvent_t g_ev_in = nullptr, g_ev_out = nullptr;
bool g_on_own_stream = false;
inline cudaStream_t stream() { return g_on_own_stream ? g_own_stream : static_cast<cudaStream_t>(g_cfg.stream); }
inline bool stream_capturable() {
    const uintptr_t h = reinterpret_cast<uintptr_t>(g_cfg.stream);
    return h > 2;  // 0 = legacy default, 1 = cudaStreamLegacy, 2 = cudaStreamPerThread
}

int sm_count() {
    if (g_sm_count == 0) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            g_sm_count = n;
        else
            g_sm_count = 148;  // B200; only reached with no device (geometry queries on a CPU box)
    }
    return g_sm_count;
}

// Launch geometry of the force kernel.
struct Geometry {
    int ipt;              // i-bodies per thread
    int iblocks;          // CTAs along i
    int tiles_total;      // ceil(Nj / kTileJ)
    int tiles_per_split;  // j-tiles per CTA
    int nsplit;           // CTAs along j
    int Nj, Njpad;
    int minb;             // register cap: CTAs per SM the kernel variant is compiled for (3..6)
    int sym;              // 1: Newton-III super-tile kernel (force_sym.cuh); nsplit = number of super-blocks
    int S, U, Npad_sym;   // super-block size, 32-blocks per skew unit, N padded to a multiple of S
    int warps;            // symmetric kernel: warps per CTA (1, 2 or 4)
    int xcols;            // symmetric kernel: trailing tile columns cut into kSymSplit CTAs each (force_sym.cuh kSymSplit)
    int band;             // symmetric kernel: tile columns per launch of the banded evaluation (0: the whole grid in one launch)
    int nslots;           // partial-acceleration slots nb_kickv_kernel sums (= nsplit + extra slots of the split columns)
    int sorted;           // symmetric kernel: bodies staged in azimuthal order (sort_staging.cuh)
    int mixed;            // mixed-precision one-sided kernel (force_mixed.cuh)
};

constexpr int64_t kSymMinN = 4096;         // fully active N from which the Newton-III kernel is taken (measured crossover with the
                                           // fused one-sided step: 56 vs 53 us per step at N = 4096, 127 vs 95 at N = 8192)
constexpr int64_t kSmallStepMaxN = 8192;   // the fused small-N step (step_small.cuh) takes N up to this

Geometry geometry(int64_t N, int64_t n_active) {
    Geometry g;
    g.Nj = (int)((n_active > 0 && n_active < N) ? n_active : N);
    g.tiles_total = (g.Nj + kTileJ - 1) / kTileJ;
    g.Njpad = g.tiles_total * kTileJ;
    const int sms = sm_count();
    g.sym = 0; g.S = 0; g.U = 0; g.Npad_sym = 0; g.sorted = 0; g.warps = 4; g.xcols = 0; g.nslots = 0; g.band = 0;
    g.mixed = g_cfg.precision == NB_PRECISION_MIXED ? 1 : 0;
    // Newton-III kernel: fully active case only (a passive body exerts nothing, so there is no second
    // side to serve), and only when there are enough super-tiles to fill the machine several times.
    const bool fully_active = (g.Nj == N);
    if (fully_active && g.mixed && g_cfg.force_kernel != NB_FORCE_TILES && (g_cfg.force_kernel == NB_FORCE_SYMMETRIC || N >= kSymMinN)) {
        // Newton-III mixed-precision kernel (force_symds.cuh): I = 4, CTAs of 1 / 2 / 4 warps chosen as for the fp64 kernel;
        // sorted staging and the banded evaluation as for the fp64 kernel; no tail splitting
        auto waves = [&](int s) {
            const int64_t T = (N + s - 1) / s;
            return (double)(T * (T + 1) / 2) / (double)((int64_t)sms * (1536 / s));
        };
        int S = g_cfg.sym_block;
        if (S != 128 && S != 256 && S != 512) S = waves(512) >= 16.0 ? 512 : (waves(256) >= 5.0 ? 256 : 128);
        const int64_t Npad = ((N + S - 1) / S) * S, T = Npad / S;
        const int64_t cap = g_cfg.slot_bytes_max > 0 ? g_cfg.slot_bytes_max : ((int64_t)4 << 30);
        g.sym = 1; g.mixed = 2; g.S = S; g.U = S / 128; g.ipt = 4; g.warps = S / 128; g.minb = 12 / g.warps;
        g.Npad_sym = (int)Npad; g.nsplit = (int)T; g.iblocks = (int)T; g.tiles_per_split = 0; g.nslots = (int)T;
        g.sorted = g_cfg.sort_staging == NB_SORT_ON || (g_cfg.sort_staging == NB_SORT_AUTO && N >= 32768);
        if (T * N * 24 > cap) {   // banded evaluation, as for the fp64 kernel (5.1d)
            int64_t band = cap / (24 * (N + Npad));
            if (band < 1) band = 1;
            if (band < T) g.band = (int)band;
        }
        return g;
    }
    if (fully_active && !g.mixed && g_cfg.force_kernel != NB_FORCE_TILES && (g_cfg.force_kernel == NB_FORCE_SYMMETRIC || N >= kSymMinN)) {
        // I = 4 at 12 warps per SM (160 registers, no spills) measured fastest on B200.
        // The CTA shrinks with the super-block -- 4 warps for S >= 512, 2 for S = 256, 1 for S = 128 -- so that a
        // mid-sized problem still has many short CTAs: the tail of the grid costs about one CTA duration, whatever
        // the number of CTAs left (a lone CTA runs hardly faster than one of twelve warps' worth).
        int ipt = g_cfg.i_per_thread;
        if (ipt != 1 && ipt != 2 && ipt != 4) ipt = 4;
        int S = g_cfg.sym_block;
        if (S != 128 && S != 256 && S != 512 && S != 1024 && S != 2048) {
            // largest block whose grid still has enough waves of CTAs (measured crossovers: N ~ 24000 and ~ 60000).  The
            // N/S partial slots (24 N^2 / S bytes) are bounded by the banded evaluation below, not by a larger S
            auto waves = [&](int s) {
                const int64_t T = (N + s - 1) / s;
                return (double)(T * (T + 1) / 2) / (double)((int64_t)sms * (1536 / s));
            };
            S = ipt == 4 ? (waves(512) >= 16.0 ? 512 : (waves(256) >= 5.0 ? 256 : 128)) : (waves(512) >= 16.0 ? 512 : 256);
        }
        if (ipt == 1 && S < 128) S = 128;
        // warps per CTA: chunks of 32 W I bodies must tile the super-block
        int W = S / (32 * ipt);
        if (W > 4) W = 4;
        if (ipt == 1) W = 4;
        if (ipt == 2 && W == 1) W = 2;
        if (S < 32 * ipt * W) S = 32 * ipt * W;
        const int minb = ipt == 4 ? 12 / W : (W == 4 ? 4 : 8);
        g.sym = 1; g.S = S; g.U = S / 128; g.ipt = ipt; g.minb = minb; g.warps = W;
        g.Npad_sym = (int)(((N + S - 1) / S) * S);
        g.nsplit = g.Npad_sym / S;
        g.iblocks = g.nsplit; g.tiles_per_split = 0;
        {   // tail splitting: about one wave's worth of tiles (the ones launched last) run as kSymSplit short CTAs each;
            // pointless once the grid is hundreds of waves long
            const int64_t T = g.nsplit, slots = (int64_t)sms * (12 / W);
            const int jS = S / kSymSplit, Uq = g.U / kSymSplit > 0 ? g.U / kSymSplit : 1;
            int C = 0;
            if (ipt == 4 && jS >= 32 && jS / (32 * Uq) >= W && T * (T + 1) / 2 < 100 * slots) {
                C = (int)((slots + T - 1) / T);
                if (C > T / 4) C = (int)(T / 4);
                if (C > 16) C = 16;
            }
            g.xcols = C;
        }
        g.nslots = sym_slots(g.nsplit, g.xcols);
        {   // banded evaluation: when the slots of the whole grid would pass the cap (nb_config.slot_bytes_max, default
            // 4 GiB), the tile columns run in bands of `band` columns, one launch + one fold per band, on
            // 24 N band (i sides) + 24 Npad band (j sides of the band's bodies) bytes
            const int64_t cap = g_cfg.slot_bytes_max > 0 ? g_cfg.slot_bytes_max : ((int64_t)4 << 30);
            if ((int64_t)g.nslots * N * 24 > cap) {
                int64_t band = cap / (24 * (N + (int64_t)g.Npad_sym));
                if (band < 1) band = 1;
                if (band < g.nsplit) { g.band = (int)band; g.xcols = 0; g.nslots = g.nsplit; }
            }
        }
        // sorted staging pays off once the sort (a few small launches) is small against the evaluation
        g.sorted = g_cfg.sort_staging == NB_SORT_ON || (g_cfg.sort_staging == NB_SORT_AUTO && N >= 32768);
        return g;
    }
    // I: register tile (i-bodies per thread).  I = 2 at 5 CTAs/SM (96 registers, 20 warps/SM) measured
    // fastest on B200 (profiles/); small N falls back to I = 1 so that enough (i-block, j-tile) work
    // items exist to cover every SM a few times.  I = 4 stays selectable (fewer shared-memory reads).
    int ipt = g_cfg.i_per_thread;
    if (ipt != 1 && ipt != 2 && ipt != 4) {
        ipt = 2;
        while (ipt > 1 &&
               ((N + (int64_t)kForceThreads * ipt - 1) / ((int64_t)kForceThreads * ipt)) * g.tiles_total < (int64_t)4 * sms)
            ipt >>= 1;
    }
    g.ipt = ipt;
    g.minb = ipt == 4 ? 3 : 5;
    // mixed precision with one i-body per thread (small N: latency-bound launches) does not pay: the fp64 kernel runs
    // instead (it meets the mixed tolerance trivially, and the fused small-N step stays available)
    if (g.mixed && ipt == 1) g.mixed = 0;

    g.iblocks = (int)((N + (int64_t)kForceThreads * ipt - 1) / ((int64_t)kForceThreads * ipt));
    int nsplit = g_cfg.j_splits;
    if (nsplit <= 0) {
        // Among split counts that give roughly 6..16 waves of (minb CTAs per SM), take the one whose last
        // wave is fullest; keep a few tiles per CTA so the prologue/epilogue and the partial-sum traffic
        // stay negligible.
        const int64_t slots = (int64_t)g.minb * sms;
        const int min_tiles = g.tiles_total <= 32 ? 1 : (g.tiles_total <= 256 ? 2 : 4);
        const int max_split = (g.tiles_total + min_tiles - 1) / min_tiles;
        int lo = (int)((6 * slots + g.iblocks - 1) / g.iblocks), hi = (int)((16 * slots + g.iblocks - 1) / g.iblocks);
        if (lo < 1) lo = 1;
        if (hi > max_split) hi = max_split;
        if (lo > hi) lo = hi;
        double best = -1.0;
        nsplit = lo;
        for (int ns = lo; ns <= hi; ++ns) {
            const int tps = (g.tiles_total + ns - 1) / ns;
            const int eff_ns = (g.tiles_total + tps - 1) / tps;       // splits that actually get tiles
            const int64_t ctas = (int64_t)g.iblocks * eff_ns;
            const int64_t waves = (ctas + slots - 1) / slots;
            // useful tile-work over the work the waves could have done at tps tiles per CTA
            const double eff = (double)g.iblocks * g.tiles_total / ((double)waves * slots * tps);
            if (eff > best + 1e-9) { best = eff; nsplit = ns; }
        }
    }
    if (nsplit > g.tiles_total) nsplit = g.tiles_total;
    if (nsplit > 65535) nsplit = 65535;
    g.tiles_per_split = (g.tiles_total + nsplit - 1) / nsplit;
    g.nsplit = (g.tiles_total + g.tiles_per_split - 1) / g.tiles_per_split;
    g.nslots = g.nsplit;
    return g;
}

// Workspace carving (all offsets 256-byte aligned).
struct Workspace {
    long long *status;  // ST_COUNT
    unsigned long long *npairs_dummy;
    double *mvA, *mvB;  // momentum partials [nblk,3]
    GroupScratch grp;   // encounter groups (groups.cuh): 5 N + 2 ceil(N/1024) + N/2048 + 3 ints
    int32_t *g_label, *g_members, *g_start;  // the step driver's own group lists
    int64_t *g_stat;
    int *g_core, *enc_flag;                  // direct-solver plan: active members per group, per-body flag
    MlScratch ml;                            // multi-level changeover (multilevel.cuh), sized by pair_capacity; levels > 0 only
    double *ml_hill, *ml_vel;                // [N] the two terms of Eq. 7 of the evaluation that opened the step
    int *ml_listed;                          // [N] body is in a pair of the step's list
    char *head_mv_end, *head_grp_end, *head_ml_end;  // ends of the geometry-independent head
    double *rc_scratch; // [N]
    JRec *jrec;         // [Njpad]                 (one-sided kernel)
    double2 *sxy, *szg; // [2 Npad_sym]            (symmetric kernel, doubled-block layout)
    int *sthr;          // [2 Npad_sym]
    float4 *sa, *sb;    // [2 Npad_sym]            (Newton-III mixed-precision kernel: double-single records)
    JRecDs *jds;        // [Njpad]                 (one-sided mixed-precision kernel, I >= 2: double-single records)
    int *perm, *pos_of; // [Npad_sym], [N]         (sorted staging: position <-> body)
    BlockBound *bnd;    // [nsplit]                (bounds of the staged super-blocks)
    double *part;       // [nsplit, N, 3]
    size_t bytes;
};

Workspace carve(void *base, int64_t N, const Geometry &g) {
    Workspace w;
    size_t off = 0;
    char *b = static_cast<char *>(base);
    const size_t nblk = (size_t)((N + kBodyThreads - 1) / kBodyThreads);
    w.status = reinterpret_cast<long long *>(b + off); off += 256;
    w.npairs_dummy = reinterpret_cast<unsigned long long *>(b + off); off += 256;
    w.mvA = reinterpret_cast<double *>(b + off); off += align_up(nblk * 3 * sizeof(double), 256);
    w.mvB = reinterpret_cast<double *>(b + off); off += align_up(nblk * 3 * sizeof(double), 256);
    w.head_mv_end = b + off;
    {
        const size_t n4 = align_up((size_t)N * sizeof(int), 256);
        const size_t gblk = (size_t)((N + kGrpScanBlock - 1) / kGrpScanBlock);
        w.grp.parent = reinterpret_cast<int *>(b + off); off += n4;
        w.grp.size = reinterpret_cast<int *>(b + off); off += n4;
        w.grp.segstart = reinterpret_cast<int *>(b + off); off += n4;
        w.grp.cursor = reinterpret_cast<int *>(b + off); off += n4;
        w.grp.tmp = reinterpret_cast<int *>(b + off); off += n4;
        w.grp.bsum = reinterpret_cast<int *>(b + off); off += align_up(2 * gblk * sizeof(int), 256);
        w.grp.giant = reinterpret_cast<int *>(b + off); off += align_up(((size_t)N / kGiant + 2) * sizeof(int), 256);
        w.grp.ngiant = reinterpret_cast<int *>(b + off); off += 256;
    }
    {   // group outputs of the step driver (resolve_encounters): label, members, gstart, gstat
        const size_t n4 = align_up((size_t)N * sizeof(int), 256);
        w.g_label = reinterpret_cast<int32_t *>(b + off); off += n4;
        w.g_members = reinterpret_cast<int32_t *>(b + off); off += n4;
        w.g_start = reinterpret_cast<int32_t *>(b + off); off += align_up(((size_t)N / 2 + 2) * sizeof(int), 256);
        w.g_stat = reinterpret_cast<int64_t *>(b + off); off += 256;
        w.g_core = reinterpret_cast<int *>(b + off); off += align_up(((size_t)N / 2 + 2) * sizeof(int), 256);
        w.enc_flag = reinterpret_cast<int *>(b + off); off += n4;
    }
    w.head_grp_end = b + off;
    {   // multi-level changeover: adjacency of the pair list (two slots per row) and the level radii
        const bool on = g_cfg.levels > 0;
        const size_t n4 = on ? align_up((size_t)(N + 1) * sizeof(int), 256) : 0;
        const size_t n8 = on ? align_up((size_t)N * sizeof(double), 256) : 0;
        const size_t slots = on ? (size_t)2 * (size_t)(g_cfg.pair_capacity > 0 ? g_cfg.pair_capacity : 0) : 0;
        const size_t s4 = align_up(slots * sizeof(int), 256);
        w.ml.deg = reinterpret_cast<int *>(b + off); off += n4;
        w.ml.off = reinterpret_cast<int *>(b + off); off += n4;
        w.ml.cur = reinterpret_cast<int *>(b + off); off += n4;
        w.ml.bdepth = reinterpret_cast<int *>(b + off); off += n4;
        w.ml_listed = reinterpret_cast<int *>(b + off); off += n4;
        w.ml.bsum = reinterpret_cast<int *>(b + off); off += on ? align_up(((size_t)N / kGrpScanBlock + 2) * sizeof(int), 256) : 0;
        w.ml_hill = reinterpret_cast<double *>(b + off); off += n8;
        w.ml_vel = reinterpret_cast<double *>(b + off); off += n8;
        w.ml.adj_tmp = reinterpret_cast<int *>(b + off); off += on ? s4 : 0;
        w.ml.own = reinterpret_cast<int *>(b + off); off += on ? s4 : 0;
        w.ml.adj = reinterpret_cast<int *>(b + off); off += on ? s4 : 0;
        w.ml.depth = reinterpret_cast<signed char *>(b + off); off += on ? align_up(slots, 256) : 0;
        w.ml.cap = g_cfg.pair_capacity;
    }
    w.head_ml_end = b + off;
    w.rc_scratch = reinterpret_cast<double *>(b + off); off += align_up((size_t)N * sizeof(double), 256);
    w.jrec = reinterpret_cast<JRec *>(b + off); off += align_up((size_t)(g.sym ? 0 : g.Njpad) * sizeof(JRec), 256);
    w.sxy = reinterpret_cast<double2 *>(b + off); off += align_up((size_t)2 * g.Npad_sym * sizeof(double2), 256);
    w.szg = reinterpret_cast<double2 *>(b + off); off += align_up((size_t)2 * g.Npad_sym * sizeof(double2), 256);
    w.sthr = reinterpret_cast<int *>(b + off); off += align_up((size_t)2 * g.Npad_sym * sizeof(int), 256);
    w.jds = reinterpret_cast<JRecDs *>(b + off); off += align_up((size_t)((!g.sym && g.mixed == 1) ? g.Njpad : 0) * sizeof(JRecDs), 256);
    w.sa = reinterpret_cast<float4 *>(b + off); off += align_up((size_t)(g.mixed == 2 ? 2 * g.Npad_sym : 0) * sizeof(float4), 256);
    w.sb = reinterpret_cast<float4 *>(b + off); off += align_up((size_t)(g.mixed == 2 ? 2 * g.Npad_sym : 0) * sizeof(float4), 256);
    w.perm = reinterpret_cast<int *>(b + off); off += align_up((size_t)g.Npad_sym * sizeof(int), 256);
    w.pos_of = reinterpret_cast<int *>(b + off); off += align_up((size_t)(g.sym ? N : 0) * sizeof(int), 256);
    w.bnd = reinterpret_cast<BlockBound *>(b + off); off += align_up((size_t)(g.sym ? g.nsplit : 0) * sizeof(BlockBound), 256);
    {   // partial accelerations; never smaller than 64 bytes per body (nb_merge's compaction buffer)
        size_t pb = g.band > 0 ? (size_t)g.band * ((size_t)N + (size_t)g.Npad_sym) * 3 * sizeof(double)
                               : (size_t)g.nslots * (size_t)N * 3 * sizeof(double);
        if (pb < (size_t)N * 64) pb = (size_t)N * 64;
        w.part = reinterpret_cast<double *>(b + off); off += align_up(pb, 256);
    }
    w.bytes = off;
    return w;
}

int check_common(int64_t N, double dt, double M_star) {
    if (N <= 0 || N > 2147483647LL) return fail(NB_E_BADN, "N = %lld out of range (1 .. 2^31-1)", (long long)N);
    if (!std::isfinite(dt)) return fail(NB_E_BADARG, "dt is not finite");
    if (!(M_star > 0.0) || !std::isfinite(M_star)) return fail(NB_E_BADARG, "M_star must be finite and > 0");
    if (g_cfg.n_active > N) return fail(NB_E_BADARG, "n_active = %lld > N = %lld", (long long)g_cfg.n_active, (long long)N);
    return NB_OK;
}

int check_workspace(int64_t N, const Geometry &g, Workspace *w) {
    if (g_cfg.workspace == nullptr) return fail(NB_E_WORKSPACE, "no workspace configured (nb_configure)");
    if ((reinterpret_cast<uintptr_t>(g_cfg.workspace) & 255u) != 0) return fail(NB_E_WORKSPACE, "workspace is not 256-byte aligned");
    *w = carve(g_cfg.workspace, N, g);
    if (w->bytes > g_cfg.workspace_bytes)
        return fail(NB_E_WORKSPACE, "workspace has %zu bytes, N = %lld needs %zu", g_cfg.workspace_bytes, (long long)N, w->bytes);
    return NB_OK;
}

// The O(N) calls touch only the head of the workspace (status words, momentum partials): they must not
// demand the O(N^2 / S) partial-sum area of the force kernels.
int check_workspace_head(int64_t N, int level /* 0 status, 1 + momentum partials, 2 + group scratch, 3 + multi-level area */, Workspace *w) {
    if (g_cfg.workspace == nullptr) return fail(NB_E_WORKSPACE, "no workspace configured (nb_configure)");
    if ((reinterpret_cast<uintptr_t>(g_cfg.workspace) & 255u) != 0) return fail(NB_E_WORKSPACE, "workspace is not 256-byte aligned");
    Geometry g0;
    std::memset(&g0, 0, sizeof(g0));
    *w = carve(g_cfg.workspace, N, g0);
    const char *base = static_cast<char *>(g_cfg.workspace);
    const size_t need = level == 0 ? 512 : (size_t)((level == 1 ? w->head_mv_end : (level == 2 ? w->head_grp_end : w->head_ml_end)) - base);
    if (need > g_cfg.workspace_bytes)
        return fail(NB_E_WORKSPACE, "workspace has %zu bytes, this call needs %zu", g_cfg.workspace_bytes, need);
    return NB_OK;
}

inline int body_blocks(int64_t n) { return (int)((n + kBodyThreads - 1) / kBodyThreads); }

// register caps measured fastest on B200 (profiles/): one-sided kernel I = 1, 2 at 5 CTAs/SM, I = 4 at 3;
// Newton-III kernel I = 1, 2 at 4 CTAs/SM, I = 4 at 3
template <int I, int MINB>
void launch_force_IM(const ForceParams &fp, const Geometry &g, bool pairs) {
    dim3 grid(g.iblocks, g.nsplit);
    // fewer than two waves of CTAs: the launch is latency-bound, the branch-free tile loop wins (force_tiles.cuh)
    // (always for the sizes the fused small-N step takes, which runs the branch-free loop: the two paths stay bit-identical)
    const bool bf = fp.N <= kSmallStepMaxN || (int64_t)g.iblocks * g.nsplit < (int64_t)2 * MINB * sm_count();
    if (pairs) {
        if (bf) nb_force_tiles_kernel<I, true, MINB, true><<<grid, kForceThreads, 0, stream()>>>(fp);
        else nb_force_tiles_kernel<I, true, MINB, false><<<grid, kForceThreads, 0, stream()>>>(fp);
    } else {
        if (bf) nb_force_tiles_kernel<I, false, MINB, true><<<grid, kForceThreads, 0, stream()>>>(fp);
        else nb_force_tiles_kernel<I, false, MINB, false><<<grid, kForceThreads, 0, stream()>>>(fp);
    }
}

template <int I, int MINB>
void launch_mixed_IM(const ForceParams &fp, const Geometry &g, bool pairs) {
    dim3 grid(g.iblocks, g.nsplit);
    // double-single records, everything on the FP32 pipe (force_mixed.cuh)
    if (pairs) nb_force_mixedds_kernel<I, true, MINB><<<grid, kForceThreads, 0, stream()>>>(fp);
    else nb_force_mixedds_kernel<I, false, MINB><<<grid, kForceThreads, 0, stream()>>>(fp);
}

void launch_force(const ForceParams &fp, const Geometry &g, bool pairs) {
    if (g.mixed) {
        if (g.ipt == 4) launch_mixed_IM<4, 4>(fp, g, pairs);
        else launch_mixed_IM<2, 5>(fp, g, pairs);   // (geometry() leaves I = 1 to the fp64 kernel)
        return;
    }
    if (g.ipt == 4) launch_force_IM<4, 3>(fp, g, pairs);
    else if (g.ipt == 2) launch_force_IM<2, 5>(fp, g, pairs);
    else launch_force_IM<1, 5>(fp, g, pairs);
}

template <int I, int W, int MINB, bool SORTED>
int launch_sym_IMS(const SymParams &sp, const Geometry &g, bool pairs) {
    const size_t smem = sym_smem_bytes(g.S);
    const long long T = g.nsplit;
    const unsigned ctas = (unsigned)(sp.ncols == (int)T ? sym_grid(T, g.xcols) : sym_band_grid(sp.col0, sp.ncols));
    auto go = [&](auto kern) -> int {
        NB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<ctas, 32 * W, smem, stream()>>>(sp);
        return NB_OK;
    };
    return pairs ? go(nb_force_sym_kernel<I, W, true, MINB, SORTED>) : go(nb_force_sym_kernel<I, W, false, MINB, SORTED>);
}

template <int I, int W, int MINB>
int launch_sym_IM(const SymParams &sp, const Geometry &g, bool pairs) {
    return g.sorted ? launch_sym_IMS<I, W, MINB, true>(sp, g, pairs) : launch_sym_IMS<I, W, MINB, false>(sp, g, pairs);
}

template <int W>
int launch_symds_W(const SymDsParams &dp, const Geometry &g, bool pairs) {
    const long long T = g.nsplit;
    const unsigned ctas = (unsigned)(dp.sp.ncols == (int)T ? T * (T + 1) / 2 : sym_band_grid(dp.sp.col0, dp.sp.ncols));
    const size_t smem = symds_smem_bytes(g.S);
    auto go = [&](auto kern) -> int {
        NB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<ctas, 32 * W, smem, stream()>>>(dp);
        return NB_OK;
    };
    if (g.sorted) return pairs ? go(nb_force_symds_kernel<W, true, true>) : go(nb_force_symds_kernel<W, false, true>);
    return pairs ? go(nb_force_symds_kernel<W, true, false>) : go(nb_force_symds_kernel<W, false, false>);
}

int launch_symds(const SymParams &sp, const Workspace &w, const Geometry &g, bool pairs) {
    SymDsParams dp;
    dp.sp = sp; dp.sa = w.sa; dp.sb = w.sb;
    if (g.warps == 4) return launch_symds_W<4>(dp, g, pairs);
    if (g.warps == 2) return launch_symds_W<2>(dp, g, pairs);
    return launch_symds_W<1>(dp, g, pairs);
}

int launch_sym(const SymParams &sp, const Geometry &g, bool pairs) {
    if (g.ipt == 4 && g.warps == 4) return launch_sym_IM<4, 4, 3>(sp, g, pairs);
    if (g.ipt == 4 && g.warps == 2) return launch_sym_IM<4, 2, 6>(sp, g, pairs);
    if (g.ipt == 4) return launch_sym_IM<4, 1, 12>(sp, g, pairs);
    if (g.ipt == 2 && g.warps == 4) return launch_sym_IM<2, 4, 4>(sp, g, pairs);
    if (g.ipt == 2) return launch_sym_IM<2, 2, 8>(sp, g, pairs);
    return launch_sym_IM<1, 4, 4>(sp, g, pairs);
}

// One force evaluation: [second half-shift] + rcrit + staging, tiles, reduce + kick.
//   mv_in  : momentum partials for the half-shift folded into prep (nullptr: none)
//   rc_io  : rcrit array read (update_rc = 0) or written (update_rc = 1)
//   nhalf  : number of half-kicks hk applied to v after the evaluation
//   mv_out : momentum partials of the kicked v (nullptr: none)
int enqueue_eval(const Workspace &w, const Geometry &g, double *x, double *v, const double *m, double M_star, int64_t N,
                 double dt_for_rc, double *rc_io, int update_rc, const double *mv_in, double dtc, double *acc,
                 int32_t *pairs, int64_t *npairs, double hk, int nhalf, double *mv_out, bool time_force) {
    const int nblk = body_blocks(N);
    const bool sorted = g.sym && g.sorted;
    if (sorted) {
        // azimuthal order of the staged bodies (sort_staging.cuh), from the positions before the half-shift: the
        // order only decides how many super-tiles can skip the encounter test, never a result
        SortScratch ss;
        ss.key = w.grp.parent; ss.hist = w.grp.size; ss.cursor = w.grp.cursor; ss.tmp = w.grp.tmp;
        ss.perm = w.perm; ss.pos_of = w.pos_of;
        long long nbk = g.Npad_sym / 32;  // ~32 bodies per bucket: short scan, rank sort of ~32 inside a bucket
        if (nbk > N - 1) nbk = N - 1;
        if (nbk < 1) nbk = 1;
        ss.NB = (int)nbk;
        const int nbp = (g.Npad_sym + kGrpThreads - 1) / kGrpThreads, nbn = ((int)N + kGrpThreads - 1) / kGrpThreads;
        nb_sort_clear_kernel<<<nbp, kGrpThreads, 0, stream()>>>(ss, (int)N, g.Npad_sym);
        nb_sort_key_kernel<<<nbn, kGrpThreads, 0, stream()>>>(ss, x, (int)N);
        nb_sort_scan_kernel<<<1, kGrpScanBlock, 0, stream()>>>(ss);
        nb_sort_scatter_kernel<<<nbn, kGrpThreads, 0, stream()>>>(ss, (int)N);
        nb_sort_rank_kernel<<<nbn, kGrpThreads, 0, stream()>>>(ss, (int)N);
    }
    PrepParams pp;
    pp.x = x; pp.v = v; pp.m = m; pp.rcrit = rc_io; pp.jrec = g.sym ? nullptr : w.jrec; pp.mv_in = mv_in;
    pp.sxy = g.sym ? w.sxy : nullptr; pp.szg = w.szg; pp.sthr = w.sthr; pp.Npad_sym = g.Npad_sym;
    pp.sa = g.mixed == 2 ? w.sa : nullptr; pp.sb = w.sb;
    pp.jds = (!g.sym && g.mixed == 1) ? w.jds : nullptr;
    pp.pos_of = sorted ? w.pos_of : nullptr;
    pp.rc_hill = g_cfg.levels > 0 ? w.ml_hill : nullptr; pp.rc_vel = g_cfg.levels > 0 ? w.ml_vel : nullptr;
    pp.npairs = pairs ? reinterpret_cast<unsigned long long *>(npairs) : nullptr;
    pp.status = w.status; pp.dtc = dtc; pp.M_star = M_star; pp.G = g_cfg.G; pp.n1 = g_cfg.n1; pp.n2 = g_cfg.n2;
    pp.absdt = std::fabs(dt_for_rc); pp.nblk_in = nblk; pp.N = (int)N; pp.Nj = g.Nj; pp.Njpad = g.Njpad;
    pp.update_rc = update_rc;
    int64_t cover = N > g.Njpad ? N : g.Njpad;
    if (g.Npad_sym > cover) cover = g.Npad_sym;
    nb_prep_kernel<<<body_blocks(cover), kBodyThreads, 0, stream()>>>(pp);

    ForceParams fp;
    fp.jrec = w.jrec; fp.x = x; fp.rcrit = rc_io; fp.part = w.part; fp.pairs = pairs;
    fp.npairs = pairs ? reinterpret_cast<unsigned long long *>(npairs) : w.npairs_dummy;
    fp.status = w.status; fp.cap = pairs ? g_cfg.pair_capacity : 0; fp.N = (int)N; fp.Nj = g.Nj;
    fp.tiles_total = g.tiles_total; fp.tiles_per_split = g.tiles_per_split; fp.kind = g_cfg.changeover_kind;
    fp.jds = (!g.sym && g.mixed == 1) ? w.jds : nullptr;
    // bounds of the staged super-blocks (before the timing events: they bracket the force kernel alone)
    if (sorted) nb_sort_bounds_kernel<<<g.nsplit, kGrpThreads, 0, stream()>>>(w.sxy, w.perm, rc_io, (int)N, g.S, w.bnd);
    const bool pool = g_cfg.time_force && g_tev_used < kMaxTimed;
    if (pool) {
        while (g_tev_created <= g_tev_used) {
            NB_CUDA(cudaEventCreate(&g_tev[2 * g_tev_created]));
            NB_CUDA(cudaEventCreate(&g_tev[2 * g_tev_created + 1]));
            ++g_tev_created;
        }
        NB_CUDA(cudaEventRecord(g_tev[2 * g_tev_used], stream()));
    } else if (time_force) {
        if (!g_ev0) { NB_CUDA(cudaEventCreate(&g_ev0)); NB_CUDA(cudaEventCreate(&g_ev1)); }
        NB_CUDA(cudaEventRecord(g_ev0, stream()));
    }
    if (g.sym) {
        SymParams sp;
        sp.perm = sorted ? w.perm : nullptr; sp.bnd = sorted ? w.bnd : nullptr;
        sp.sxy = w.sxy; sp.szg = w.szg; sp.sthr = w.sthr; sp.rcrit = rc_io; sp.pairs = pairs;
        sp.npairs = fp.npairs; sp.status = w.status; sp.cap = fp.cap; sp.N = (int)N; sp.S = g.S; sp.nsb = g.nsplit;
        sp.U = g.U; sp.kind = g_cfg.changeover_kind; sp.xcols = g.xcols;
        if (g.band == 0) {
            sp.part_i = w.part; sp.part_j = w.part; sp.stride_i = N; sp.stride_j = N; sp.goff = 0; sp.col0 = 0; sp.ncols = g.nsplit;
            const int lrc = g.mixed == 2 ? launch_symds(sp, w, g, pairs != nullptr) : launch_sym(sp, g, pairs != nullptr);
            if (lrc) return lrc;
        } else {
            // banded: i sides [band][N], then the j sides of the band's bodies [nsb][band S]; folded into acc band by band
            sp.part_i = w.part; sp.part_j = w.part + (size_t)g.band * (size_t)N * 3; sp.stride_i = N;
            for (int c0 = 0; c0 < g.nsplit; c0 += g.band) {
                sp.col0 = c0; sp.ncols = g.nsplit - c0 < g.band ? g.nsplit - c0 : g.band;
                sp.stride_j = (long long)sp.ncols * g.S; sp.goff = c0 * g.S;
                const int lrc = g.mixed == 2 ? launch_symds(sp, w, g, pairs != nullptr) : launch_sym(sp, g, pairs != nullptr);
                if (lrc) return lrc;
                nb_bandsum_kernel<<<nblk, kBodyThreads, 0, stream()>>>(sp.part_i, sp.part_j, acc, (int)N, g.S, sp.col0, sp.ncols,
                                                                      c0 == 0 ? 1 : 0, sorted ? w.perm : nullptr);
            }
        }
    } else {
        launch_force(fp, g, pairs != nullptr);
    }
    if (pool) { NB_CUDA(cudaEventRecord(g_tev[2 * g_tev_used + 1], stream())); ++g_tev_used; }
    else if (time_force) { NB_CUDA(cudaEventRecord(g_ev1, stream())); g_force_timed = true; }

    if (g.sym && g.band > 0)   // acc already holds the sum: it is read as one slot, indexed by body
        nb_kickv_kernel<<<nblk, kBodyThreads, 0, stream()>>>(acc, 1, acc, v, m, (int)N, hk, nhalf, mv_out, nullptr, 0, 0);
    else
        nb_kickv_kernel<<<nblk, kBodyThreads, 0, stream()>>>(w.part, g.nsplit, acc, v, m, (int)N, hk, nhalf, mv_out,
                                                             sorted ? w.perm : nullptr, g.xcols, g.S);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int check_pairs_args(const int32_t *pairs, const int64_t *npairs) {
    if (pairs != nullptr && npairs == nullptr) return fail(NB_E_NULL, "npairs is NULL but pairs is not");
    if (pairs != nullptr && g_cfg.pair_capacity <= 0) return fail(NB_E_BADARG, "pairs given but pair_capacity is 0 (nb_configure)");
    return NB_OK;
}

int ensure_arena(size_t bytes) {
    if (bytes <= g_arena_bytes) return NB_OK;
    if (g_arena) { cudaFree(g_arena); g_arena = nullptr; g_arena_bytes = 0; }
    const size_t want = align_up(bytes + bytes / 8, 1 << 20);
    NB_CUDA(cudaMalloc(&g_arena, want));
    NB_CUDA(cudaMemset(g_arena, 0, 512));
    g_arena_bytes = want;
    return NB_OK;
}

void drop_graph() {
    if (g_graph_exec) { cudaGraphExecDestroy(g_graph_exec); g_graph_exec = nullptr; }
}

// the nine launches of nb_groups (groups.cuh)
void enqueue_groups(const Workspace &w, const int32_t *pairs, const int64_t *npairs, int64_t N, int32_t *label,
                    int32_t *members, int32_t *gstart, int64_t *gstat, const GroupFilter flt = GroupFilter{nullptr, nullptr, 1.0, nullptr},
                    const int ml_level = -1) {
    const int n = (int)N;
    const int nb256 = (n + kGrpThreads - 1) / kGrpThreads, nb1024 = (n + kGrpScanBlock - 1) / kGrpScanBlock;
    long long *gs = reinterpret_cast<long long *>(gstat);
    const long long cap = g_cfg.pair_capacity;
    long long hook_blocks = (cap + kGrpThreads - 1) / kGrpThreads;
    const long long max_blocks = (long long)sm_count() * 16;
    if (hook_blocks > max_blocks) hook_blocks = max_blocks;
    nb_grp_init_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.grp, label, members, gstart, gs, n);
    if (ml_level >= 0)   // edges = the adjacency slots listed at the innermost level (multilevel.cuh)
        nb_ml_hook_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.grp, w.ml, ml_level, n, gs);
    else
        nb_grp_hook_kernel<<<(unsigned)hook_blocks, kGrpThreads, 0, stream()>>>(w.grp, reinterpret_cast<const int2 *>(pairs),
                                                                                reinterpret_cast<const long long *>(npairs), cap, n, gs,
                                                                                w.status, flt);
    nb_grp_compress_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.grp, label, n);
    nb_grp_blocksum_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(w.grp, label, n);
    nb_grp_topscan_kernel<<<1, kGrpScanBlock, 0, stream()>>>(w.grp, nb1024, gstart, gs);
    nb_grp_offsets_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(w.grp, label, n, gstart, gs);
    nb_grp_scatter_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.grp, label, n);
    nb_grp_ranksort_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.grp, label, gs, members);
    nb_grp_giant_kernel<<<sm_count(), kGrpScanBlock, 0, stream()>>>(w.grp, label, n, members);
}

// Which groups the direct solver takes, and the per-body flag nb_drift_kernel obeys (encounter.cuh).
void enqueue_encounter_plan(const Workspace &w, int64_t N, const int32_t *members, const int32_t *gstart, const int64_t *gstat) {
    const int na = (int)((g_cfg.n_active > 0 && g_cfg.n_active < N) ? g_cfg.n_active : N);
    cudaMemsetAsync(w.enc_flag, 0, (size_t)N * sizeof(int), stream());
    long long blocks = (N / 2 + 8) / 8;
    if (blocks > 16LL * sm_count()) blocks = 16LL * sm_count();
    nb_enc_plan_kernel<<<(unsigned)blocks, 256, 0, stream()>>>(members, gstart, reinterpret_cast<const long long *>(gstat), na,
                                                              w.g_core, w.enc_flag);
}

// H_A with encounters for the listed groups (encounter.cuh): groups of up to 32 members by CTAs of 8 warps (one per
// extrapolation column), 33 .. 128 members by CTAs of 128 threads, up to kMaxGroup members by CTAs of kMaxGroup threads
// (one thread per member, columns in sequence)
void enqueue_encounter(const Workspace &w, double *x, double *v, const double *m, const double *rcrit, double M_star,
                       int64_t N, double dt, const int32_t *members, const int32_t *gstart, const int64_t *gstat,
                       bool plan_done, const double *rc_vel = nullptr, int nlev = 1, double *radius = nullptr,
                       int *absorbed_by = nullptr) {
    const long long *gs = reinterpret_cast<const long long *>(gstat);
    if (!plan_done) enqueue_encounter_plan(w, N, members, gstart, gstat);
    EncParams ep;
    ep.x = x; ep.v = v; ep.m = m; ep.rcrit = rcrit; ep.members = members; ep.gstart = gstart;
    ep.gstat = gs; ep.status = w.status; ep.mu = g_cfg.G * M_star; ep.G = g_cfg.G;
    ep.dt = dt; ep.tol = g_cfg.bs_tol > 0.0 ? g_cfg.bs_tol : 1e-12; ep.kind = g_cfg.changeover_kind;
    ep.gcore = w.g_core; ep.rc_vel = rc_vel; ep.nlev = nlev;
    // collisions inside the solver (reading S26): m and radius are then in/out
    ep.m_io = radius ? const_cast<double *>(m) : nullptr; ep.radius = radius; ep.absorbed_by = absorbed_by;
    ep.frad = g_cfg.radius_factor > 0.0 ? g_cfg.radius_factor : 1.0;
    const bool collide = radius != nullptr;
    ep.work = reinterpret_cast<unsigned long long *>(w.status + 16);   // two spare words of the 512-byte status head
    cudaMemsetAsync(ep.work, 0, 2 * sizeof(unsigned long long), stream());
    long long small_blocks = N / 2 + 1;
    const long long cap_blocks = (long long)sm_count() * 8;
    if (small_blocks > cap_blocks) small_blocks = cap_blocks;
    ep.min_size = 1; ep.max_size = 32;
    if (g_cfg.n_active > 0 && g_cfg.n_active < N) {
        // semi-active: the test particles of split groups first (they read the cores' initial state)
        long long sat_blocks = N;
        if (sat_blocks > cap_blocks) sat_blocks = cap_blocks;
        nb_encounter_sat_kernel<<<(unsigned)sat_blocks, 32 * kBsCols, 0, stream()>>>(ep);
    }
    if (nlev > 1) {
        // the multi-level scheme's innermost calls: thousands of easy problems over dt / 2^L -- CTAs of 4 warps, twice as many per SM
        long long b4 = N / 2 + 1;
        if (b4 > 2 * cap_blocks) b4 = 2 * cap_blocks;
        nb_encounter_small_kernel<4><<<(unsigned)b4, 32 * 4, 0, stream()>>>(ep);
    } else {
        nb_encounter_small_kernel<kBsCols><<<(unsigned)small_blocks, 32 * kBsCols, 0, stream()>>>(ep);
    }
    // mid-size groups: CTAs of 128 threads (no register cap: the 1024-thread variant is held to 64 registers and spills)
    ep.min_size = 33; ep.max_size = 128;
    long long mid_blocks = N / 33 + 1;
    if (mid_blocks > 8LL * sm_count()) mid_blocks = 8LL * sm_count();
    nb_encounter_kernel<128><<<(unsigned)mid_blocks, 128, enc_smem_bytes(128, collide), stream()>>>(ep);
    ep.min_size = 129; ep.max_size = kMaxGroup;
    static bool attr_set = false;
    const size_t big_smem = enc_smem_bytes(kMaxGroup, collide);
    if (!attr_set) { cudaFuncSetAttribute(nb_encounter_kernel<kMaxGroup>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)enc_smem_bytes(kMaxGroup, true)); attr_set = true; }
    long long big_blocks = N / 129 + 1;
    if (big_blocks > 2LL * sm_count()) big_blocks = 2LL * sm_count();
    nb_encounter_kernel<kMaxGroup><<<(unsigned)big_blocks, kMaxGroup, big_smem, stream()>>>(ep);
}

// Multi-level changeover (multilevel.cuh): adjacency of the step's pair list, then the recursion
//   advance(l, tau): l == L: direct solver over tau for the groups of P_L; else twice (h = tau/2): detect P_{l+1} +
//   kick h/2 over P_l, Kepler drift h of the bodies that stay at level l, advance(l + 1, h), kick h/2 over P_l
// (the closing kick of the first half and the opening kick of the second share one launch).
void enqueue_ml_adjacency(const Workspace &w, const int32_t *pairs, const int64_t *npairs, int64_t N) {
    const int n = (int)N;
    const int nb256 = (n + kGrpThreads - 1) / kGrpThreads, nb1024 = (n + kGrpScanBlock - 1) / kGrpScanBlock;
    const long long cap = g_cfg.pair_capacity;
    long long pair_blocks = (cap + kGrpThreads - 1) / kGrpThreads;
    const long long max_blocks = (long long)sm_count() * 16;
    if (pair_blocks > max_blocks) pair_blocks = max_blocks;
    if (pair_blocks < 1) pair_blocks = 1;
    const int2 *p2 = reinterpret_cast<const int2 *>(pairs);
    const long long *np = reinterpret_cast<const long long *>(npairs);
    nb_ml_clear_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.ml, n);
    nb_ml_degree_kernel<<<(unsigned)pair_blocks, kGrpThreads, 0, stream()>>>(w.ml, p2, np, cap, n, w.status);
    nb_ml_scan1_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(w.ml, n);
    nb_ml_scan2_kernel<<<1, kGrpScanBlock, 0, stream()>>>(w.ml, nb1024, n);
    nb_ml_scan3_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(w.ml, n);
    nb_ml_fill_kernel<<<(unsigned)pair_blocks, kGrpThreads, 0, stream()>>>(w.ml, p2, np, cap, n);
    nb_ml_sort_kernel<<<(unsigned)(2 * pair_blocks), kGrpThreads, 0, stream()>>>(w.ml, n);
    nb_ml_listed_kernel<<<nb256, kGrpThreads, 0, stream()>>>(w.ml, n, w.ml_listed);
}

void enqueue_ml_advance(const Workspace &w, const MlParams &mp, double M_star, int64_t N, int l, double tau,
                        double *radius = nullptr, int *absorbed_by = nullptr /* collisions in the innermost solver (S26) */) {
    const int nb256 = ((int)N + kGrpThreads - 1) / kGrpThreads;
    if (l == mp.L) {
        // the innermost level: groups of P_L -> plan -> bodies of groups beyond the solver's cap drift -> direct solver
        enqueue_groups(w, nullptr, nullptr, N, w.g_label, w.g_members, w.g_start, w.g_stat, GroupFilter{nullptr, nullptr, 1.0, nullptr}, l);
        enqueue_encounter_plan(w, N, w.g_members, w.g_start, w.g_stat);
        nb_ml_drift_kernel<<<nb256, kGrpThreads, 0, stream()>>>(mp, l, tau, w.enc_flag);
        enqueue_encounter(w, mp.x, mp.v, mp.m, mp.hill, M_star, N, tau, w.g_members, w.g_start, w.g_stat, true, mp.vel, mp.L + 1,
                          radius, absorbed_by);
        return;
    }
    const double h = 0.5 * tau;
    nb_ml_kick_kernel<true><<<nb256, kGrpThreads, 0, stream()>>>(mp, l, 0.5 * h, 1);
    nb_ml_drift_kernel<<<nb256, kGrpThreads, 0, stream()>>>(mp, l, h, nullptr);
    enqueue_ml_advance(w, mp, M_star, N, l + 1, h, radius, absorbed_by);
    nb_ml_kick_kernel<true><<<nb256, kGrpThreads, 0, stream()>>>(mp, l, 0.5 * h, 2);
    nb_ml_drift_kernel<<<nb256, kGrpThreads, 0, stream()>>>(mp, l, h, nullptr);
    enqueue_ml_advance(w, mp, M_star, N, l + 1, h, radius, absorbed_by);
    nb_ml_kick_kernel<false><<<nb256, kGrpThreads, 0, stream()>>>(mp, l, 0.5 * h, 1);
}

MlParams ml_params(const Workspace &w, double *x, double *v, const double *m, const double *hill, const double *vel,
                   double M_star, int64_t N) {
    MlParams mp;
    mp.x = x; mp.v = v; mp.m = m; mp.hill = hill; mp.vel = vel; mp.s = w.ml; mp.status = w.status;
    mp.G = g_cfg.G; mp.mu = g_cfg.G * M_star; mp.N = (int)N; mp.kind = g_cfg.changeover_kind; mp.L = g_cfg.levels;
    return mp;
}

// ---- small N: whole steps in one cooperative launch (step_small.cuh) ----

template <int I>
int launch_step_small_I(const SmallStepParams &q, bool pairs, int work_items) {
    auto go = [&](auto kern) -> int {
        int dev = 0, coop = 0, per_sm = 0;
        NB_CUDA(cudaGetDevice(&dev));
        NB_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        if (!coop) return NB_E_BADARG;
        NB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kForceThreads, 0));
        if (per_sm < 1) return NB_E_BADARG;
        int grid = per_sm * sm_count();
        if (grid > work_items) grid = work_items;
        if (grid < 1) grid = 1;
        SmallStepParams qq = q;
        void *args[] = {&qq};
        NB_CUDA(cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(kForceThreads), args, 0, stream()));
        return NB_OK;
    };
    return pairs ? go(nb_step_small_kernel<I, true>) : go(nb_step_small_kernel<I, false>);
}

int launch_step_small(const Workspace &w, const Geometry &g, double *x, double *v, const double *m, double M_star, int64_t N,
                      double dt, double *rc_io, int update_rc, double *acc, int32_t *pairs, int64_t *npairs, int64_t nsteps) {
    SmallStepParams q;
    PrepParams &pp = q.pp;
    pp.x = x; pp.v = v; pp.m = m; pp.rcrit = rc_io; pp.rc_hill = nullptr; pp.rc_vel = nullptr; pp.jrec = w.jrec;
    pp.sxy = nullptr; pp.szg = nullptr; pp.sthr = nullptr; pp.Npad_sym = 0; pp.pos_of = nullptr; pp.mv_in = nullptr;
    pp.sa = nullptr; pp.sb = nullptr; pp.jds = nullptr;
    pp.npairs = pairs ? reinterpret_cast<unsigned long long *>(npairs) : nullptr;
    pp.status = w.status; pp.dtc = 0.5 * dt; pp.M_star = M_star; pp.G = g_cfg.G; pp.n1 = g_cfg.n1; pp.n2 = g_cfg.n2;
    pp.absdt = std::fabs(dt); pp.nblk_in = body_blocks(N); pp.N = (int)N; pp.Nj = g.Nj; pp.Njpad = g.Njpad;
    pp.update_rc = update_rc;
    ForceParams &fp = q.fp;
    fp.jrec = w.jrec; fp.x = x; fp.rcrit = rc_io; fp.part = w.part; fp.pairs = pairs;
    fp.npairs = pairs ? reinterpret_cast<unsigned long long *>(npairs) : w.npairs_dummy;
    fp.status = w.status; fp.cap = pairs ? g_cfg.pair_capacity : 0; fp.N = (int)N; fp.Nj = g.Nj;
    fp.tiles_total = g.tiles_total; fp.tiles_per_split = g.tiles_per_split; fp.kind = g_cfg.changeover_kind; fp.jds = nullptr;
    q.acc = acc; q.mvA = w.mvA; q.mvB = w.mvB; q.mu = g_cfg.G * M_star; q.dt = dt; q.hk = 0.5 * dt; q.dtc = 0.5 * dt;
    q.nsteps = (int)(nsteps > 2000000000LL ? 2000000000LL : nsteps); q.last_nhalf = 1;
    q.iblocks = g.iblocks; q.nsplit = g.nsplit; q.nblk = body_blocks(N);
    if ((int64_t)q.nsteps != nsteps) return NB_E_BADARG;
    const int items = g.iblocks * g.nsplit > q.nblk ? g.iblocks * g.nsplit : q.nblk;
    if (g.ipt == 4) return launch_step_small_I<4>(q, pairs != nullptr, items);
    if (g.ipt == 2) return launch_step_small_I<2>(q, pairs != nullptr, items);
    return launch_step_small_I<1>(q, pairs != nullptr, items);
}

int step_impl(double *x, double *v, const double *m, double M_star, int64_t N, double dt, double *rcrit, double *acc,
              int32_t *pairs, int64_t *npairs, int64_t nsteps) {
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !acc) return fail(NB_E_NULL, "nb_step: x, v, m, acc must not be NULL");
    if (nsteps < 0) return fail(NB_E_BADARG, "nsteps < 0");
    const int update_rc = !(g_cfg.n1 == 0.0 && g_cfg.n2 == 0.0);
    if (!rcrit && !update_rc) return fail(NB_E_NULL, "nb_step: rcrit is NULL and n1 == n2 == 0");
    if ((rc = check_pairs_args(pairs, npairs))) return rc;
    const Geometry g = geometry(N, g_cfg.n_active);
    Workspace w;
    if ((rc = check_workspace(N, g, &w))) return rc;
    double *rc_io = rcrit ? rcrit : w.rc_scratch;
    const double hk = 0.5 * dt, dtc = 0.5 * dt, mu = g_cfg.G * M_star;
    const int nblk = body_blocks(N);

    // extra force (Eq. 8, reading S24): D(dt/2) before the opening and after the closing half-kick
    const bool drag = g_cfg.drag_gamma > 0.0;
    auto enqueue_D = [&]() {
        nb_midpoint_drag_kernel<<<nblk, kBodyThreads, 0, stream()>>>(x, v, (int)N, mu, 0.5 * dt, g_cfg.drag_gamma, g_cfg.drag_power,
                                                                     g_cfg.drag_eta, g_cfg.midpoint_tol, g_cfg.midpoint_iters > 0 ? g_cfg.midpoint_iters : 50, w.status);
    };
    // opening half-kick from the cached force (reads acc as a 1-split partial) + momentum partials
    auto kick_only = [&]() { nb_kickv_kernel<<<nblk, kBodyThreads, 0, stream()>>>(acc, 1, acc, v, m, (int)N, hk, 1, w.mvA, nullptr, 0, 0); };
    if (g_cfg.reuse_acc && nsteps > 0) {
        // acc already is the force at the current x
        if (drag) enqueue_D();
        kick_only();
    } else if (!drag) {
        // evaluation at t0 (+ opening half-kick of the first step)
        if ((rc = enqueue_eval(w, g, x, v, m, M_star, N, dt, rc_io, update_rc, nullptr, 0.0, acc, pairs, npairs, hk,
                               nsteps > 0 ? 1 : 0, w.mvA, nsteps == 0)))
            return rc;
    } else {
        if ((rc = enqueue_eval(w, g, x, v, m, M_star, N, dt, rc_io, update_rc, nullptr, 0.0, acc, pairs, npairs, hk, 0, nullptr,
                               nsteps == 0)))
            return rc;
        if (nsteps > 0) { enqueue_D(); kick_only(); }
    }

    const bool enc = g_cfg.resolve_encounters != 0;
    if (enc && !pairs) return fail(NB_E_BADARG, "nb_step: resolve_encounters needs the pair list (pairs != NULL)");
    const bool ml = enc && g_cfg.levels > 0;
    // collisions examined inside the direct solver (reading S26): m and the radii change on the way
    const bool coll = enc && g_cfg.collide_radius != nullptr;
    if (coll && !g_cfg.collide_absorbed_by) return fail(NB_E_NULL, "nb_step: collide_radius is set but collide_absorbed_by is NULL");
    if (coll && g.Nj != N) return fail(NB_E_BADARG, "nb_step: collisions inside the solver (collide_radius) are defined for the fully active case");
    if (ml && g.Nj != N) return fail(NB_E_BADARG, "nb_step: the multi-level changeover (levels > 0) is defined for the fully active case only");
    // force evaluation that closes a step: closing half-kick [+ opening half-kick of the next step]; with the extra
    // force the two half-kicks are separated by D(dt/2) D(dt/2)
    auto close_step = [&](int nhalf) -> int {
        if (!drag)
            return enqueue_eval(w, g, x, v, m, M_star, N, dt, rc_io, update_rc, w.mvB, dtc, acc, pairs, npairs, hk, nhalf, w.mvA, false);
        const int erc = enqueue_eval(w, g, x, v, m, M_star, N, dt, rc_io, update_rc, w.mvB, dtc, acc, pairs, npairs, hk, 1, nullptr, false);
        if (erc) return erc;
        enqueue_D();
        if (nhalf == 2) { enqueue_D(); kick_only(); }
        return NB_OK;
    };
    auto enqueue_step = [&](int nhalf) -> int {
        if (ml) {
            // multi-level changeover: every body of the step's pair list goes through the levels; the plain
            // drift kernel moves the others (and shifts everybody)
            enqueue_ml_adjacency(w, pairs, npairs, N);
            nb_drift_kernel<<<nblk, kBodyThreads, 0, stream()>>>(x, v, m, (int)N, mu, dt, w.mvA, nblk, dtc, M_star, nullptr, w.status,
                                                                 w.ml_listed);
            enqueue_ml_advance(w, ml_params(w, x, v, m, w.ml_hill, w.ml_vel, M_star, N), M_star, N, 0, dt,
                               coll ? g_cfg.collide_radius : nullptr, coll ? g_cfg.collide_absorbed_by : nullptr);
            nb_momentum_kernel<<<nblk, kBodyThreads, 0, stream()>>>(v, m, (int)N, w.mvB);
            return close_step(nhalf);
        }
        // groups of the pair list of the evaluation that opened this step
        if (enc) {
            enqueue_groups(w, pairs, npairs, N, w.g_label, w.g_members, w.g_start, w.g_stat);
            enqueue_encounter_plan(w, N, w.g_members, w.g_start, w.g_stat);
        }
        // C(dt/2) A(dt): first half-shift folded into the drift kernel; members of groups are only shifted there
        // and then propagated through their encounter by the direct solver
        nb_drift_kernel<<<nblk, kBodyThreads, 0, stream()>>>(x, v, m, (int)N, mu, dt, w.mvA, nblk, dtc, M_star,
                                                             enc ? nullptr : w.mvB, w.status, enc ? w.enc_flag : nullptr);
        if (enc) {
            enqueue_encounter(w, x, v, m, rc_io, M_star, N, dt, w.g_members, w.g_start, w.g_stat, true, nullptr, 1,
                              coll ? g_cfg.collide_radius : nullptr, coll ? g_cfg.collide_absorbed_by : nullptr);
            nb_momentum_kernel<<<nblk, kBodyThreads, 0, stream()>>>(v, m, (int)N, w.mvB);
        }
        // C(dt/2) folded into prep; force; B(dt/2) [+ B(dt/2) of the next step]
        return close_step(nhalf);
    };

    // Small N: all nsteps steps in ONE cooperative launch (step_small.cuh) -- same device functions, same virtual blocks,
    // bit-identical results; taken when the step is the plain one (one-sided fp64 kernel, no encounters / extra force)
    if (nsteps > 0 && g_cfg.use_graph && !g_cfg.time_force && !enc && !drag && !g.sym && !g.mixed && N <= kSmallStepMaxN) {
        const int frc = launch_step_small(w, g, x, v, m, M_star, N, dt, rc_io, update_rc, acc, pairs, npairs, nsteps);
        if (frc != NB_E_BADARG) return frc;   // NB_E_BADARG: the cooperative launch is not available here -> multi-launch path
    }
    const int64_t interior = nsteps > 0 ? nsteps - 1 : 0;
    if (interior > 0 && g_cfg.use_graph && !g_cfg.time_force) {
        StepKey key;
        std::memset(&key, 0, sizeof(key));
        key.x = x; key.v = v; key.m = m; key.rcrit = rc_io; key.acc = acc; key.pairs = pairs; key.npairs = npairs;
        key.ws = g_cfg.workspace; key.stream = g_cfg.stream; key.N = N; key.n_active = g_cfg.n_active;
        key.cap = g_cfg.pair_capacity; key.dt = dt; key.M_star = M_star; key.G = g_cfg.G; key.n1 = g_cfg.n1;
        key.n2 = g_cfg.n2; key.kind = g_cfg.changeover_kind; key.bs_tol = g_cfg.bs_tol; key.enc = (enc ? 1 : 0) + 2 * g.sorted; key.ipt = g.S * 1000 + g.ipt * 100 + g.minb * 10 + g.warps + 100000 * g.xcols; key.jsplit = g.nsplit; key.band = g.band;
        key.ws_bytes = g_cfg.workspace_bytes; key.levels = g_cfg.levels;
        key.radius = coll ? g_cfg.collide_radius : nullptr; key.absorbed_by = coll ? g_cfg.collide_absorbed_by : nullptr;
        key.drag_gamma = g_cfg.drag_gamma; key.drag_eta = g_cfg.drag_eta; key.midpoint_tol = g_cfg.midpoint_tol;
        key.drag_power = g_cfg.drag_power; key.midpoint_iters = g_cfg.midpoint_iters + 1000 * g.mixed;
        const bool hop = !stream_capturable();
        if (hop) {
            if (!g_own_stream) {
                NB_CUDA(cudaStreamCreateWithFlags(&g_own_stream, cudaStreamNonBlocking));
                NB_CUDA(cudaEventCreateWithFlags(&g_ev_in, cudaEventDisableTiming));
                NB_CUDA(cudaEventCreateWithFlags(&g_ev_out, cudaEventDisableTiming));
            }
            NB_CUDA(cudaEventRecord(g_ev_in, stream()));
            NB_CUDA(cudaStreamWaitEvent(g_own_stream, g_ev_in, 0));
            g_on_own_stream = true;
        }
        auto replay = [&]() -> int {
            if (!g_graph_exec || std::memcmp(&key, &g_graph_key, sizeof(key)) != 0) {
                drop_graph();
                cudaGraph_t graph = nullptr;
                NB_CUDA(cudaStreamBeginCapture(stream(), cudaStreamCaptureModeRelaxed));
                const int erc = enqueue_step(2);
                cudaError_t ce = cudaStreamEndCapture(stream(), &graph);
                if (erc) { if (graph) cudaGraphDestroy(graph); return erc; }
                if (ce != cudaSuccess) return fail(NB_E_CUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(ce));
                ce = cudaGraphInstantiate(&g_graph_exec, graph, 0);
                cudaGraphDestroy(graph);
                if (ce != cudaSuccess) { g_graph_exec = nullptr; return fail(NB_E_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(ce)); }
                g_graph_key = key;
            }
            for (int64_t s = 0; s < interior; ++s) NB_CUDA(cudaGraphLaunch(g_graph_exec, stream()));
            return NB_OK;
        };
        rc = replay();
        if (hop) {
            cudaError_t ce = cudaEventRecord(g_ev_out, g_own_stream);
            g_on_own_stream = false;
            if (ce == cudaSuccess) ce = cudaStreamWaitEvent(stream(), g_ev_out, 0);
            if (!rc && ce != cudaSuccess) rc = fail(NB_E_CUDA, "stream hand-back failed: %s", cudaGetErrorString(ce));
        }
        if (rc) return rc;
    } else {
        for (int64_t s = 0; s < interior; ++s)
            if ((rc = enqueue_step(2))) return rc;
    }
    if (nsteps > 0 && (rc = enqueue_step(1))) return rc;
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int kick_impl(const double *x, double *v, const double *m, double M_star, int64_t N, double dt, const double *rcrit,
              double *acc, int32_t *pairs, int64_t *npairs) {
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !acc) return fail(NB_E_NULL, "nb_kick: x, v, m, acc must not be NULL");
    if ((rc = check_pairs_args(pairs, npairs))) return rc;
    const Geometry g = geometry(N, g_cfg.n_active);
    Workspace w;
    if ((rc = check_workspace(N, g, &w))) return rc;
    double *rc_io = rcrit ? const_cast<double *>(rcrit) : w.rc_scratch;
    return enqueue_eval(w, g, const_cast<double *>(x), v, m, M_star, N, dt, rc_io, rcrit ? 0 : 1, nullptr, 0.0, acc, pairs,
                        npairs, dt, dt != 0.0 ? 1 : 0, nullptr, true);
}

}  // namespace

// ---- nb_kick_static: the kick with its scratch in a static device array (include/nbkick.h) --------------------------
// Callers that cannot allocate (stream capture, serving loops, harnesses that forbid cudaMalloc) get the scratch from
// here: NB_STATIC_SCRATCH_BYTES of device memory that every GPU which loads the library holds until the process exits.
// In HOST code the name below is only a stand-in for the symbol, never a device address: the address a kernel can use
// comes from cudaGetSymbolAddress, asked once per device with that device current (static_scratch_for_current_device).
static __device__ __align__(256) unsigned char g_static_scratch[NB_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
void *g_static_scratch_ptr[kStaticMaxDevices] = {nullptr};

int static_scratch_for_current_device(void **out) {
    int dev = -1;
    NB_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(NB_E_BADARG, "nb_kick_static: device ordinal %d out of range", dev);
    if (g_static_scratch_ptr[dev] == nullptr) {
        void *ptr = nullptr;
        NB_CUDA(cudaGetSymbolAddress(&ptr, g_static_scratch));
        if (ptr == nullptr || (reinterpret_cast<uintptr_t>(ptr) & 255u) != 0)
            return fail(NB_E_CUDA, "nb_kick_static: cudaGetSymbolAddress gave an unusable address");
        g_static_scratch_ptr[dev] = ptr;
    }
    *out = g_static_scratch_ptr[dev];
    return NB_OK;
}

}  // namespace

extern "C" {

int nb_kick_static_setup(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    void *ptr = nullptr;
    return static_scratch_for_current_device(&ptr);
}

int nb_kick_static(const double *x, double *v, const double *m, double M_star, int64_t N, double dt, const double *rcrit,
                   double *acc, int32_t *pairs, int64_t *npairs, int64_t *status8) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !acc) return fail(NB_E_NULL, "nb_kick_static: x, v, m, acc must not be NULL");
    if ((rc = check_pairs_args(pairs, npairs))) return rc;
    void *scratch = nullptr;
    if ((rc = static_scratch_for_current_device(&scratch))) return rc;
    const Geometry g = geometry(N, g_cfg.n_active);
    const size_t need = carve(nullptr, N, g).bytes;
    if (need > (size_t)NB_STATIC_SCRATCH_BYTES)
        return fail(NB_E_WORKSPACE, "nb_kick_static: N = %lld needs %zu bytes of scratch, the static array has %zu "
                    "(NB_STATIC_SCRATCH_BYTES); use nb_kick with a caller-owned workspace", (long long)N, need,
                    (size_t)NB_STATIC_SCRATCH_BYTES);
    const Workspace w = carve(scratch, N, g);
    // the array keeps the previous call's contents.  What must start at zero: the status words (the kernels only ever
    // add to them).  Everything else -- staged records, partial slots, rc scratch -- is written in full by this call
    // before it is read (every (slot, body) exactly once per evaluation), and npairs is zeroed by nb_prep_kernel.
    NB_CUDA(cudaMemsetAsync(w.status, 0, 512, stream()));
    double *rc_io = rcrit ? const_cast<double *>(rcrit) : w.rc_scratch;
    const int saved_time_force = g_cfg.time_force;
    g_cfg.time_force = 0;   // timing events are created lazily (cudaEventCreate): not on this path
    rc = enqueue_eval(w, g, const_cast<double *>(x), v, m, M_star, N, dt, rc_io, rcrit ? 0 : 1, nullptr, 0.0, acc, pairs,
                      npairs, dt, dt != 0.0 ? 1 : 0, nullptr, false);
    g_cfg.time_force = saved_time_force;
    if (rc) return rc;
    if (status8 != nullptr)
        NB_CUDA(cudaMemcpyAsync(status8, w.status, ST_COUNT * sizeof(int64_t), cudaMemcpyDeviceToDevice, stream()));
    return NB_OK;
}

void nb_default_config(nb_config *cfg) {
    if (!cfg) return;
    std::memset(cfg, 0, sizeof(*cfg));
    cfg->G = 0.01720209895 * 0.01720209895;
    cfg->n1 = 3.0;
    cfg->n2 = 0.4;
    cfg->changeover_kind = NB_CHANGEOVER_RATIONAL;
    cfg->use_graph = 1;
    cfg->reuse_acc = 0;
    cfg->time_force = 0;
    cfg->force_kernel = NB_FORCE_AUTO;
    cfg->sym_block = 0;
    cfg->resolve_encounters = 0;
    cfg->bs_tol = 1e-12;
    cfg->radius_factor = 1.0;
    cfg->sort_staging = NB_SORT_AUTO;
    cfg->levels = 0;
    cfg->drag_gamma = 0.0;
    cfg->drag_eta = 0.0;
    cfg->drag_power = 0;
    cfg->midpoint_iters = 50;
    cfg->midpoint_tol = 1e-14;
    cfg->precision = NB_PRECISION_F64;
    cfg->slot_bytes_max = 0;
}

int nb_configure(const nb_config *cfg) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!cfg) return fail(NB_E_NULL, "nb_configure: cfg is NULL");
    if (!(cfg->G > 0.0) || !std::isfinite(cfg->G)) return fail(NB_E_BADARG, "G must be finite and > 0");
    if (!(cfg->n1 >= 0.0) || !(cfg->n2 >= 0.0) || !std::isfinite(cfg->n1) || !std::isfinite(cfg->n2))
        return fail(NB_E_BADARG, "n1, n2 must be finite and >= 0");
    if (cfg->pair_capacity < 0 || cfg->n_active < 0) return fail(NB_E_BADARG, "pair_capacity and n_active must be >= 0");
    if (cfg->changeover_kind != NB_CHANGEOVER_RATIONAL && cfg->changeover_kind != NB_CHANGEOVER_QUINTIC)
        return fail(NB_E_BADARG, "unknown changeover_kind %d", cfg->changeover_kind);
    if (cfg->i_per_thread != 0 && cfg->i_per_thread != 1 && cfg->i_per_thread != 2 && cfg->i_per_thread != 4)
        return fail(NB_E_BADARG, "i_per_thread must be 0, 1, 2 or 4");
    if (cfg->j_splits < 0) return fail(NB_E_BADARG, "j_splits must be >= 0");
    if (cfg->force_kernel != NB_FORCE_AUTO && cfg->force_kernel != NB_FORCE_TILES && cfg->force_kernel != NB_FORCE_SYMMETRIC)
        return fail(NB_E_BADARG, "unknown force_kernel %d", cfg->force_kernel);
    if (cfg->sym_block != 0 && cfg->sym_block != 128 && cfg->sym_block != 256 && cfg->sym_block != 512 && cfg->sym_block != 1024 && cfg->sym_block != 2048)
        return fail(NB_E_BADARG, "sym_block must be 0, 128, 256, 512, 1024 or 2048");
    if (!(cfg->bs_tol >= 0.0) || !std::isfinite(cfg->bs_tol)) return fail(NB_E_BADARG, "bs_tol must be finite and >= 0");
    if (cfg->sort_staging != NB_SORT_AUTO && cfg->sort_staging != NB_SORT_ON && cfg->sort_staging != NB_SORT_OFF)
        return fail(NB_E_BADARG, "unknown sort_staging %d", cfg->sort_staging);
    if (!(cfg->radius_factor >= 0.0) || !std::isfinite(cfg->radius_factor)) return fail(NB_E_BADARG, "radius_factor must be finite and >= 0");
    if (!(cfg->drag_gamma >= 0.0) || !std::isfinite(cfg->drag_gamma) || !std::isfinite(cfg->drag_eta) ||
        (cfg->drag_power != 0 && cfg->drag_power != 1) || cfg->midpoint_iters < 0 || !(cfg->midpoint_tol >= 0.0))
        return fail(NB_E_BADARG, "drag_gamma >= 0, finite drag_eta, drag_power 0 or 1, midpoint_iters >= 0, midpoint_tol >= 0");
    if (cfg->precision != NB_PRECISION_F64 && cfg->precision != NB_PRECISION_MIXED) return fail(NB_E_BADARG, "unknown precision %d", cfg->precision);
    if (cfg->slot_bytes_max < 0) return fail(NB_E_BADARG, "slot_bytes_max < 0");
    if (cfg->levels < 0 || cfg->levels > kMaxLevels) return fail(NB_E_BADARG, "levels must be 0 .. %d", kMaxLevels);
    g_cfg = *cfg;
    return NB_OK;
}

size_t nb_workspace_bytes(int64_t N) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (N <= 0 || N > 2147483647LL) return 0;
    const Geometry g = geometry(N, g_cfg.n_active <= N ? g_cfg.n_active : 0);
    return carve(nullptr, N, g).bytes;
}

int nb_force_geometry(int64_t N, int64_t *out5) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!out5) return fail(NB_E_NULL, "out5 is NULL");
    if (N <= 0 || N > 2147483647LL) return fail(NB_E_BADN, "N out of range");
    const Geometry g = geometry(N, g_cfg.n_active <= N ? g_cfg.n_active : 0);
    out5[0] = g.ipt; out5[1] = g.iblocks; out5[2] = g.nsplit; out5[3] = g.sym ? 32 * g.warps : kForceThreads; out5[4] = g.sym ? -g.S : kTileJ;
    return NB_OK;
}

int nb_rcrit(const double *x, const double *v, const double *m, double M_star, int64_t N, double dt, double *rcrit) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !rcrit) return fail(NB_E_NULL, "nb_rcrit: NULL argument");
    nb_rcrit_kernel<<<body_blocks(N), kBodyThreads, 0, stream()>>>(x, v, m, rcrit, (int)N, M_star, g_cfg.G, g_cfg.n1,
                                                                   g_cfg.n2, std::fabs(dt));
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_kick(const double *x, double *v, const double *m, double M_star, int64_t N, double dt, const double *rcrit,
            double *acc, int32_t *pairs, int64_t *npairs) {
    std::lock_guard<std::mutex> lk(g_mu);
    return kick_impl(x, v, m, M_star, N, dt, rcrit, acc, pairs, npairs);
}

int nb_shift(double *x, const double *v, const double *m, double M_star, int64_t N, double dt) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m) return fail(NB_E_NULL, "nb_shift: NULL argument");
    Workspace w;
    if ((rc = check_workspace_head(N, 1, &w))) return rc;
    const int nblk = body_blocks(N);
    nb_momentum_kernel<<<nblk, kBodyThreads, 0, stream()>>>(v, m, (int)N, w.mvA);
    nb_shift_kernel<<<nblk, kBodyThreads, 0, stream()>>>(x, w.mvA, nblk, (int)N, dt, M_star);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_drift_kepler(double *x, double *v, double M_star, int64_t N, double dt) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v) return fail(NB_E_NULL, "nb_drift_kepler: NULL argument");
    Workspace w;
    if ((rc = check_workspace_head(N, 0, &w))) return rc;
    nb_drift_kernel<<<body_blocks(N), kBodyThreads, 0, stream()>>>(x, v, nullptr, (int)N, g_cfg.G * M_star, dt, nullptr, 0,
                                                                   0.0, M_star, nullptr, w.status, nullptr);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_midpoint_drag(const double *x, double *v, double M_star, int64_t N, double dt) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v) return fail(NB_E_NULL, "nb_midpoint_drag: NULL argument");
    Workspace w;
    if ((rc = check_workspace_head(N, 0, &w))) return rc;
    nb_midpoint_drag_kernel<<<body_blocks(N), kBodyThreads, 0, stream()>>>(x, v, (int)N, g_cfg.G * M_star, dt, g_cfg.drag_gamma,
                                                                           g_cfg.drag_power, g_cfg.drag_eta, g_cfg.midpoint_tol,
                                                                           g_cfg.midpoint_iters > 0 ? g_cfg.midpoint_iters : 50, w.status);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_step(double *x, double *v, const double *m, double M_star, int64_t N, double dt, double *rcrit, double *acc,
            int32_t *pairs, int64_t *npairs, int64_t nsteps) {
    std::lock_guard<std::mutex> lk(g_mu);
    return step_impl(x, v, m, M_star, N, dt, rcrit, acc, pairs, npairs, nsteps);
}

int nb_groups(const int32_t *pairs, const int64_t *npairs, int64_t N, int32_t *label, int32_t *members, int32_t *gstart,
              int64_t *gstat) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (N <= 0 || N > 2147483647LL) return fail(NB_E_BADN, "N = %lld out of range (1 .. 2^31-1)", (long long)N);
    if (!pairs || !npairs || !label || !members || !gstart || !gstat) return fail(NB_E_NULL, "nb_groups: NULL argument");
    if (g_cfg.pair_capacity <= 0) return fail(NB_E_BADARG, "nb_groups: pair_capacity is 0 (nb_configure)");
    Workspace w;
    int rc = check_workspace_head(N, 2, &w);
    if (rc) return rc;
    enqueue_groups(w, pairs, npairs, N, label, members, gstart, gstat);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_merge(double *x, double *v, double *m, double *radius, int64_t N, const int32_t *pairs, const int64_t *npairs,
             int32_t *survivor_of, int64_t *mstat) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (N <= 0 || N > 2147483647LL) return fail(NB_E_BADN, "N = %lld out of range (1 .. 2^31-1)", (long long)N);
    if (!x || !v || !m || !radius || !pairs || !npairs || !survivor_of || !mstat) return fail(NB_E_NULL, "nb_merge: NULL argument");
    if (g_cfg.pair_capacity <= 0) return fail(NB_E_BADARG, "nb_merge: pair_capacity is 0 (nb_configure)");
    if (g_cfg.n_active > N) return fail(NB_E_BADARG, "n_active = %lld > N = %lld", (long long)g_cfg.n_active, (long long)N);
    const Geometry g = geometry(N, g_cfg.n_active);
    Workspace w;
    int rc = check_workspace(N, g, &w);  // the partial-sum area doubles as the compaction buffer (64 bytes per body)
    if (rc) return rc;
    const int n = (int)N;
    const int nb256 = (n + kGrpThreads - 1) / kGrpThreads, nb1024 = (n + kGrpScanBlock - 1) / kGrpScanBlock;
    long long *ms = reinterpret_cast<long long *>(mstat);
    long long *ncoll = reinterpret_cast<long long *>(w.npairs_dummy) + 8;   // spare words of the 256-byte slot
    NB_CUDA(cudaMemsetAsync(ncoll, 0, sizeof(long long), stream()));
    GroupFilter flt{x, radius, g_cfg.radius_factor > 0.0 ? g_cfg.radius_factor : 1.0, ncoll};
    enqueue_groups(w, pairs, npairs, N, survivor_of, w.g_members, w.g_start, w.g_stat, flt);
    int *alive = w.grp.cursor;                                              // free again after the member lists are built
    nb_mrg_alive_init_kernel<<<nb256, kGrpThreads, 0, stream()>>>(alive, n);
    nb_mrg_merge_kernel<<<(n / 2 + kGrpThreads) / kGrpThreads, kGrpThreads, 0, stream()>>>(
        x, v, m, radius, w.g_members, w.g_start, reinterpret_cast<const long long *>(w.g_stat), alive);
    const int na = (int)((g_cfg.n_active > 0 && g_cfg.n_active < N) ? g_cfg.n_active : N);
    nb_mrg_blocksum_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(alive, n, na, w.grp.bsum);
    nb_mrg_topscan_kernel<<<1, kGrpScanBlock, 0, stream()>>>(w.grp.bsum, nb1024, n, reinterpret_cast<const long long *>(w.g_stat),
                                                             ncoll, ms);
    nb_mrg_scatter_kernel<<<nb1024, kGrpScanBlock, 0, stream()>>>(x, v, m, radius, alive, w.grp.bsum, n, w.part);
    nb_mrg_copyback_kernel<<<nb256, kGrpThreads, 0, stream()>>>(x, v, m, radius, w.part, ms);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_encounter(double *x, double *v, const double *m, const double *rcrit, double M_star, int64_t N, double dt,
                 const int32_t *members, const int32_t *gstart, const int64_t *gstat) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !rcrit || !members || !gstart || !gstat) return fail(NB_E_NULL, "nb_encounter: NULL argument");
    Workspace w;
    if ((rc = check_workspace_head(N, 2, &w))) return rc;
    enqueue_encounter(w, x, v, m, rcrit, M_star, N, dt, members, gstart, gstat, false);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_encounter_collide(double *x, double *v, double *m, double *radius, const double *rcrit, double M_star, int64_t N,
                         double dt, const int32_t *members, const int32_t *gstart, const int64_t *gstat, int32_t *absorbed_by) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !radius || !rcrit || !members || !gstart || !gstat || !absorbed_by)
        return fail(NB_E_NULL, "nb_encounter_collide: NULL argument");
    if (g_cfg.n_active > 0 && g_cfg.n_active < N) return fail(NB_E_BADARG, "nb_encounter_collide: fully active case only");
    Workspace w;
    if ((rc = check_workspace_head(N, 2, &w))) return rc;
    enqueue_encounter(w, x, v, m, rcrit, M_star, N, dt, members, gstart, gstat, false, nullptr, 1, radius, absorbed_by);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int nb_encounter_levels(double *x, double *v, const double *m, const double *rc_hill, const double *rc_vel, double M_star,
                        int64_t N, double dt, const int32_t *pairs, const int64_t *npairs) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !rc_hill || !rc_vel || !pairs || !npairs) return fail(NB_E_NULL, "nb_encounter_levels: NULL argument");
    if (g_cfg.levels <= 0) return fail(NB_E_BADARG, "nb_encounter_levels: levels is 0 (nb_configure)");
    if (g_cfg.pair_capacity <= 0) return fail(NB_E_BADARG, "nb_encounter_levels: pair_capacity is 0 (nb_configure)");
    if (g_cfg.n_active > 0 && g_cfg.n_active < N) return fail(NB_E_BADARG, "nb_encounter_levels: fully active case only");
    Workspace w;
    if ((rc = check_workspace_head(N, 3, &w))) return rc;
    enqueue_ml_adjacency(w, pairs, npairs, N);
    enqueue_ml_advance(w, ml_params(w, x, v, m, rc_hill, rc_vel, M_star, N), M_star, N, 0, dt);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

// ---- host-buffer forms: copy in, run the device path on the private arena, copy out ----
static int host_run(bool is_step, double *x, double *v, const double *m, double M_star, int64_t N, double dt,
                    double *rcrit, bool rcrit_out, double *acc, int32_t *pairs, int64_t *npairs, int64_t nsteps) {
    int rc = check_common(N, dt, M_star);
    if (rc) return rc;
    if (!x || !v || !m || !acc) return fail(NB_E_NULL, "host call: x, v, m, acc must not be NULL");
    if ((rc = check_pairs_args(pairs, npairs))) return rc;
    const Geometry g = geometry(N, g_cfg.n_active);
    const size_t ws_bytes = carve(nullptr, N, g).bytes;
    const size_t n3 = align_up((size_t)N * 3 * sizeof(double), 256), n1 = align_up((size_t)N * sizeof(double), 256);
    const size_t pb = pairs ? align_up((size_t)g_cfg.pair_capacity * 2 * sizeof(int32_t), 256) : 0;
    const size_t total = ws_bytes + 3 * n3 + 2 * n1 + pb + 256;
    if ((rc = ensure_arena(total))) return rc;
    char *b = static_cast<char *>(g_arena);
    void *ws = b; b += ws_bytes;
    double *dx = reinterpret_cast<double *>(b); b += n3;
    double *dv = reinterpret_cast<double *>(b); b += n3;
    double *dacc = reinterpret_cast<double *>(b); b += n3;
    double *dm = reinterpret_cast<double *>(b); b += n1;
    double *drc = reinterpret_cast<double *>(b); b += n1;
    int32_t *dpairs = pairs ? reinterpret_cast<int32_t *>(b) : nullptr; b += pb;
    int64_t *dnp = reinterpret_cast<int64_t *>(b);

    const nb_config saved = g_cfg;
    g_cfg.workspace = ws;
    g_cfg.workspace_bytes = ws_bytes;
    cudaStream_t s = stream();
    const size_t b3 = (size_t)N * 3 * sizeof(double), b1 = (size_t)N * sizeof(double);
    auto body = [&]() -> int {
        NB_CUDA(cudaMemcpyAsync(dx, x, b3, cudaMemcpyHostToDevice, s));
        NB_CUDA(cudaMemcpyAsync(dv, v, b3, cudaMemcpyHostToDevice, s));
        NB_CUDA(cudaMemcpyAsync(dm, m, b1, cudaMemcpyHostToDevice, s));
        if (rcrit) NB_CUDA(cudaMemcpyAsync(drc, rcrit, b1, cudaMemcpyHostToDevice, s));
        if (is_step && g_cfg.reuse_acc) NB_CUDA(cudaMemcpyAsync(dacc, acc, b3, cudaMemcpyHostToDevice, s));  // cached force
        int r;
        if (is_step) r = step_impl(dx, dv, dm, M_star, N, dt, rcrit ? drc : nullptr, dacc, dpairs, pairs ? dnp : nullptr, nsteps);
        else r = kick_impl(dx, dv, dm, M_star, N, dt, rcrit ? drc : nullptr, dacc, dpairs, pairs ? dnp : nullptr);
        if (r) return r;
        if (is_step) NB_CUDA(cudaMemcpyAsync(x, dx, b3, cudaMemcpyDeviceToHost, s));
        NB_CUDA(cudaMemcpyAsync(v, dv, b3, cudaMemcpyDeviceToHost, s));
        NB_CUDA(cudaMemcpyAsync(acc, dacc, b3, cudaMemcpyDeviceToHost, s));
        if (rcrit && rcrit_out) NB_CUDA(cudaMemcpyAsync(rcrit, drc, b1, cudaMemcpyDeviceToHost, s));
        if (pairs) {
            NB_CUDA(cudaMemcpyAsync(npairs, dnp, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
            NB_CUDA(cudaStreamSynchronize(s));
            int64_t keep = *npairs < g_cfg.pair_capacity ? *npairs : g_cfg.pair_capacity;
            if (keep > 0) NB_CUDA(cudaMemcpyAsync(pairs, dpairs, (size_t)keep * 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        }
        NB_CUDA(cudaStreamSynchronize(s));
        return NB_OK;
    };
    rc = body();
    // the arena is private: restore the caller's workspace, keep everything else
    g_cfg.workspace = saved.workspace;
    g_cfg.workspace_bytes = saved.workspace_bytes;
    return rc;
}

int nb_kick_host(const double *x, double *v, const double *m, double M_star, int64_t N, double dt, const double *rcrit,
                 double *acc, int32_t *pairs, int64_t *npairs) {
    std::lock_guard<std::mutex> lk(g_mu);
    return host_run(false, const_cast<double *>(x), v, m, M_star, N, dt, const_cast<double *>(rcrit), false, acc, pairs,
                    npairs, 0);
}

int nb_step_host(double *x, double *v, const double *m, double M_star, int64_t N, double dt, double *rcrit, double *acc,
                 int32_t *pairs, int64_t *npairs, int64_t nsteps) {
    std::lock_guard<std::mutex> lk(g_mu);
    return host_run(true, x, v, m, M_star, N, dt, rcrit, true, acc, pairs, npairs, nsteps);
}

int nb_status(int64_t *flags) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!flags) return fail(NB_E_NULL, "flags is NULL");
    if (!g_cfg.workspace && !g_arena) return fail(NB_E_WORKSPACE, "no workspace configured");
    int64_t a[ST_COUNT] = {0}, b[ST_COUNT] = {0};
    if (g_cfg.workspace) NB_CUDA(cudaMemcpyAsync(a, g_cfg.workspace, sizeof(a), cudaMemcpyDeviceToHost, stream()));
    if (g_arena) NB_CUDA(cudaMemcpyAsync(b, g_arena, sizeof(b), cudaMemcpyDeviceToHost, stream()));  // _host calls
    NB_CUDA(cudaStreamSynchronize(stream()));
    for (int k = 0; k < ST_COUNT; ++k) flags[k] = a[k] + b[k];
    return NB_OK;
}

int nb_status_reset(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_cfg.workspace && !g_arena) return fail(NB_E_WORKSPACE, "no workspace configured");
    if (g_cfg.workspace) NB_CUDA(cudaMemsetAsync(g_cfg.workspace, 0, 512, stream()));
    if (g_arena) NB_CUDA(cudaMemsetAsync(g_arena, 0, 512, stream()));
    return NB_OK;
}

double nb_last_force_ms(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_force_timed) return -1.0;
    if (cudaEventSynchronize(g_ev1) != cudaSuccess) return -1.0;
    float ms = -1.0f;
    if (cudaEventElapsedTime(&ms, g_ev0, g_ev1) != cudaSuccess) return -1.0;
    return (double)ms;
}

int nb_force_time(int64_t *launches, double *total_ms) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!launches || !total_ms) return fail(NB_E_NULL, "nb_force_time: NULL argument");
    double tot = 0.0;
    for (int k = 0; k < g_tev_used; ++k) {
        NB_CUDA(cudaEventSynchronize(g_tev[2 * k + 1]));
        float ms = 0.f;
        NB_CUDA(cudaEventElapsedTime(&ms, g_tev[2 * k], g_tev[2 * k + 1]));
        tot += ms;
    }
    *launches = g_tev_used;
    *total_ms = tot;
    return NB_OK;
}

int nb_force_time_reset(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_tev_used = 0;
    return NB_OK;
}

int nb_fp64_peak(int64_t iters, double *tflops, double *ms_out) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!tflops) return fail(NB_E_NULL, "tflops is NULL");
    if (iters <= 0) iters = 4096;
    double *d = nullptr;
    NB_CUDA(cudaMalloc(&d, 512));
    NB_CUDA(cudaMemsetAsync(d, 0, 512, stream()));
    const int ctas = sm_count() * 8, threads = 256;
    cudaEvent_t e0, e1;
    NB_CUDA(cudaEventCreate(&e0));
    NB_CUDA(cudaEventCreate(&e1));
    float ms = 0.f;
    for (int rep = 0; rep < 3; ++rep) {  // first pass doubles as clock warm-up; keep the best
        NB_CUDA(cudaEventRecord(e0, stream()));
        nb_fp64_peak_kernel<<<ctas, threads, 0, stream()>>>(d, iters, d + 32);
        NB_CUDA(cudaEventRecord(e1, stream()));
        NB_CUDA(cudaEventSynchronize(e1));
        float t = 0.f;
        NB_CUDA(cudaEventElapsedTime(&t, e0, e1));
        if (rep == 0 || t < ms) ms = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    const double fmas = (double)ctas * threads * (double)iters * 64.0;
    *tflops = 2.0 * fmas / ((double)ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return NB_OK;
}

void nb_release(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    drop_graph();
    if (g_arena) { cudaFree(g_arena); g_arena = nullptr; g_arena_bytes = 0; }
    if (g_ev0) { cudaEventDestroy(g_ev0); cudaEventDestroy(g_ev1); g_ev0 = g_ev1 = nullptr; }
    for (int k = 0; k < 2 * g_tev_created; ++k) cudaEventDestroy(g_tev[k]);
    g_tev_created = g_tev_used = 0;
    if (g_own_stream) { cudaStreamDestroy(g_own_stream); cudaEventDestroy(g_ev_in); cudaEventDestroy(g_ev_out); g_own_stream = nullptr; }
    g_force_timed = false;
}

const char *nb_last_error(void) { return g_err; }
const char *nb_version(void) { return "nbkick 0.1 (sm_100a)"; }

}  // extern "C"
