#!/usr/bin/env python
"""bench.py -- whole hot path (one nb_step = rcrit + O(N^2) kick tiles + pair list + H_C shifts + Kepler
drift) on the synthetic N = 65536 ring of BASELINE.json:configs[2], the configuration the metric
("fp64 pairwise interactions/sec ...; steps/sec at N=65536") is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference] [--config k]

Prints ONE JSON line (rank 0).  `value` = ordered (i,j) interactions evaluated per second by all ranks,
inputs resident in HBM; `e2e` = the same through the host-buffer C-ABI call (nb_step_host) with the
host<->device copies inside the timed region; `roofline` = the force-tile kernel against the B200 fp64
FMA peak (bound "alu"); `cpu_baseline` = the CPU oracle timed beside it on a bounded sample.
--impl reference times the CPU oracle alone (test infrastructure; the one other place that runs it).
The path does not shard (BASELINE.json:north_star: one GPU, no collectives): --gpus N runs N
independent replicas ("replicas only"), one process per GPU, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import nb_inputs  # noqa: E402  (seeded input generators only; none of the method's arithmetic)
from nb_inputs import G_GAUSS  # noqa: E402

METRIC = "fp64_pairwise_interactions_per_sec"
UNIT = "interactions/s"
FLOPS_PER_INTERACTION = 20.0  # BASELINE.json:north_star "about 20 flops counted per interaction"
# fp64 FMA peak of a B200 from unit counts and clocks: 148 SMs x 64 fp64 lanes
# x 2 flop x 1.965 GHz (clocks.max.sm)
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
N1, N2 = 3.0, 0.0  # headline radius: 3 Hill radii (BASELINE.json:configs[0]; S7)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json:configs (default 2: N=65536)")
    ap.add_argument("--n", type=int, default=None, help="override the body count (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-drift-point", action="store_true", help="skip the N = 2^24 drift-only HBM point")
    ap.add_argument("--no-mixed-point", action="store_true", help="skip the mixed-precision side line (fully active configs)")
    ap.add_argument("--force-kernel", type=int, default=0, choices=[0, 1, 2],
                    help="nb_config.force_kernel: 0 auto, 1 one-sided tiles, 2 Newton-III (comparison runs)")
    ap.add_argument("--i-per-thread", type=int, default=0, choices=[0, 1, 2, 4], help="nb_config.i_per_thread: 0 auto (comparison runs)")
    ap.add_argument("--j-splits", type=int, default=0,
                    help="nb_config.j_splits: 0 auto, k > 0 a grid of k j-splits, -1 balanced pieces (comparison runs, one-sided kernel)")
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="f64 (default, the metric) or the mixed-precision kick variant (NB_PRECISION_MIXED; a side line)")
    ap.add_argument("--trajectory", action="store_true",
                    help="instead of the step benchmark: the config's own trajectory (all its steps) as ONE nb_step call "
                         "(CUDA-graph replay / fused small-N launch), timed with CUDA events; prints one JSON line with mode=trajectory")
    ap.add_argument("--n2", type=float, default=None, help="--trajectory: velocity factor of Eq. 7 (default 0: 3 R_Hill; 0.4: full Eq. 7)")
    ap.add_argument("--encounters", action="store_true", help="--trajectory: resolve close encounters (direct solver)")
    ap.add_argument("--collide", type=float, default=0.0,
                    help="--trajectory --encounters: examine collisions inside the direct solver with the radii (2 g/cm^3) inflated by this factor (PAPER.md:98, 130, 168); 0 = off")
    ap.add_argument("--levels", type=int, default=0, help="--trajectory --encounters: intermediate changeover levels (PAPER.md:106)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 100 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = f"/tmp/nb_clocks_{os.getpid()}.csv"

    def start(self):
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = dict(sm_mhz=None, sm_max_mhz=None, power_w_max=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [t.strip() for t in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
                except ValueError:
                    continue
                for nm, val in zip(names, f[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            os.remove(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def workload(args):
    d = nb_inputs.make_config(args.config, n_override=args.n)
    na = d.n_active if d.n_active < d.N else 0
    return d, na


def workload_name(d, na):
    return (f"{d.name}: N={d.N}" + (f" (n_active={na})" if na else "") +
            f", dt={d.dt:g} d, rcrit = {N1:g} R_Hill (n2={N2:g}), seed {d.seed}, synthetic disk (DESIGN.md input recipe)")


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (test infrastructure, timed as it stands; never tuned for this)
# ------------------------------------------------------------------------------------------------
def oracle_sample_step(d, na, rows, state):
    """One pass of the hot path by the oracle with the O(N^2) parts restricted to `rows` i-bodies
    (all j): rcrit, accelerations + pairs of the sampled rows, half-kicks, H_C shifts, Kepler drift.
    Returns (seconds, interactions evaluated)."""
    import oracle
    x, v = state
    t0 = time.perf_counter()
    rc = oracle.rcrit(x, v, d.m, d.M_star, d.dt, G_GAUSS, N1, N2)
    acc, _, _ = oracle.accel(x, d.m, rc, G_GAUSS, n_active=na, rows=rows)
    oracle.pairs(x, rc, n_active=na, rows=rows)
    v = v.copy()
    v[rows] = v[rows] + (0.5 * d.dt) * acc
    x = oracle.shift(x, v, d.m, d.M_star, 0.5 * d.dt)
    x, v, _ = oracle.drift_kepler(x, v, d.M_star, d.dt, G_GAUSS)
    x = oracle.shift(x, v, d.m, d.M_star, 0.5 * d.dt)
    dt = time.perf_counter() - t0
    state[0], state[1] = x, v
    return dt, rows.size * (na or d.N)


def cpu_baseline(d, na, budget_s=12.0):
    import oracle
    rng = np.random.default_rng(77)
    state = [d.x.copy(), d.v.copy()]
    probe = np.sort(rng.choice(d.N, size=min(2048, d.N), replace=False))  # large enough that thread start-up does not bias the rate
    t, n = oracle_sample_step(d, na, probe, state)
    rate = n / t
    R = int(min(d.N, max(256, budget_s * rate / (na or d.N))))
    rows = np.sort(rng.choice(d.N, size=R, replace=False))
    t, n = oracle_sample_step(d, na, rows, state)
    return dict(value=n / t, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                note="extended-precision checker (x87 long double sums), not a tuned CPU kernel",
                sample=f"one oracle step with the O(N^2) kick + pair test on {R} seeded-random i-rows x all "
                       f"{na or d.N} j (rcrit, shifts, Kepler drift on all N): {n:.3e} interactions in {t:.2f} s")


def run_reference(args):
    """--impl reference: the CPU oracle as it stands on this box's host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    d, na = workload(args)
    rng = np.random.default_rng(78)
    state = [d.x.copy(), d.v.copy()]
    probe = np.sort(rng.choice(d.N, size=min(128, d.N), replace=False))
    t, n = oracle_sample_step(d, na, probe, state)
    total_steps = args.steps + args.warmup
    budget = 150.0  # seconds for the whole run
    R = int(min(d.N, max(32, budget / total_steps * (n / t) / (na or d.N))))
    rows = np.sort(rng.choice(d.N, size=R, replace=False))
    for _ in range(args.warmup):
        oracle_sample_step(d, na, rows, state)
    tt, nn = 0.0, 0
    for _ in range(args.steps):
        t, n = oracle_sample_step(d, na, rows, state)
        tt += t
        nn += n
    value = nn / tt
    sample = (f"each step: oracle O(N^2) kick + pair test on {R} seeded-random i-rows x all {na or d.N} j, "
              f"O(N) parts on all N; {args.steps} steps, {nn:.3e} interactions in {tt:.2f} s")
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * tt / max(args.steps, 1), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64 (x87 extended accumulators)", data="synthetic",
                config=dict(workload=workload_name(d, na), sample=sample),
                cpu_baseline=dict(value=value, unit=UNIT, cores=oracle.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------------------
def _traffic_from_profile(kernel, N, geom, sorted_staging, precision):
    """(dram bytes per launch, source) from the committed ncu capture (profiles/force_kernel_traffic.json) -- only when the
    launch that ran here has the profiled geometry (kernel, N, S or tile, I, sorted staging, precision); the figure is
    NOT measured in this run (ncu counters cannot be read outside a profiler)."""
    p = os.path.join(ROOT, "profiles", "force_kernel_traffic.json")
    try:
        for e in json.load(open(p))["captures"]:
            if (e["kernel"] == kernel and e["N"] == N and e["tile_j"] == geom.tile_j and e["i_per_thread"] == geom.i_per_thread
                    and e["j_splits"] == geom.j_splits and bool(e["sorted_staging"]) == bool(sorted_staging)
                    and e.get("precision", "f64") == precision):
                return e["dram_bytes_per_launch"], e["source"] + " (ncu capture of the same geometry; not measured in this run)"
    except Exception:
        pass
    return None, "no ncu capture of this geometry under profiles/ (not measured in this run)"


def _extra_band_launches(N, geom, cap=4 << 30):
    """Launches a banded evaluation of the Newton-III kernel adds to a step: 2 per band minus the one force launch already
    counted (the library's rule: slots of the whole grid over nb_config.slot_bytes_max, default 4 GiB)."""
    if geom.tile_j >= 0:
        return 0
    S, T = -geom.tile_j, geom.j_splits
    if 24 * N * T <= cap:
        return 0
    band = max(1, cap // (24 * (N + T * S)))
    return 2 * (-(-T // band)) - 1


def _hbm_peak_gbs():
    """(GB/s, source): the driver-measured copy bandwidth, else the profiling guide's fallback."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json (burst copy)"
    except Exception:
        return 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


def drift_roofline(d, n_bodies=1 << 24, launches=5):
    """HBM point of the Kepler drift (a6): the workload's bodies tiled to n_bodies (x, v: 96 bytes per
    body in and out, 1.6 GB -- far beyond L2), nb_drift_kepler timed alone with CUDA events."""
    import torch
    import paper_2604_09184_b200 as nb
    reps = -(-n_bodies // d.N)
    x = torch.from_numpy(np.tile(d.x, (reps, 1))[:n_bodies].copy()).cuda()
    v = torch.from_numpy(np.tile(d.v, (reps, 1))[:n_bodies].copy()).cuda()
    nb.configure(n_bodies, G=G_GAUSS, workspace_bytes=4096)  # the O(N) calls need only the workspace head
    nb.nb_status_reset()
    for _ in range(2):
        nb.nb_drift_kepler(x, v, d.M_star, d.dt)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(launches):
        nb.nb_drift_kepler(x, v, d.M_star, d.dt)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / launches
    fails = nb.nb_status()["kepler_fail"]
    peak, src = _hbm_peak_gbs()
    gbs = 96.0 * n_bodies / (ms * 1e-3) / 1e9
    del x, v
    return dict(kernel="nb_drift_kernel", bound="hbm", bodies=n_bodies, bytes_per_body=96, avg_launch_ms=ms,
                achieved=gbs, peak=peak, unit="GB/s", frac=gbs / peak, peak_source=src, kepler_fail=fails,
                bodies_per_sec=n_bodies / (ms * 1e-3))


def mixed_point(d, launches=10):
    """Side line (PAPER.md:160 contrasts FP32 and FP64 runs): the same kick in NB_PRECISION_MIXED
    (fully active N >= 4096: Newton-III kernel on double-single positions, FP32 pipe), nb_kick timed alone with CUDA
    events, and its error against the fp64 kernel's accelerations on the same input (reading S25).  Not the metric."""
    import torch
    import paper_2604_09184_b200 as nb
    N = d.N
    x = torch.from_numpy(d.x).cuda(); v = torch.from_numpy(d.v).cuda(); m = torch.from_numpy(d.m).cuda()
    rc = torch.zeros(N, dtype=torch.float64, device="cuda")
    out = {}
    for prec in (0, 1):
        nb.configure(N, G=G_GAUSS, n1=N1, n2=N2, precision=prec)
        nb.nb_rcrit(x, v, m, d.M_star, d.dt, rc)
        acc = torch.zeros_like(x)
        for _ in range(2):
            nb.nb_kick(x, v, m, d.M_star, 0.0, rc, acc)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(launches):
            nb.nb_kick(x, v, m, d.M_star, 0.0, rc, acc)
        e1.record()
        torch.cuda.synchronize()
        out[prec] = (e0.elapsed_time(e1) / launches, acc, nb.force_geometry(N))
    a64, a32 = out[0][1], out[1][1]
    scale = torch.clamp(a64.abs(), min=1e-3 * float(a64.norm(dim=1).max()))
    rel = ((a32 - a64).abs() / scale)
    g = out[1][2]
    return dict(precision="NB_PRECISION_MIXED", kernel="nb_force_symds_kernel" if g.tile_j < 0 else ("nb_force_mixedds_kernel" if g.i_per_thread >= 2 else "nb_force_tiles_kernel (fp64: one i-body per thread)"),
                ms_per_kick=out[1][0], interactions_per_sec=float(N) * float(N) / (out[1][0] * 1e-3),
                ms_per_kick_f64=out[0][0], speedup_vs_f64=out[0][0] / out[1][0],
                rel_err_vs_f64_median=float(rel.median()), rel_err_vs_f64_max=float(rel.max()),
                # 22 FP32 lane-operations per unordered pair (Newton-III kernel; S25 / 8.6) against 148 SM x 128 lanes x clock
                fp32_lane_frac=(22.0 * float(N) * float(N) / 2.0 / (out[1][0] * 1e-3) / (148 * 128 * 1.965e9)) if g.tile_j < 0 else None,
                note="whole nb_kick (staging + force + slot sum), no L2 flush; tolerance reading S25 (DESIGN.md)")


def max_over_ranks(values, device="cuda"):
    """Replicas only: the single cross-rank step of the benchmark is this MAX over the ranks' timings (no
    data-path collective).  Works with any initialised backend (nccl on the GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu().tolist()]


def whole_job_value(world, steps, interactions_per_step, max_total_ms):
    """Whole-job aggregate: every replica does `steps` steps in the slowest rank's time."""
    return world * steps * interactions_per_step / (max_total_ms * 1e-3)


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2604_09184_b200 as nb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl cuda needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    d, na = workload(args)
    N, Nj = d.N, (na or d.N)
    inter_per_step = float(N) * float(Nj)
    cap = 1 << 22
    K, W = args.steps, max(args.warmup, 0)

    # ---- device-resident arm: inputs in HBM before the timed region -------------------------------
    mixed = args.precision == "mixed"
    nb.configure(N, pair_capacity=cap, n_active=na, G=G_GAUSS, n1=N1, n2=N2, reuse_acc=False, time_force=True,
                 force_kernel=args.force_kernel, j_splits=args.j_splits, i_per_thread=args.i_per_thread, precision=1 if mixed else 0)
    nb.nb_status_reset()
    x = torch.from_numpy(d.x).cuda(); v = torch.from_numpy(d.v).cuda(); m = torch.from_numpy(d.m).cuda()
    acc = torch.zeros_like(x); rc = torch.zeros(N, dtype=torch.float64, device="cuda")
    pairs = torch.zeros((cap, 2), dtype=torch.int32, device="cuda")
    npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    geom = nb.force_geometry(N)

    nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 0)  # evaluation at t0 (start-up, untimed)
    nb.set_flags(reuse_acc=1)  # from here on: exactly one force evaluation per step
    for _ in range(W):
        nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 1)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    nb.nb_force_time_reset()
    sampler.start()
    wall0 = time.perf_counter()
    for k in range(K):
        flush.fill_(k & 0xFF)  # L2 flush between timed iterations (outside the per-step events)
        ev[k][0].record()
        nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 1)
        ev[k][1].record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    n_force, force_ms = nb.nb_force_time()
    status = nb.nb_status()
    npairs_last = int(npairs.item())
    peak_tf, _ = nb.nb_fp64_peak(8192)

    # ---- encounter groups of the last step's pair list: reported beside
    # the step, not part of the timed region
    g_label = torch.empty(N, dtype=torch.int32, device="cuda"); g_members = torch.empty(N, dtype=torch.int32, device="cuda")
    g_start = torch.empty(N // 2 + 2, dtype=torch.int32, device="cuda"); g_stat = torch.zeros(4, dtype=torch.int64, device="cuda")
    for _ in range(2):
        nb.nb_groups(pairs, npairs, N, g_label, g_members, g_start, g_stat)
    ge0, ge1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ge0.record()
    for _ in range(10):
        nb.nb_groups(pairs, npairs, N, g_label, g_members, g_start, g_stat)
    ge1.record()
    torch.cuda.synchronize()
    gs = [int(t) for t in g_stat.cpu().tolist()]
    groups_info = dict(call="nb_groups", ms=ge0.elapsed_time(ge1) / 10, launches_per_call=9, pairs=gs[3], groups=gs[0],
                       members=gs[1], largest=gs[2])
    # direct solver of those groups for one dt, on copies of the state
    xe, ve = x.clone(), v.clone()
    nb.nb_encounter(xe, ve, m, rc, d.M_star, d.dt, g_members, g_start, g_stat)
    xe.copy_(x); ve.copy_(v)
    ge0.record()
    nb.nb_encounter(xe, ve, m, rc, d.M_star, d.dt, g_members, g_start, g_stat)
    ge1.record()
    torch.cuda.synchronize()
    st_enc = nb.nb_status()
    groups_info.update(encounter_call="nb_encounter", encounter_ms=ge0.elapsed_time(ge1), bs_tol=1e-12,
                       groups_skipped=st_enc["groups_skipped"], bs_fail=st_enc["bs_fail"])
    del xe, ve

    # ---- end-to-end arm: host buffers through nb_step_host, copies inside the timed region ---------
    e2e = None
    if not args.no_e2e:
        Ke = max(3, min(K, 20))
        nb.set_flags(reuse_acc=0, time_force=0)
        def pinned(shape, dtype):
            # page-locked host buffers (torch only allocates them; the library sees plain host pointers)
            return torch.zeros(shape, dtype=dtype).pin_memory().numpy()
        hx, hv, hm = pinned((N, 3), torch.float64), pinned((N, 3), torch.float64), pinned((N,), torch.float64)
        hx[:] = d.x; hv[:] = d.v; hm[:] = d.m
        hacc, hrc = pinned((N, 3), torch.float64), pinned((N,), torch.float64)
        hpairs, hnp = pinned((cap, 2), torch.int32), pinned((1,), torch.int64)
        nb.nb_step_host(hx, hv, hm, d.M_star, d.dt, hrc, hacc, hpairs, hnp, 0)  # t0 evaluation, result lands on the host
        nb.set_flags(reuse_acc=1)
        for _ in range(min(W, 3)):
            nb.nb_step_host(hx, hv, hm, d.M_star, d.dt, hrc, hacc, hpairs, hnp, 1)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            nb.nb_step_host(hx, hv, hm, d.M_star, d.dt, hrc, hacc, hpairs, hnp, 1)  # synchronises
        barrier()
        te = time.perf_counter() - t0
        h2d = 8 * (3 * N + 3 * N + N + N + 3 * N)            # x, v, m, rcrit, acc (cached force)
        d2h = 8 * (3 * N + 3 * N + 3 * N + N) + 8 + 8 * int(hnp[0])  # x, v, acc, rcrit, npairs, pairs
        e2e = dict(te=te, Ke=Ke, h2d=h2d, d2h=d2h)
        nb.set_flags(reuse_acc=0)

    # ---- max over ranks (replicas: no data-path collective; this is only the timing reduction) -----
    if world > 1:
        red = max_over_ranks([total_ms, e2e["te"] if e2e else 0.0])
        total_ms = red[0]
        if e2e:
            e2e["te"] = red[1]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = whole_job_value(world, K, inter_per_step, total_ms)
    symmetric = geom.tile_j < 0
    kernel = ("nb_force_symds_kernel" if mixed else "nb_force_sym_kernel") if symmetric else ("nb_force_mixedds_kernel" if mixed and geom.i_per_thread >= 2 else "nb_force_tiles_kernel")
    sorted_staging = symmetric and N >= 32768   # NB_SORT_AUTO (include/nbkick.h), both Newton-III kernels
    traffic, traffic_source = _traffic_from_profile(kernel, N, geom, sorted_staging, args.precision)
    # FP64-pipe instructions per ORDERED interaction on the fast path: 20 per unordered pair (Newton III)
    # or 15 (one-sided); DESIGN.md section 5
    pipe_instr = 10.0 if symmetric else 15.0
    force_avg_ms = force_ms / max(n_force, 1)
    achieved_tf = FLOPS_PER_INTERACTION * inter_per_step / (force_avg_ms * 1e-3) / 1e12
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=total_ms / K,
        higher_is_better=True, scaling="weak", vs_baseline=None,
        dtype="f64" if not mixed else "double-single (Newton-III kernel) or f64 differences, f32 pair arithmetic, f64 accumulation (NB_PRECISION_MIXED; not the metric's precision)",
        data="synthetic",
        config=dict(workload=workload_name(d, na), parallelism="replicas only (path does not shard)" if world > 1 else "1 GPU",
                    l2="256 MiB buffer written between timed steps (L2 flush), outside the per-step CUDA events",
                    force_evaluations_per_step=1, interactions_per_step=inter_per_step,
                    geometry=dict(i_per_thread=geom.i_per_thread, i_blocks=geom.i_blocks, j_splits=geom.j_splits,
                                  threads=geom.threads, tile_j=geom.tile_j),
                    pairs_last_step=npairs_last, status=status, wall_s_incl_flush=wall),
        steps_per_sec=world * K / (total_ms * 1e-3),
        roofline=dict(bound="alu", achieved=achieved_tf, peak=FP64_PEAK_NOMINAL_TFLOPS, unit="TFLOP/s",
                      frac=achieved_tf / FP64_PEAK_NOMINAL_TFLOPS, traffic=traffic, traffic_source=traffic_source,
                      kernel=kernel, launches_timed=n_force, avg_launch_ms=force_avg_ms,
                      flops_per_interaction=FLOPS_PER_INTERACTION,
                      peak_source="nominal: 148 SM x 64 fp64 lanes x 2 x 1.965 GHz (DESIGN.md); MEASURED_PEAKS.json has no fp64 entry",
                      peak_measured_dfma=peak_tf, frac_of_measured_dfma=achieved_tf / peak_tf if peak_tf > 0 else None,
                      fp64_pipe_instr_per_interaction=pipe_instr,
                      fp64_pipe_util_est=pipe_instr * inter_per_step / (force_avg_ms * 1e-3) / (peak_tf * 1e12 / 2.0) if peak_tf > 0 else None),
        clocks=clocks,
        # per timed step: opening half-kick, drift, prep, force, slot sum + closing half-kick; with the Newton-III kernel's
        # sorted staging (automatic for N >= 32768) also five sort kernels and the bounds kernel
        # banded evaluation (N beyond ~180 000: DESIGN.md 5.1d): one force launch and one fold per band instead of one launch
        gpu_launches=((11 if sorted_staging else 5) + _extra_band_launches(N, geom)) * K,
        groups=groups_info,
    )
    if e2e:
        line["e2e"] = dict(value=world * e2e["Ke"] * inter_per_step / e2e["te"], unit=UNIT,
                           h2d_bytes_per_step=e2e["h2d"], d2h_bytes_per_step=e2e["d2h"], steps=e2e["Ke"],
                           call="nb_step_host(nsteps=1, reuse_acc=1): pinned host buffers in, results out, stream synchronised")
    if not args.no_drift_point:
        line["drift_roofline"] = drift_roofline(d)
    if not args.no_mixed_point and not mixed and not na:
        line["mixed_precision"] = mixed_point(d)
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(d, na)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_trajectory(args):
    """The config's own trajectory as ONE nb_step call after the evaluation at t0 (what a user of nb_step runs): CUDA events
    around the call.  Energies are not computed here (the O(N^2) diagnostic is test infrastructure: tests/ write them to
    profiles/r2_parity.md); this line carries timing, pair counts and the library's status counters."""
    import torch
    import paper_2604_09184_b200 as nb
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --trajectory needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    d, na = workload(args)
    N = d.N
    n2 = N2 if args.n2 is None else args.n2
    cap = 1 << 24
    collide = args.encounters and args.collide > 0.0
    radius = torch.from_numpy(d.radius).cuda() if collide else None
    absorbed_by = torch.full((N,), -1, dtype=torch.int32, device="cuda") if collide else None
    nb.configure(N, pair_capacity=cap, n_active=na, G=G_GAUSS, n1=N1, n2=n2, resolve_encounters=args.encounters,
                 levels=args.levels, precision=1 if args.precision == "mixed" else 0, force_kernel=args.force_kernel, j_splits=args.j_splits, i_per_thread=args.i_per_thread,
                 radius_factor=args.collide if collide else 1.0, collide_radius=radius, collide_absorbed_by=absorbed_by)
    nb.nb_status_reset()
    x = torch.from_numpy(d.x).cuda(); v = torch.from_numpy(d.v).cuda(); m = torch.from_numpy(d.m).cuda()
    acc = torch.zeros_like(x); rc = torch.zeros(N, dtype=torch.float64, device="cuda")
    pairs = torch.zeros((cap, 2), dtype=torch.int32, device="cuda"); npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    nsteps = args.steps if args.steps != 100 else d.nsteps
    nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 0)
    nb.set_flags(reuse_acc=1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, nsteps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    geom = nb.force_geometry(N)
    print(json.dumps(dict(mode="trajectory", config=workload_name(d, na).replace(f"(n2={N2:g})", f"(n2={n2:g})"), N=N, nsteps=nsteps,
                          a_substep=("direct solver for the encounter groups" + (f", {args.levels} intermediate levels" if args.levels else "") + (f", collisions inside the solver (f = {args.collide:g})" if collide else "")) if args.encounters else "Kepler drift",
                          total_ms=ms, ms_per_step=ms / nsteps, steps_per_sec=nsteps / (ms * 1e-3),
                          interactions_per_sec=nsteps * float(N) * float(na or N) / (ms * 1e-3), pairs_last_step=int(npairs.item()),
                          status=nb.nb_status(), precision=args.precision,
                          geometry=dict(i_per_thread=geom.i_per_thread, i_blocks=geom.i_blocks, j_splits=geom.j_splits, tile_j=geom.tile_j))),
          flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.trajectory:
        run_trajectory(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
