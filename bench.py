"""bench.py -- throughput of the whole hot path on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1..C5] [--impl ours|reference]

A "step" is one sph_step (eqs. 52-53): TWO complete right-hand-side evaluations
(Morton order, octree, pseudo-particles, interaction partners, SPH sums, self-gravity; the sub-step
list of PAPER.md:693) and two updates.  metric = particle-updates/s = N * RHS evaluations / time
(SURVEY.md 8(d)).  Prints ONE JSON line (contract in DESIGN.md "Measurement").

  value         device-resident state, CUDA-event time of exactly K steps, max over ranks
  e2e           the same step through the C ABI with HOST buffers: sph_step_host (= sph_upload of the pinned host state
                x v rho u S dmg h n_act + sph_step, the copies on a second stream beside the first evaluation) ->
                sph_download (host state) inside the timed region
  roofline      dominant kernel of the step, timed live by the library's CUDA-event stage brackets
  cpu_baseline  the CPU oracle (oracle/, tree mode, as it stands) on a bounded sample, rank 0, N=1: on all host
                cores and (value_1core) on one core, the paper's own comparison
  workloads     the other BASELINE.json configs (C1-C4) measured in the same process: value, ms per step,
                dominant stage and its roofline fraction
  config.ms_per_step_twin   the headline workload again on its parity twin state (same geometry, perturbed
                state: the viscosity branch and the principal-stress iteration of the pair kernel run)
  --impl reference   the oracle alone, same metric/config (there is no upstream code: PAPER.md only)

Multi-GPU (--gpus N under torchrun): ONE workload sharded by Morton ranges over the N GPUs (DESIGN.md section 9:
replicated cheap stages, partner search / pair sums / walk on the rank's slice, one NCCL all-gather of the rate
arrays per evaluation), strong scaling; value = particles * evaluations / max over ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import sph_inputs  # noqa: E402

METRIC = "particle-updates/s (full FP64 SPH RHS incl. tree gravity); % FP64/HBM roofline"
UNIT = "particle-updates/s"
DEFAULT_WORKLOAD = "C5"
L2_BYTES = 126 << 20
# algorithmic FP64 flop per unit (add = mul = cmp = 1, fma = 2, div = sqrt = 1)
FLOP_PER_INTERACTION = 20.0     # eq. 51 per ACCEPTED pseudo-particle or particle: 3 sub, 5 for r^2, +eps^2, rsqrt, cube (2),
                                # G*M, 3 fma (6) -- the distance of an accepted cell is in here, not in the test
FLOP_PER_OPENED_CELL = 9.0      # eq. 50 for a cell that is OPENED: 3 sub, 5 for r^2, compare (no force follows)
FLOP_PER_VISIT_SURVEY = 3.0     # SURVEY.md 8(d) as written: "20 flop x I_a + 3 x visited nodes" (reported beside it)
FLOP_PER_PAIR = {(3, True): 130.0, (2, True): 80.0, (3, False): 60.0, (2, False): 45.0}


def _peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) for HBM; FP64 is measured live."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.gpu)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.t = threading.Thread(target=self._read, daemon=True)
        self.t.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except ValueError:
                continue
            for k, name in enumerate(names):
                if r[5 + k].lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# algorithmic work per stage
# ---------------------------------------------------------------------------------------------
def stage_work(stage, w, counters, evals):
    """(bound, unit, amount per evaluation) of one stage: algorithmic bytes or flops, NOT traffic."""
    n, D = w.n, w.dim
    solid = bool(w.flags & sph_inputs.F_SOLID)
    damage = bool(w.flags & sph_inputs.F_DAMAGE)
    nstate = 2 * D + 4 + (6 if solid else 0) + (1 if damage else 0)      # doubles moved by the reorder
    passes = (D * 21 + 7) // 8
    if stage == "gravity":
        return "alu", "TFLOP/s", FLOP_PER_INTERACTION * counters["n_inter"] + FLOP_PER_OPENED_CELL * counters["n_open"]
    if stage == "pairs":
        return "alu", "TFLOP/s", FLOP_PER_PAIR[(D, solid)] * counters["n_pairs"]
    if stage == "density":
        return "alu", "TFLOP/s", 30.0 * counters["n_pairs"]
    by = {"keys": 8 * D * 2 + 12,                       # bbox read + key pass read, key + index written
          "sort": passes * 24,                          # (key, index) read + written per 8-bit pass
          "reorder": nstate * 16 + 12,                  # every state array read + written, perm + mat
          "tree": 8 + counters["n_nodes"] / max(n, 1) * (12 + 4 * (2 * (1 << D) + 1) + 24),
          "moments": counters["n_nodes"] / max(n, 1) * (8 * (4 + 2 * D + 1) + 4 * (2 * (1 << D) + 1)) + 8 * (D + 2),
          "neighbours": 4 * counters["n_pairs"] / max(n, 1) + 8 * (D + 1) + 4,
          "prepass": 8 * (3 + (6 if solid else 0) + (1 if damage else 0)) + 4 + 8 * 9,
          "update": 3 * 8 * 15}[stage]
    return "hbm", "GB/s", float(by) * n


def measure_workload(P, torch, name, args, rank, world, dev, full):
    """Times one workload on this rank's GPU.  Region A: exactly args.steps steps as the library runs them (sph_step
    replays its CUDA graph), CUDA events on the library's stream.  Region B: the same steps with the library's
    per-stage CUDA-event brackets (plain launches).  full: also the twin-state timing and the end-to-end arm."""
    t_gen = time.time()
    w = sph_inputs.make(name, scale=args.scale, seed=sph_inputs_seed(name))     # the same particles on every rank
    t_gen = time.time() - t_gen
    cfg, mats = P.config_of(w)
    stream = torch.cuda.Stream(device=dev)     # a stream of our own: sph_step may capture it into a CUDA graph
    torch.cuda.set_stream(stream)              # torch's events, fills and copies below go to the same stream
    ctx = P.sph_create(cfg, mats, device=dev, stream=stream)
    ctx.upload_workload(w)
    if world > 1:                              # Morton-range sharding: this rank's slice, all-gather through NCCL
        ctx.set_partition(rank, world)
    lo, hi, _ = P.sph_partition(w.n, world, rank)
    ws_bytes = ctx.workspace_bytes
    small = ws_bytes < 4 * L2_BYTES       # working set may sit in the 126 MB L2: flush between steps
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev) if small else None

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            torch.distributed.barrier()

    def timed_steps():
        """exactly args.steps steps, CUDA events on the library's stream; returns device ms"""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        barrier()
        for k in range(args.steps):
            if flush is not None:
                flush.fill_(k & 1)
            ev[k][0].record(stream)
            ctx.step(w.dt)
            ev[k][1].record(stream)
        barrier()
        ctx.sync()
        if flush is not None:
            return sum(a.elapsed_time(b) for a, b in ev)
        return ev[0][0].elapsed_time(ev[-1][1])

    # ---- device-resident arm ----
    for _ in range(args.warmup):
        ctx.step(w.dt)                       # the second step with the same dt captures the step graph
    ctx.sync()
    launches0 = ctx.launch_count()
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", rank)))
    sampler.start()
    ms_dev = timed_steps()
    clocks = sampler.stop()
    launches = ctx.launch_count() - launches0
    snap = ctx.download(P.STATE_FIELDS, device=True)      # the state region B starts from (device copy, untimed)
    ctx.timing_enable(True)                  # region B: stage brackets around the kernels of the timed region
    ctx.timing_read()
    ms_bracketed = timed_steps()
    stages = ctx.timing_read()
    ctx.timing_enable(False)
    # the algorithmic units of the rooflines, on the SAME states as the bracketed region: back to the snapshot, the same K
    # steps once more, untimed, with the walk's work counters on (the counting variant of the walk is 15 % slower and is
    # not the kernel the brackets time); the counters of a step are those of its second evaluation, averaged over the steps
    ctx.upload(device=True, **snap)
    ctx.counters_enable(True)
    per_step = []
    for _ in range(args.steps):
        ctx.step(w.dt)
        per_step.append(ctx.get_counters())
    ctx.counters_enable(False)
    counters = {k: int(round(sum(c[k] for c in per_step) / len(per_step))) for k in per_step[0]}
    del snap
    out = dict(w=w, ms_dev=ms_dev, ms_bracketed=ms_bracketed, launches=launches, stages=stages, counters=counters,
               clocks=clocks, l2_flush=small, ws_bytes=ws_bytes, t_gen=t_gen, n_own=hi - lo)
    if not full:
        ctx.close()
        return out

    # ---- the same geometry on its parity twin state: the data-dependent paths of the pair kernel run ----
    wt = sph_inputs.twin_of(w, seed=sph_inputs_seed(name) + 100)
    ctx.upload_workload(wt)
    for _ in range(args.warmup):
        ctx.step(w.dt)
    ctx.sync()
    out["ms_twin"] = timed_steps()
    ctx.timing_enable(True)
    ctx.timing_read()
    timed_steps()
    out["stages_twin"] = ctx.timing_read()
    ctx.timing_enable(False)
    ctx.upload_workload(w)

    # ---- end-to-end arm: host buffers through the C ABI every step ----
    e2e_steps = max(1, args.steps)                          # the same K as the device-resident arm
    n = w.n
    pin = lambda shape, dt: torch.empty(shape, dtype=dt, pin_memory=True)
    host = dict(x=pin((3, n), torch.float64), v=pin((3, n), torch.float64), rho=pin((n,), torch.float64),
                u=pin((n,), torch.float64), S=pin((6, n), torch.float64), dmg=pin((n,), torch.float64),
                h=pin((n,), torch.float64), n_act=pin((n,), torch.int32))
    ctx.download(tuple(host), out=host)                     # current state -> host (untimed)
    # the step's input is the STATE (x v rho u S dmg h n_act); masses, material indices and the flaw table are
    # parameters of the run, uploaded once with the workload (sph_upload leaves NULL members unchanged)
    h2d = sum(t.numel() * t.element_size() for t in host.values())
    d2h = sum(t.numel() * t.element_size() for t in host.values())
    if w.dim == 2:
        h2d -= 2 * n * 8                                    # z rows of x and v are not copied in 2-D

    def e2e_step():
        ctx.step_host(w.dt, **host)                         # sph_step_host: upload + step, the copies beside the first evaluation
        ctx.download(tuple(host), out=host)                 # synchronises (host destination)

    e2e_step()                                              # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    out.update(ms_e2e=(time.perf_counter() - t0) * 1e3 / e2e_steps, h2d=h2d, d2h=d2h)
    ctx.close()
    return out


def stage_tables(r, evals, fp64_peak, hbm_peak):
    """per-stage times, shares and rooflines of one measured workload (region B)"""
    w = r["w"]
    tot_ms = sum(v[0] for v in r["stages"].values()) or 1.0
    stages, roofs = {}, {}
    for name, (ms, ln) in r["stages"].items():
        if ln == 0:
            continue
        bound, unit, amount = stage_work(name, w, r["counters"], evals)
        avg_ms = ms / evals
        ach = amount / (avg_ms * 1e-3) * (1e-12 if bound == "alu" else 1e-9)
        peak = fp64_peak if bound == "alu" else hbm_peak
        stages[name] = {"ms_per_eval": round(avg_ms, 4), "share": round(ms / tot_ms, 4), "launches_per_eval": ln / evals}
        roofs[name] = {"bound": bound, "achieved": round(ach, 3), "peak": round(peak, 2), "unit": unit,
                       "frac": round(ach / peak, 4)}
    return stages, roofs


def run_ours(args, rank, world):
    import torch
    import paper_1604_03290_b200 as P
    from paper_1604_03290_b200 import build as sph_build

    sph_build.build()                       # fails loudly if nvcc or the sources are missing: no fallback
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", rank))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    r = measure_workload(P, torch, args.workload, args, rank, world, dev, full=True)
    r["others"] = {}
    if world == 1 and not args.no_other_workloads and args.workload == DEFAULT_WORKLOAD and args.scale == 1.0:
        for name in ("C1", "C2", "C3", "C4"):      # north_star: "throughput on the five synthetic workloads"
            torch.cuda.empty_cache()
            r["others"][name] = measure_workload(P, torch, name, args, rank, world, dev, full=False)
    r["fp64_peak"] = P.sph_measure_fp64_peak()
    r["copy_gbs"] = P.sph_measure_copy_bw(1 << 30)
    return r


def sph_inputs_seed(name):
    return {"C1": 1604, "C1x": 1604, "C2": 1605, "C3": 1606, "C4": 1607, "C5": 1608, "C6": 1609}[name]


# ---------------------------------------------------------------------------------------------
# CPU oracle arm (test infrastructure timed as a baseline; never on the product path)
# ---------------------------------------------------------------------------------------------
def oracle_time(w, budget_s=20.0):
    """Time the oracle (tree mode, as it stands, OpenMP on the host cores) on one complete RHS
    evaluation of workload `w`.  Small workloads are evaluated whole.  Large ones on a bounded
    sample: the evaluation is run for M1 and M2 target particles (the tree and the per-particle
    pre-pass always cover all N particles), and  T(N) = T_fixed + N * t_per  is formed from the two.
    Returns (seconds per complete evaluation, description of the sample, details dict)."""
    from oracle import oracle as orc
    n = w.n
    orc.lib()
    if n <= 100_000:
        t0 = time.perf_counter()
        orc.evaluate(w, mode="tree")
        t = time.perf_counter() - t0
        return t, f"one complete RHS evaluation of all {n} particles (oracle tree mode)", \
            {"extrapolated": False, "measured_s": round(t, 3), "n_particles": n}
    rng = np.random.default_rng(12345)
    m1 = 2000
    t1s = np.sort(rng.choice(n, m1, replace=False))
    t0 = time.perf_counter()
    orc.evaluate(w, mode="tree", targets=t1s)
    T1 = time.perf_counter() - t0
    # choose M2 so that the second run takes about the budget
    m2 = int(min(n // 2, max(4 * m1, m1 * budget_s / max(T1 * 0.2, 1e-3))))
    t2s = np.sort(rng.choice(n, m2, replace=False))
    t0 = time.perf_counter()
    orc.evaluate(w, mode="tree", targets=t2s)
    T2 = time.perf_counter() - t0
    if T2 - T1 < budget_s / 3.0 and m2 < n // 2:       # the first guess was too small: one larger sample
        m2 = int(min(n // 2, m2 * budget_s / max(T2 - T1, 1e-3)))
        t2s = np.sort(rng.choice(n, m2, replace=False))
        t0 = time.perf_counter()
        orc.evaluate(w, mode="tree", targets=t2s)
        T2 = time.perf_counter() - t0
    per = max((T2 - T1) / (m2 - m1), 1e-12)
    fixed = max(T1 - per * m1, 0.0)
    desc = (f"rates of {m2} random target particles of the full {n}-particle workload "
            f"({T2:.1f} s) and of {m1} ({T1:.1f} s); tree, order and pre-pass over all "
            f"particles both times; T(N) = {fixed:.2f} s + N * {per * 1e6:.2f} us")
    return fixed + per * n, desc, {"extrapolated": True, "measured_s": [round(T1, 3), round(T2, 3)],
                                   "measured_targets": [m1, m2], "n_particles": n}


def oracle_time_one_core(name, scale, budget_s=8.0):
    """The same measurement on ONE host core (the paper compares its GPU code with one CPU core: PAPER.md:687,
    :705), in a child process started with OMP_NUM_THREADS=1, on a 1/8-size instance of the workload where the full
    one would take more than ~10 minutes.  Returns a dict or None."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    cmd = [sys.executable, os.path.abspath(__file__), "--impl", "oracle-probe", "--workload", name, "--scale", str(scale),
           "--oracle-budget", str(budget_s)]
    try:
        out = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception as e:                                   # the baseline is context: never fail the bench line for it
        return {"error": repr(e)[:200]}


def host_cores():
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def config_of_workload(w, args, extra=None):
    c = {"workload": w.name, "n_particles": w.n, "dim": w.dim, "rhs_evaluations_per_step": 2, "dt": w.dt,
         "flags": int(w.flags), "scale": args.scale}
    if extra:
        c.update(extra)
    return c


def run_reference(args, rank, world):
    """--impl reference: there is no upstream code (the reference is PAPER.md); the reference arm is the CPU oracle,
    timed as it stands on the host cores.  Every one of the W + K steps really runs: a step is a bounded sample of
    the workload (one complete evaluation for small workloads; for large ones the evaluation of two target subsets,
    from which the time of a complete evaluation is formed), sized so that the whole run ends within a few minutes.
    `ms_per_step` is the MEASURED wall time of such a step (it agrees with the driver's clock around the run);
    `value` is the throughput a complete step would have, extrapolated from the samples (`cpu_baseline.extrapolated`,
    `ms_per_full_step_extrapolated`)."""
    if rank != 0:
        return None
    w = sph_inputs.make(args.workload, scale=args.scale)
    per_step_budget = max(1.0, min(8.0, 150.0 / max(args.warmup + args.steps, 1)))
    full, wall = [], []
    sample, det = "", {}
    for k in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        t_eval, sample, det = oracle_time(w, budget_s=0.5 * per_step_budget)
        dt = time.perf_counter() - t0
        if k >= args.warmup:
            full.append(2.0 * t_eval)                 # a step is two evaluations
            wall.append(dt)
    T = float(np.mean(full))
    value = 2.0 * w.n / T
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(wall)) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of_workload(w, args, {"ms_per_full_step_extrapolated": T * 1e3,
                                                   "step": "bounded sample of the workload (see cpu_baseline.sample); "
                                                           "ms_per_step is its measured wall time"}),
            "cpu_baseline": dict({"value": value, "unit": UNIT, "cores": host_cores(), "kind": "oracle", "sample": sample}, **det),
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    return line


def make_reducers(world, device):
    """(max, sum) over ranks of one float through torch.distributed (identity for world == 1)."""
    if world == 1:
        return float, float
    import torch

    def reduce(x, op):
        t = torch.tensor([float(x)], dtype=torch.float64, device=device)
        torch.distributed.all_reduce(t, op=op)
        return float(t.item())

    return (lambda x: reduce(x, torch.distributed.ReduceOp.MAX)), (lambda x: reduce(x, torch.distributed.ReduceOp.SUM))


def aggregate(ms_local, n_local, world, reduce_max, reduce_sum):
    """Whole-job value from per-rank numbers: units all ranks processed / max over ranks of the time."""
    ms = reduce_max(ms_local)
    total = reduce_sum(n_local)
    return ms, total


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "oracle-probe"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=list(sph_inputs.CONFIGS))
    ap.add_argument("--scale", type=float, default=1.0, help="< 1: smaller instance of the same workload (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-workloads", action="store_true", help="skip the C1-C4 lines of the default run")
    ap.add_argument("--oracle-budget", type=float, default=8.0, help=argparse.SUPPRESS)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))

    if args.impl == "oracle-probe":          # child of oracle_time_one_core: one timing, threads from the environment
        w = sph_inputs.make(args.workload, scale=args.scale)
        t_eval, sample, det = oracle_time(w, budget_s=args.oracle_budget)
        print(json.dumps(dict({"value": w.n / t_eval, "unit": UNIT, "cores": host_cores(), "sample": sample,
                               "scale": args.scale}, **det)), flush=True)
        return 0
    if args.impl == "reference":
        line = run_reference(args, rank, world)
        if line is not None:
            print(json.dumps(line), flush=True)
        return 0

    import torch
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.distributed.init_process_group("nccl")

    r = run_ours(args, rank, world)
    w = r["w"]
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", rank)))

    rmax, rsum = make_reducers(world, dev)
    # every rank contributes the particles of its own slice: the sum is the workload, the time is the slowest rank's
    ms_dev, n_total = aggregate(r["ms_dev"], r["n_own"], world, rmax, rsum)
    ms_e2e, _ = aggregate(r["ms_e2e"], r["n_own"], world, rmax, rsum)
    ms_twin, _ = aggregate(r["ms_twin"], r["n_own"], world, rmax, rsum)
    launches = int(rsum(r["launches"]))
    if rank != 0:
        torch.distributed.destroy_process_group()
        return 0

    evals = 2 * args.steps
    value = n_total * evals / (ms_dev * 1e-3)
    e2e_value = n_total * 2 / (ms_e2e * 1e-3)
    hbm_peak, hbm_src = _peaks()

    # per-stage table and rooflines (rank 0's replica)
    stages, roofs = stage_tables(r, evals, r["fp64_peak"], hbm_peak)
    top = max(stages, key=lambda k: stages[k]["share"])
    roofline = dict(roofs[top])
    roofline.update({"kernel": top, "traffic": traffic_of(args.workload, top),
                     "traffic_source": "profiles/traffic.json (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch)",
                     "peak_source": ("FP64 FMA micro-benchmark measured in this run (sph_measure_fp64_peak); nominal "
                                     "148 SM x 64 lanes x 2 x 1.965 GHz = 37.2 TFLOP/s") if roofline["bound"] == "alu"
                     else hbm_src})
    if top == "gravity":
        c = r["counters"]
        t_s = stages[top]["ms_per_eval"] * 1e-3
        roofline["accounting"] = ("20 flop per accepted interaction (eq. 51) + 9 per OPENED cell (eq. 50); the distance of an "
                                  "accepted cell is counted once, inside the 20")
        roofline["frac_survey_8d"] = round((FLOP_PER_INTERACTION * c["n_inter"] + FLOP_PER_VISIT_SURVEY * c["n_visit"])
                                           / t_s * 1e-12 / r["fp64_peak"], 4)      # "20 x I + 3 x visited nodes" as written
    # the twin state of the same geometry (stage shares of its bracketed run)
    twin_stages = {k: round(v[0] / evals, 4) for k, v in r["stages_twin"].items() if v[1]}

    others = {}
    for name, ro in r["others"].items():
        st_o, rf_o = stage_tables(ro, evals, r["fp64_peak"], hbm_peak)
        top_o = max(st_o, key=lambda k: st_o[k]["share"])
        wo = ro["w"]
        others[name] = {"workload": wo.name, "n_particles": wo.n, "value": wo.n * evals / (ro["ms_dev"] * 1e-3), "unit": UNIT,
                        "ms_per_step": ro["ms_dev"] / args.steps, "ms_per_step_bracketed": ro["ms_bracketed"] / args.steps,
                        "gpu_launches": ro["launches"], "dominant_stage": top_o, "dominant_ms_per_eval": st_o[top_o]["ms_per_eval"],
                        "dominant_share": st_o[top_o]["share"], "roofline": rf_o[top_o],
                        "l2": "L2 flushed between timed steps" if ro["l2_flush"] else "working set larger than L2",
                        "clocks": ro["clocks"], "stages_ms_per_eval": {k: v["ms_per_eval"] for k, v in st_o.items()}}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_dev / args.steps, "higher_is_better": True,
            "scaling": "weak" if world == 1 else "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of_workload(w, args, {
                "parallelism": "single GPU" if world == 1 else
                               f"one workload sharded by Morton ranges over {world} GPUs: tree build replicated, partner search / "
                               f"pair sums / gravity walk on the rank's slice, one NCCL all-gather of the rates per evaluation; "
                               f"stages, roofline and counters below are rank 0's slice",
                "l2": "L2 flushed (252 MB write) between timed steps" if r["l2_flush"]
                      else "working set larger than L2 (%.1f GB workspace)" % (r["ws_bytes"] / 1e9),
                "particle_steps_per_s": n_total * args.steps / (ms_dev * 1e-3),
                "timing": "value: K steps as the library runs them (sph_step replays its CUDA graph), CUDA events; "
                          "stages/roofline: the same K steps again with per-stage CUDA-event brackets (plain launches)",
                "ms_per_step_bracketed": r["ms_bracketed"] / args.steps,
                "ms_per_step_twin": ms_twin / args.steps,
                "twin": "same geometry and flaws, perturbed state (sph_inputs.twin_of): every branch of the rate equations "
                        "runs on every particle; value/ms_per_step above are the nominal t = 0 state of BASELINE.json",
                "twin_stages_ms_per_eval": twin_stages,
                "hbm_copy_gbs_this_run": round(r["copy_gbs"], 1),
                "counters_per_eval": r["counters"]}),
            "clocks": r["clocks"],
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(r["h2d"]),
                    "d2h_bytes_per_step": int(r["d2h"]), "ms_per_step": ms_e2e},
            "gpu_launches": launches,
            "roofline": roofline, "stages": stages, "rooflines_all": roofs}
    if others:
        line["workloads"] = others
    if world == 1 and not args.no_cpu_baseline:
        t_eval, sample, det = oracle_time(w)
        cb = dict({"value": w.n / t_eval, "unit": UNIT, "cores": host_cores(), "kind": "oracle", "sample": sample}, **det)
        # one core, the paper's comparison: on a 1/8-size instance (labelled) when generating and evaluating the full
        # one on a single core would not fit the few minutes of a default run
        sc1 = args.scale if w.n * 60e-6 < 60.0 else args.scale / 8.0     # ~60 us per particle and core
        one = oracle_time_one_core(args.workload, sc1)
        if one and "value" in one:
            cb["value_1core"] = one["value"]
            cb["one_core"] = {k: one[k] for k in ("sample", "scale", "extrapolated", "measured_s", "n_particles") if k in one}
        elif one:
            cb["one_core"] = one
        line["cpu_baseline"] = cb
    print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


# dram__bytes_read.sum + dram__bytes_write.sum per launch of a stage's kernel: profiles/traffic.json, written from the
# committed `ncu --set full` capture of the same kernels (the file names the capture); None = not captured.
def traffic_of(workload, stage):
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
        e = t["kernels"].get(workload, {}).get(stage)
        return None if e is None else float(e["dram_bytes_read"]) + float(e["dram_bytes_write"])
    except (OSError, ValueError, KeyError):
        return None


if __name__ == "__main__":
    sys.exit(main())
