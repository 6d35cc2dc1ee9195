#!/usr/bin/env python
"""bench.py -- the C-PCM hot path on the seeded synthetic workload of BASELINE.json configs[3] (the largest single-GPU
config: 2 000 atoms, s/p/d shells, ~102k surface points), with every other config reported beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-sweep] [--no-cpu] [--no-extras] [--no-configs]

A timed iteration is one pass of the whole hot path on device-resident inputs:
    v = pcm_potential(P)  ||  pcm_rbj_build_async(64) on a side stream  ->  pcm_cg_solve(A q = v, tol 1e-8, RBJ)  ->  F = pcm_fock(q)
with CUDA events between the calls.  BASELINE.json's metric has three clauses and they are reported separately:
  * `ms_per_step` = ms per pcm_potential + pcm_fock call and `value` = primitive-pair x point per second over those two
    calls (2 * prim_pair_points / (potential ms + Fock ms): each call evaluates every surviving primitive pair against
    every surface point).  The solver's time is NOT in this figure; it is in `step` (the whole C-PCM step) and `solver`.
  * `amatvec`: the A q sweep of configs[4] (M = 10k .. 200k) with its fraction of the FP64 peak; `solver`: pcm_cg_solve
    at those sizes, RBJ-64 against Jacobi.
  * `roofline`: the dominant kernel of the headline, `per_config`: configs[0..3], `cpu_baseline`: the oracle on the host
    cores, `e2e`: the same two calls through the host-buffer C ABI.

`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same two calls per step and prints the same
line with "impl": "reference" (ms_per_step = the measured time of that sample).  N > 1: the path does not shard
(north_star: one GPU) -- every rank runs an independent replica ("replicas only"), value = N * units /
max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "prim_pair_point_per_s"
UNIT = "prim-pair*point/s"
CONFIG_INDEX = 3
RBJ_BLOCK = 64
CG_TOL = 1e-8
PERSIST_MAX = 26_000   # points below which the library runs A q / PCG through the persistent sweep (pcm_internal.h AMAT_PERSIST_MAX)
SWEEP_M = (2_500, 10_000, 50_000, 100_000, 200_000)
STORED_M = (2_500, 5_000, 10_000, 50_000)   # stored-A variant against the on-the-fly sweep
SOLVER_M = (2_500, 10_000, 50_000, 200_000)   # configs[4]: full pcm_cg_solve, RBJ-64 against Jacobi
RBJ_SWEEP_M, RBJ_SWEEP_BLOCKS = 50000, (8, 32, 100, 256, 800)   # block-size study of PAPER.md:192-196 at one size

WORKLOADS = {
    0: "configs[0]: 12-atom chain, 6-31G-shaped s/sp shells, 50 points/atom",
    1: "configs[1]: 300-atom peptide-like chain, 6-31G-shaped s/sp shells, 110 points/atom",
    2: "configs[2]: 1000-atom chain, 6-31G-shaped s/sp shells, 110 points/atom",
    3: "configs[3]: 2000-atom chain, 6-31G-shaped s/sp shells + one d shell per heavy atom, 194 points/atom",
}

# Work per unit.  The figures bench.py uses come from the committed ncu counter capture under profiles/ (workmodel.load:
# 2 DFMA + DADD + DMUL and the FP64 thread instructions of one launch divided by the units it processed).  The table below
# is the hand count from the kernels' arithmetic: used, and labelled "hand count", only for a kernel the
# capture does not list.  [FP64-pipe instructions, flop (FMA = 2)] per unit, L = 0..4.
HAND_WORK = {
    "amatvec_R4": (11.44, 19.5), "amatvec_R2": (11.69, 19.75), "amatvec_cgp": (12.0, 20.5),
    "potential": [(12, 18), (17, 26), (28, 45), (51, 85), (97, 164)],
    "fock": [(12, 18), (17, 27), (28, 44), (51, 81), (90, 146)],
}


def work_of(model: dict, op: str, L: int = 0, M: int = 0, amat_key: str | None = None) -> dict:
    """{instr, flop, traffic_per_unit, source} of one unit of kernel `op` (integral class L, or the A q sweep at M points)."""
    key = f"{op}_L{L}" if op in ("potential", "fock") else (amat_key or ("amatvec_R4" if M >= PERSIST_MAX else "amatvec_cgp"))
    rec = model.get(key)
    if rec is None and key == "amatvec_cgp":       # an older capture: the separate-launch small-M kernel
        key = "amatvec_R2"
        rec = model.get(key)
    if rec:
        return {"key": key, "instr": rec["fp64_instr_per_unit"], "flop": rec["flop_per_unit"], "traffic_per_unit": rec["traffic_per_unit"],
                "issue_slots": rec.get("issue_slots_per_unit"),
                "source": f"ncu counters, {model['_source']['file']} ({rec['workload']})"}
    hw = HAND_WORK[op][L] if op in ("potential", "fock") else HAND_WORK.get(key, HAND_WORK["amatvec_R4"])
    return {"key": key, "instr": hw[0], "flop": hw[1], "traffic_per_unit": None, "issue_slots": None,
            "source": "hand count (no capture of this kernel under profiles/)"}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ----------------------------------------------------------------------------- N > 1: replicas only
def max_over_ranks(ms: float, dist, device) -> float:
    """The contract's timing rule: the slowest rank's device time.  dist = torch.distributed (initialised) or None."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world: int, units_per_step: float, ms_per_step: float) -> float:
    """Whole-job throughput of `world` independent replicas of the step (weak scaling: every rank does the same work)."""
    return world * units_per_step / (ms_per_step * 1e-3)


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, window=None):
        """window = (t0, t1) in time.perf_counter(): only the samples that arrived inside it count (the sampler is started
        before the warm-up steps because nvidia-smi needs ~0.1 s to deliver its first line); all samples if none did."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        lines = list(self.lines)
        inside = [ln for (t, ln) in lines if window and window[0] <= t <= window[1] + 0.02]
        scope = "timed region" if inside else "warm-up + timed region"
        for ln in (inside if inside else [ln for (_, ln) in lines]):
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(power), "samples": len(sm),
                "sampled_over": scope, "reasons": sorted(reasons)}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


# ----------------------------------------------------------------------------- the CPU oracle legs
def pair_table(w, cutoff=1e-20, eps=1e-12, chunk=250_000):
    """Unordered shell pairs (I <= J) that keep at least one primitive pair at the oracle's cutoff |c_i c_j| K_AB >= 1e-20, and per
    pair: `kept` = primitive pairs the oracle evaluates, `nominal` = primitive pairs an Eq. 15 screening at 1e-12 keeps, estimated
    from the s-type bound |c_i c_j| (2 pi^{5/2}/(p^2 sqrt(2p)))^{1/2} K_AB (diagonal shell pairs counted i <= j).  Plain numpy
    bookkeeping, evaluated in chunks, used to size and extrapolate the oracle samples; it is part of neither arithmetic path."""
    from scipy.spatial import cKDTree
    b = w.basis
    ns, po = b.nshell, b.prim_offset
    E = np.ones((ns, 6))
    Cf = np.zeros((ns, 6))
    for sh in range(ns):
        n = int(b.shell_nprim[sh])
        E[sh, :n] = b.prim_exp[po[sh]:po[sh] + n]
        Cf[sh, :n] = np.abs(b.prim_coef[po[sh]:po[sh] + n])
    emin = np.where(Cf > 0, E, np.inf).min(axis=1)
    cmax = Cf.max(axis=1)
    # |c c| exp(-mu r^2) >= cutoff needs r^2 <= ln(c c / cutoff)/mu_min: one radius for the tree, the exact test per chunk
    mu_floor = float(emin.min()) / 2.0
    radius = float(np.sqrt(max(np.log(max(cmax.max() ** 2, 1e-300) / cutoff), 1.0) / mu_floor))
    pairs = np.concatenate([cKDTree(b.shell_xyz).query_pairs(radius, output_type="ndarray"), np.stack([np.arange(ns)] * 2, axis=1)])
    pairs = pairs.astype(np.int32)
    kept = np.zeros(len(pairs), np.int64)
    nominal = np.zeros(len(pairs), np.int64)
    tri = np.triu(np.ones((6, 6), bool))[None]
    for c0 in range(0, len(pairs), chunk):
        I, J = pairs[c0:c0 + chunk, 0], pairs[c0:c0 + chunk, 1]
        a, c = E[I][:, :, None], E[J][:, None, :]
        cc = Cf[I][:, :, None] * Cf[J][:, None, :]
        p = a + c
        r2 = np.sum((b.shell_xyz[I] - b.shell_xyz[J]) ** 2, axis=1)[:, None, None]
        k = cc * np.exp(-a * c / p * r2)
        kept[c0:c0 + chunk] = (k >= cutoff).sum(axis=(1, 2))
        keep = k * np.sqrt(2 * np.pi ** 2.5 / (p * p * np.sqrt(2 * p))) >= eps
        diag = (I == J)[:, None, None]
        nominal[c0:c0 + chunk] = np.where(diag, keep & tri, keep).sum(axis=(1, 2))
    alive = kept > 0
    return pairs[alive], kept[alive], nominal[alive]


def oracle_sample(w, table, n_points: int, n_pairs: int, threads: int | None = None, seed: int = 99):
    """Times the oracle, as it stands, on a bounded sample of pcm_potential + pcm_fock and extrapolates to the full calls.
    potential: n_points of the M surface points x the full square of shell pairs (scaled by M / n_points); Fock: n_pairs
    shell-pair blocks x all points, scaled by the primitive pairs the oracle keeps over the full ORDERED square (the oracle
    evaluates (I, J) and (J, I) independently, as orc_potential does)."""
    import oracle
    if threads:
        oracle.set_num_threads(threads)
    b, s = w.basis, w.surface
    rng = np.random.default_rng(seed)
    M = s.M
    pairs, kept, nominal = table
    # two sample sizes: orc_potential first builds its keep masks over the full square of shell pairs (a fixed cost that must not
    # be multiplied by M / n_points), so the full call is extrapolated from the slope between the two
    n1 = min(n_points, M)
    n2 = min(3 * n_points, M)
    pts2 = np.sort(rng.choice(M, size=n2, replace=False))
    pts = np.sort(rng.choice(pts2, size=n1, replace=False))
    t0 = time.perf_counter()
    oracle.potential(b, s, w.P, points=pts)
    t_pot = time.perf_counter() - t0
    t_pot2 = t_pot
    if n2 > n1:
        t0 = time.perf_counter()
        oracle.potential(b, s, w.P, points=pts2)
        t_pot2 = time.perf_counter() - t0
    pick = rng.choice(len(pairs), size=min(n_pairs, len(pairs)), replace=False)
    sel = np.ascontiguousarray(pairs[pick])
    t0 = time.perf_counter()
    oracle.fock_blocks(b, s, w.q, sel)
    t_fock = time.perf_counter() - t0
    offdiag = pairs[:, 0] != pairs[:, 1]
    ordered_total = float(kept[offdiag].sum()) * 2.0 + float(kept[~offdiag].sum())
    full_pot = t_pot + max(t_pot2 - t_pot, 0.0) / (n2 - n1) * (M - n1) if n2 > n1 else t_pot * M / n1
    full_fock = t_fock * ordered_total / float(kept[pick].sum())
    npp = int(nominal.sum())
    return {"threads": oracle.num_threads(), "points_sampled": int(len(pts)), "shell_pairs_sampled": int(len(sel)),
            "shell_pairs_alive": int(len(pairs)), "potential_s_sample": t_pot, "potential_s_sample_3x": t_pot2, "fock_s_sample": t_fock,
            "potential_s_full_extrapolated": full_pot, "fock_s_full_extrapolated": full_fock,
            "sample_s": t_pot + (t_pot2 if n2 > n1 else 0.0) + t_fock, "full_s_extrapolated": full_pot + full_fock, "prim_pairs_nominal": npp,
            "sample_units": npp * float(n1 + (n2 if n2 > n1 else 0)) + float(nominal[pick].sum()) * M,
            "value": 2.0 * npp * M / (full_pot + full_fock)}


def oracle_full(w, threads: int | None = None):
    """The oracle on a whole small workload (configs[0]): potential, Fock, A q and the RBJ-64 PCG, no extrapolation."""
    import oracle
    if threads:
        oracle.set_num_threads(threads)
    b, s = w.basis, w.surface
    t0 = time.perf_counter(); oracle.potential(b, s, w.P); t_pot = time.perf_counter() - t0
    t0 = time.perf_counter(); oracle.fock(b, s, w.q); t_fock = time.perf_counter() - t0
    t0 = time.perf_counter(); y = oracle.amatvec(s, w.q); t_mv = time.perf_counter() - t0
    t0 = time.perf_counter()
    rbj = oracle.rbj_build(s, min(RBJ_BLOCK, s.M), oracle.pivot_order(7, s.M))
    _, it, _, _ = oracle.pcg(s, y, CG_TOL, 2000, precond=2, rbj=rbj)
    t_solve = time.perf_counter() - t0
    return {"threads": oracle.num_threads(), "potential_ms": t_pot * 1e3, "fock_ms": t_fock * 1e3, "amatvec_ms": t_mv * 1e3,
            "rbj_pcg_ms": t_solve * 1e3, "cg_iters": int(it)}


def cpu_baseline_block(w3, M3, prim_pairs3):
    """cpu_baseline of the JSON line: the oracle on configs[3] (stratified sample, extrapolated) and on configs[0] (in full), each
    with one thread and with all threads (SURVEY.md 8(d) 'Oracle timing')."""
    import oracle
    oracle.build()
    allthreads = os.cpu_count() or 1
    table = pair_table(w3)
    many = oracle_sample(w3, table, n_points=2 * allthreads, n_pairs=40 * allthreads, threads=allthreads)
    one = oracle_sample(w3, table, n_points=2, n_pairs=40, threads=1)
    w0 = synth.make_workload(0)
    full0 = {"all_threads": oracle_full(w0, allthreads), "one_thread": oracle_full(w0, 1)}
    oracle.set_num_threads(allthreads)
    value = 2.0 * prim_pairs3 * M3 / many["full_s_extrapolated"]
    return {"value": value, "unit": UNIT, "cores": many["threads"], "kind": "oracle", "extrapolated": True,
            "sample": (f"configs[3]: potential on {many['points_sampled']} of {M3} points, Fock on {many['shell_pairs_sampled']} of "
                       f"{many['shell_pairs_alive']} shell pairs with a surviving primitive pair ({many['sample_s']:.1f} s), both extrapolated to the "
                       f"full calls over the ordered square of shell pairs; units = the library's surviving primitive pairs x points"),
            "configs3_all_threads": many, "configs3_one_thread": dict(one, value=2.0 * prim_pairs3 * M3 / one["full_s_extrapolated"]),
            "configs0_full": full0}


# ----------------------------------------------------------------------------- the CUDA arm
def base_config(w, world: int) -> dict:
    """The `config` object of the JSON line: generator-derived fields only, so that both arms print the same keys."""
    return {"workload": WORKLOADS[w.config], "atoms": len(w.elements), "nbf": int(w.basis.nbf), "surface_points": int(w.surface.M),
            "step": "pcm_potential(P -> v) + pcm_fock(q -> F); the full C-PCM step around them (RBJ build, PCG) is timed in `step`",
            "l2": "flushed between timed iterations (256 MiB memset, untimed); P and F (2 x nbf^2 x 8 B) exceed L2 anyway",
            "parallelism": "replicas only" if world > 1 else "1 GPU", "screen_eps": 1e-12}


def frac_table(info, M, ms_by_L, op, model, peak_tflops):
    """per class L: ms of the main kernel, units, flop-based fraction of the FP64 peak and the FP64-pipe fraction"""
    out = []
    for L in range(5):
        ms = ms_by_L[L]
        n = float(info.products[L]) * M
        if n == 0 or ms <= 0:
            out.append(None)
            continue
        wk = work_of(model, op, L)
        out.append({"ms": ms, "units": n, "frac": n * wk["flop"] / (ms * 1e-3) * 1e-12 / peak_tflops,
                    "fp64_pipe_frac": n * wk["instr"] * 2.0 / (ms * 1e-3) * 1e-12 / peak_tflops})
    return out


def measure_integrals(pcm, torch, ctx, P, q, flush, reps=5, warm=3):
    """pcm_potential and pcm_fock on device-resident inputs: CUDA events around each call, L2 flushed before each call.  The call
    times are taken with the library's own per-kernel events OFF (as in the timed region: with them on the class kernels are
    serialised); a second pass with them on gives the per-class kernel times."""
    stream = torch.cuda.current_stream()
    M, nbf = ctx.M, ctx.nbf
    v = torch.empty(M, dtype=torch.float64, device=P.device)
    F = torch.empty((nbf, nbf), dtype=torch.float64, device=P.device)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]

    def one():
        flush.zero_()
        e[0].record(stream)
        pcm.pcm_potential(ctx, P, v, stream=stream)
        e[1].record(stream)
        flush.zero_()
        e[2].record(stream)
        pcm.pcm_fock(ctx, q, F, stream=stream)
        e[3].record(stream)
        torch.cuda.synchronize()
        return e[0].elapsed_time(e[1]), e[2].elapsed_time(e[3])
    pcm.pcm_set_timing(ctx, False)
    l0 = pcm.pcm_launch_count(ctx)
    one()
    launches = pcm.pcm_launch_count(ctx) - l0
    ts = [one() for _ in range(warm - 1 + reps)][warm - 1:]
    pot, fock = [t[0] for t in ts], [t[1] for t in ts]
    pcm.pcm_set_timing(ctx, True)
    one()
    best = (1e30, None, None)
    for _ in range(max(2, reps // 2)):
        tp, tf = one()
        if tp + tf < best[0]:
            best = (tp + tf, pcm.pcm_last_class_ms(ctx, pcm.OP_POTENTIAL), pcm.pcm_last_class_ms(ctx, pcm.OP_FOCK))
    lp, lf = pcm.pcm_last_kernel_ms(ctx, pcm.OP_POTENTIAL)[2], pcm.pcm_last_kernel_ms(ctx, pcm.OP_FOCK)[2]
    return {"potential_ms": min(pot), "fock_ms": min(fock), "potential_ms_median": statistics.median(pot),
            "fock_ms_median": statistics.median(fock), "potential_ms_by_L": best[1], "fock_ms_by_L": best[2],
            "launches_per_call": {"potential": lp, "fock": lf, "potential_plus_fock": launches}}, v, F


def config_entry(pcm, torch, cfg, w, ctx, info, meas, t_setup, model, peak):
    M = ctx.M
    tot = meas["potential_ms"] + meas["fock_ms"]
    return {"config": cfg, "workload": WORKLOADS[cfg], "atoms": len(w.elements), "nbf": int(ctx.nbf), "M": int(M),
            "prim_pairs": int(info.prim_pairs_total), "prim_pairs_by_class": dict(zip(pcm.CLASS_NAMES, map(int, info.prim_pairs))),
            "products_by_L": list(map(int, info.products)), "prim_pair_points_per_call": info.prim_pair_points, "setup_s": t_setup,
            **{k: meas[k] for k in ("potential_ms", "fock_ms", "potential_ms_median", "fock_ms_median", "launches_per_call")},
            "potential_plus_fock_ms": tot, "prim_pair_point_per_s": 2.0 * info.prim_pair_points / (tot * 1e-3),
            "potential_by_L": frac_table(info, M, meas["potential_ms_by_L"], "potential", model, peak),
            "fock_by_L": frac_table(info, M, meas["fock_ms_by_L"], "fock", model, peak)}


def small_config_extras(pcm, torch, w, ctx, P, q, flush):
    """configs[0] is one-block-sized: every call is launch-latency bound (SURVEY.md 7 'report it honestly').  Times A q, the RBJ
    solve and pcm_potential replayed from a CUDA graph, in microseconds."""
    dev = P.device
    stream = torch.cuda.current_stream()
    out = {}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn, reps=20):
        ts = []
        for k in range(3 + reps):
            e0.record(stream); fn(); e1.record(stream); torch.cuda.synchronize()
            if k >= 3:
                ts.append(e0.elapsed_time(e1) * 1e3)
        return min(ts), statistics.median(ts)
    y = torch.empty(ctx.M, dtype=torch.float64, device=dev)
    out["amatvec_us"], out["amatvec_us_median"] = timed(lambda: pcm.pcm_amatvec(ctx, q, y, stream=stream))
    pcm.pcm_rbj_build(ctx, min(RBJ_BLOCK, ctx.M), seed=7)
    x = torch.zeros(ctx.M, dtype=torch.float64, device=dev)
    its = []
    out["rbj_solve_us"], out["rbj_solve_us_median"] = timed(lambda: its.append(pcm.pcm_cg_solve(ctx, y, x, tol=CG_TOL, max_iter=2000, precond=2, stream=stream)[1]), reps=5)
    out["rbj_solve_iters"] = int(its[-1])
    v = torch.empty(ctx.M, dtype=torch.float64, device=dev)
    # ordinary launches (the library's per-kernel timing is on here, which also keeps it from replaying its own graph)
    out["potential_us_plain"], _ = timed(lambda: pcm.pcm_potential(ctx, P, v, stream=stream))
    try:   # the ~10 launches of one pcm_potential call replayed from a CUDA graph: the library's own (pcm_options.graph_calls,
           # on by default at this size), then one the caller captures
        pcm.pcm_set_timing(ctx, False)
        out["potential_us_library_graph"], _ = timed(lambda: pcm.pcm_potential(ctx, P, v, stream=stream))
        side = torch.cuda.Stream(device=dev)
        side.wait_stream(stream)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            pcm.pcm_potential(ctx, P, v)
        torch.cuda.synchronize()
        out["potential_us_cuda_graph"], _ = timed(lambda: g.replay())
        del g
    except Exception as ex:   # reported, not hidden
        out["potential_us_cuda_graph"] = None
        out["cuda_graph_error"] = str(ex)[:200]
    finally:
        pcm.pcm_set_timing(ctx, True)
    return out


def amat_and_solver_sweep(pcm, torch, dev, flush, model, peak_tflops, with_solver=True):
    """configs[4]: the A q sweep at M = 10k .. 200k and pcm_cg_solve (RBJ-64 against Jacobi) to 1e-8 on b = A q_true."""
    stream = torch.cuda.current_stream()
    sweep, solver = [], []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for Ms in SWEEP_M:
        s4, q4, qt4 = synth.make_solver_points(Ms)
        c4 = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0),
                           s4.xyz, s4.zeta, s4.switch)
        pcm.pcm_set_timing(c4, True)
        i4 = pcm.pcm_get_info(c4)
        qd = torch.as_tensor(q4, dtype=torch.float64, device=dev)
        yd = torch.empty_like(qd)
        for _ in range(3):
            pcm.pcm_amatvec(c4, qd, yd)
        ts = []
        for _ in range(5):
            flush.zero_()
            pcm.pcm_amatvec(c4, qd, yd)
            ts.append(sum(pcm.pcm_last_kernel_ms(c4, pcm.OP_AMATVEC)[:2]))
        ms = min(ts)
        tw = []          # the same call with whatever the previous one left in L2 (the condition inside a PCG solve); reported, not the headline
        for _ in range(5):
            pcm.pcm_amatvec(c4, qd, yd)
            tw.append(sum(pcm.pcm_last_kernel_ms(c4, pcm.OP_AMATVEC)[:2]))
        ms_warm = min(tw)
        wk = work_of(model, "amatvec", M=Ms)
        pairs = 0.5 * float(Ms) * Ms
        tf = pairs * wk["flop"] / (ms * 1e-3) * 1e-12
        sweep.append({"M": Ms, "ms": ms, "ms_median": statistics.median(ts), "ms_warm_l2": ms_warm,
                      "frac_of_fp64_peak_warm_l2": pairs * wk["flop"] / (ms_warm * 1e-3) * 1e-12 / peak_tflops,
                      "entries_per_s": float(Ms) * Ms / (ms * 1e-3),
                      "pair_evaluations_per_s": pairs / (ms * 1e-3), "tflops": tf, "frac_of_fp64_peak": tf / peak_tflops,
                      "fp64_pipe_frac": pairs * wk["instr"] * 2.0 / (ms * 1e-3) * 1e-12 / peak_tflops, "work_model": wk["key"], "work_source": wk["source"],
                      "stored_near_bytes": int(i4.amat_stored_bytes),
                      "algorithmic_hbm_gbs": (48.0 * Ms + 16.0 * Ms + float(i4.amat_stored_bytes)) / (ms * 1e-3) * 1e-9})
        if with_solver and Ms in SOLVER_M:
            b = pcm.pcm_amatvec(c4, torch.as_tensor(qt4, dtype=torch.float64, device=dev))
            x = torch.zeros_like(b)
            rec = {"M": Ms, "tol": CG_TOL, "rhs": "b = A q_true, q_true seeded uniform [-0.05, 0.05]"}
            tb = []
            for _ in range(3):
                torch.cuda.synchronize()
                e0.record(stream); pcm.pcm_rbj_build(c4, RBJ_BLOCK, seed=7, stream=stream); e1.record(stream); torch.cuda.synchronize()
                tb.append(e0.elapsed_time(e1))
            rec["rbj_build_ms"] = min(tb)
            for name, pc in (("rbj64", 2), ("jacobi", 1)):
                tsol, it, ok, rt = [], 0, False, 0.0
                for _ in range(3):
                    flush.zero_()
                    e0.record(stream)
                    _, it, rr, rt, ok = pcm.pcm_cg_solve(c4, b, x, tol=CG_TOL, max_iter=5000, precond=pc, stream=stream)
                    e1.record(stream); torch.cuda.synchronize()
                    tsol.append(e0.elapsed_time(e1))
                rec[name] = {"iters": int(it), "ms": min(tsol), "ms_per_iter": min(tsol) / max(it, 1), "converged": bool(ok), "true_resid": rt}
            if Ms == RBJ_SWEEP_M:   # PAPER.md:192-196 (Figure 8, S1, S2): the block size against CG steps, build and solve time
                rec["rbj_block_sweep"] = []
                for blk in RBJ_SWEEP_BLOCKS:
                    torch.cuda.synchronize()
                    e0.record(stream); pcm.pcm_rbj_build(c4, blk, seed=7, stream=stream); e1.record(stream); torch.cuda.synchronize()
                    tbuild = e0.elapsed_time(e1)
                    tsol, it, ok = [], 0, False
                    for _ in range(2):
                        flush.zero_()
                        e0.record(stream)
                        _, it, rr, rt, ok = pcm.pcm_cg_solve(c4, b, x, tol=CG_TOL, max_iter=5000, precond=2, stream=stream)
                        e1.record(stream); torch.cuda.synchronize()
                        tsol.append(e0.elapsed_time(e1))
                    rec["rbj_block_sweep"].append({"block": blk, "iters": int(it), "solve_ms": min(tsol), "build_ms": tbuild, "converged": bool(ok)})
            if Ms < PERSIST_MAX:   # the same solve through the separate-launch path (pcm_options.cg_path = 1), for comparison
                c1 = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0),
                                   s4.xyz, s4.zeta, s4.switch, cg_path=1)
                pcm.pcm_rbj_build(c1, RBJ_BLOCK, seed=7, stream=stream)
                tsol, it = [], 0
                for _ in range(3):
                    flush.zero_()
                    e0.record(stream)
                    _, it, rr, rt, ok = pcm.pcm_cg_solve(c1, b, x, tol=CG_TOL, max_iter=5000, precond=2, stream=stream)
                    e1.record(stream); torch.cuda.synchronize()
                    tsol.append(e0.elapsed_time(e1))
                rec["rbj64_separate_launches"] = {"iters": int(it), "ms": min(tsol), "ms_per_iter": min(tsol) / max(it, 1)}
                rec["path"] = "persistent cooperative kernel (pcm_cgp.cu); rbj64_separate_launches = the same solve with cg_path = 1"
                pcm.pcm_destroy(c1)
            solver.append(rec)
        pcm.pcm_destroy(c4)
    return sweep, solver


def stored_a_comparison(pcm, torch, dev, flush, hbm_gbs):
    """the stored-A variant against the on-the-fly sweep, same persistent-kernel path, same
    bits.  Stored, an A q streams 4 M^2 bytes of far-field 1/r values plus the stored near patches; `warm` = back-to-back calls
    (what a CG iteration sees: L2-resident when it fits), `cold` = L2 flushed before the call."""
    out = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    z, zi = np.zeros(0), np.zeros(0, np.int32)
    for Ms in STORED_M:
        s4, q4, _ = synth.make_solver_points(Ms)
        qd = torch.as_tensor(q4, dtype=torch.float64, device=dev)
        yd = torch.empty_like(qd)
        rec = {"M": Ms}
        for name, sf in (("stored", 1), ("on_the_fly", -1)):
            c = pcm.pcm_setup(zi, np.zeros((0, 3)), zi, z, z, s4.xyz, s4.zeta, s4.switch, cg_path=2, store_far=sf)
            info = pcm.pcm_get_info(c)
            if not info.amat_persistent or (sf == 1 and info.amat_far_stored_bytes == 0):
                rec[name] = None
                pcm.pcm_destroy(c)
                continue
            pcm.pcm_set_timing(c, True)
            cold, warm = [], []
            for _ in range(3):
                pcm.pcm_amatvec(c, qd, yd)
            for _ in range(5):
                flush.zero_()
                pcm.pcm_amatvec(c, qd, yd)
                cold.append(sum(pcm.pcm_last_kernel_ms(c, pcm.OP_AMATVEC)[:2]))
            for _ in range(8):
                pcm.pcm_amatvec(c, qd, yd)
                warm.append(sum(pcm.pcm_last_kernel_ms(c, pcm.OP_AMATVEC)[:2]))
            nbytes = float(info.amat_far_stored_bytes + info.amat_stored_bytes)
            rec[name] = {"ms_cold": min(cold), "ms_warm": min(warm), "bytes_streamed": nbytes}
            if sf == 1:
                rec[name].update({"bound": "hbm", "achieved_gbs_cold": nbytes / (min(cold) * 1e-3) * 1e-9,
                                  "frac_of_hbm_peak_cold": nbytes / (min(cold) * 1e-3) * 1e-9 / hbm_gbs,
                                  "achieved_gbs_warm": nbytes / (min(warm) * 1e-3) * 1e-9})
            pcm.pcm_destroy(c)
        c = pcm.pcm_setup(zi, np.zeros((0, 3)), zi, z, z, s4.xyz, s4.zeta, s4.switch)
        info = pcm.pcm_get_info(c)
        rec["default_choice"] = ("stored" if info.amat_far_stored_bytes else "on_the_fly") + (" (persistent kernel)" if info.amat_persistent else " (separate launches)")
        pcm.pcm_destroy(c)
        out.append(rec)
    return {"rule": "pcm_options.store_far = 0: the far field is stored when far + near bytes <= 96 MB (resident in the 126 MB L2), i.e. M <~ 4 500; "
                    "above that the on-the-fly sweep is used (from HBM the stored form needs 4 M^2 B / 6.5 TB/s, no faster than the arithmetic)",
            "cases": out}


def run_ours(args):
    import torch
    import paper_1505_07851_b200 as pcm
    from paper_1505_07851_b200 import workmodel

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        pcm.lib(build=True)          # compiles the library first if it is missing or stale; one rank only
    if dist is not None:
        dist.barrier()
    pcm.lib()
    dev = torch.device("cuda", local)
    model = workmodel.load()

    t0 = time.perf_counter()
    w = synth.make_workload(args.config)
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=not args.no_extras)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    info = pcm.pcm_get_info(ctx)
    M, nbf = ctx.M, ctx.nbf
    units_per_step = 2.0 * info.prim_pair_points
    P = torch.as_tensor(w.P, dtype=torch.float64, device=dev)
    v = torch.empty(M, dtype=torch.float64, device=dev)
    q = torch.zeros(M, dtype=torch.float64, device=dev)
    F = torch.empty((nbf, nbf), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    pcm.pcm_set_timing(ctx, False)      # the library's own per-kernel events serialise the class kernels: off in the timed region
    stream = torch.cuda.current_stream()
    side = torch.cuda.Stream(device=dev, priority=-1)   # the RBJ build depends on the geometry only: it overlaps pcm_potential

    # Up to 150k points the RBJ block selection is one CTA: queued on a side stream it hides behind pcm_potential.  Above, it is a
    # cooperative kernel on every SM: overlapped it would only slow the potential down, so it is queued after it.
    overlap = M <= 150_000     # up to there the RBJ selection is one CTA (pcm_solver.cu RBJ_LOCAL_MAX) and runs beside the potential

    def step():
        if overlap:
            pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=side)   # first, so that its CTA finds a free SM
        pcm.pcm_potential(ctx, P, v, stream=stream)
        if not overlap:
            pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=stream)
        pcm.pcm_cg_solve(ctx, v, q, tol=CG_TOL, max_iter=2000, precond=2, stream=stream)
        pcm.pcm_fock(ctx, q, F, stream=stream)

    peak_tflops = pcm.pcm_fp64_peak(ctx, 10)
    sampler = ClockSampler(local)
    sampler.start()                          # before the warm-up: its first line takes ~0.1 s
    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    torch.cuda.synchronize()

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    cls_pot, cls_fock, main_ms, cg_mv = [], [], [], []
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = pcm.pcm_launch_count(ctx)
    wall0 = time.perf_counter()
    iters, rt, ok = None, None, None
    for k in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (not timed)
        ev[k][0].record(stream)
        if overlap:
            side.wait_event(ev[k][0])           # the build starts inside the timed region, concurrently with the potential
            pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=side)
        pcm.pcm_potential(ctx, P, v, stream=stream)
        ev[k][1].record(stream)
        if not overlap:
            pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=stream)
        _, iters, rr, rt, ok = pcm.pcm_cg_solve(ctx, v, q, tol=CG_TOL, max_iter=2000, precond=2, stream=stream)
        ev[k][2].record(stream)
        pcm.pcm_fock(ctx, q, F, stream=stream)
        ev[k][3].record(stream)
        ev[k][3].synchronize()
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    launches = pcm.pcm_launch_count(ctx) - launches0
    clocks = sampler.stop(window=(wall0, wall0 + wall))
    if dist is not None:
        dist.barrier()
    step_ms = [e[0].elapsed_time(e[3]) for e in ev]
    pot_ms = [e[0].elapsed_time(e[1]) for e in ev]
    solve_ms = [e[1].elapsed_time(e[2]) for e in ev]
    fock_ms = [e[2].elapsed_time(e[3]) for e in ev]
    # the headline: ms per pcm_potential + pcm_fock (BASELINE.json's first clause), slowest rank
    total_ms = max_over_ranks(sum(pot_ms) + sum(fock_ms), dist, dev)
    ms_per_step = total_ms / args.steps
    value = job_value(world, units_per_step, ms_per_step)
    whole_ms = max_over_ranks(sum(step_ms), dist, dev) / args.steps

    # ---- kernel breakdown (outside the timed region): the same calls with the library's per-kernel events on, which runs the class
    # kernels one after the other -- the per-class times and roofline fractions come from here
    pcm.pcm_set_timing(ctx, True)
    for k in range(1 + 3):
        flush.zero_()
        pcm.pcm_potential(ctx, P, v, stream=stream)
        flush.zero_()
        pcm.pcm_fock(ctx, q, F, stream=stream)
        torch.cuda.synchronize()
        if k >= 1:
            cls_pot.append(pcm.pcm_last_class_ms(ctx, pcm.OP_POTENTIAL))
            cls_fock.append(pcm.pcm_last_class_ms(ctx, pcm.OP_FOCK))
            main_ms.append((pcm.pcm_last_kernel_ms(ctx, pcm.OP_POTENTIAL), pcm.pcm_last_kernel_ms(ctx, pcm.OP_FOCK)))
    pcm.pcm_cg_solve(ctx, v, q.clone(), tol=CG_TOL, max_iter=2000, precond=2, stream=stream)
    cg_mv.append(pcm.pcm_last_cg_matvec_ms(ctx)[0])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peaks, peak_src = load_peaks()
    mean = lambda xs: float(sum(xs) / len(xs))
    cp = [mean([c[L] for c in cls_pot]) for L in range(5)]
    cf = [mean([c[L] for c in cls_fock]) for L in range(5)]
    # dominant kernel of the headline = the integral kernel with the largest share of potential + Fock (one launch per call each)
    mv_ms = mean(cg_mv)
    cands = [("potential", L, cp[L]) for L in range(5)] + [("fock", L, cf[L]) for L in range(5)]
    op, Ld, ms_dom = max(cands, key=lambda c: c[2])
    n_units = float(info.products[Ld]) * M
    wk = work_of(model, op, Ld)
    achieved = n_units * wk["flop"] / (ms_dom * 1e-3) * 1e-12
    kernels = {}
    for (o, L, ms) in cands:
        if ms > 0.005:
            wo = work_of(model, o, L)
            kernels[f"{o}_L{L}"] = {"ms_per_launch": ms, "launches_per_step": 1, "flop_per_unit": wo["flop"], "fp64_instr_per_unit": wo["instr"],
                                    "frac": float(info.products[L]) * M * wo["flop"] / (ms * 1e-3) * 1e-12 / peak_tflops,
                                    "fp64_pipe_frac": float(info.products[L]) * M * wo["instr"] * 2.0 / (ms * 1e-3) * 1e-12 / peak_tflops}
    wa = work_of(model, "amatvec", M=M)
    kernels["amatvec (CG iteration of the full step)"] = {
        "ms_per_launch": mv_ms, "launches_per_step": int(iters) + 1, "flop_per_unit": wa["flop"],
        "frac": 0.5 * float(M) * M * wa["flop"] / (mv_ms * 1e-3) * 1e-12 / peak_tflops if mv_ms > 0 else None}
    tpu = wk["traffic_per_unit"]
    roofline = {"bound": "alu", "kernel": f"{op}_kernel<L={Ld}> on {WORKLOADS[args.config].split(':')[0]}", "launches_per_step": 1,
                "share_of_step": min(1.0, ms_dom / ms_per_step), "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "peak_nominal": 148 * 64 * 2 * 1.965e-3, "frac_of_nominal": achieved / (148 * 64 * 2 * 1.965e-3),
                "traffic": tpu * n_units if tpu is not None else None,
                "traffic_source": (f"dram__bytes_read.sum + dram__bytes_write.sum per unit from {model['_source']['file']} x the units of this launch"
                                   if tpu is not None else "no ncu capture of this kernel under profiles/: null"),
                "algorithmic_bytes": 40.0 * M + (32.0 + 8.0 * [1, 4, 10, 20, 35][Ld]) * float(info.products[Ld]),
                "fp64_pipe_frac": n_units * wk["instr"] * 2.0 / (ms_dom * 1e-3) * 1e-12 / peak_tflops,
                # the bound these kernels actually sit on: issue cycles = 2 per FP64 warp instruction + 1 per other
                # instruction, 592 sub-partitions issuing one cycle per clock at the SM clock sampled during the timed region
                "issue_slot_frac": (n_units * wk["issue_slots"] / (592.0 * (clocks.get("sm_mhz") or 1965.0) * 1e6 * ms_dom * 1e-3)
                                    if wk.get("issue_slots") else None),
                "timed": "launch duration from the library's CUDA events in the breakdown pass after the timed region (class kernels one after the "
                         "other); in the timed region the class kernels of a call are a chain of programmatic dependent launches (tails overlap)",
                "units_per_launch": n_units, "flop_per_unit": wk["flop"], "fp64_instr_per_unit": wk["instr"], "work_source": wk["source"],
                "work_capture": model.get("_source"), "ms_per_launch": ms_dom, "all_hot_kernels": kernels,
                "peak_source": "measured live: pcm_fp64_peak DFMA chain (MEASURED_PEAKS.json has no fp64 entry; nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2)",
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}
    cfgd = base_config(w, world)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": f"synthetic (seeded generator, BASELINE.json configs[{args.config}] recipe; stands in for the paper's PDB proteins at RHF/6-31G(*))",
        "config": cfgd,
        "counts": {"prim_pairs": int(info.prim_pairs_total), "prim_pairs_by_class": dict(zip(pcm.CLASS_NAMES, map(int, info.prim_pairs))),
                   "products_by_L": list(map(int, info.products)), "prim_pair_points_per_call": info.prim_pair_points},
        "clocks": clocks, "gpu_launches": int(launches),
        "integrals": {"potential_ms": mean(pot_ms), "fock_ms": mean(fock_ms), "potential_plus_fock_ms": mean(pot_ms) + mean(fock_ms),
                      "prim_pair_point_per_s": units_per_step / ((mean(pot_ms) + mean(fock_ms)) * 1e-3),
                      "potential_main_ms_by_L": cp, "fock_main_ms_by_L": cf,
                      "potential_transform_ms": mean([m[0][1] for m in main_ms]), "fock_transform_ms": mean([m[1][1] for m in main_ms])},
        "step": {"what": ("pcm_potential || pcm_rbj_build_async(64) on a side stream" if overlap else "pcm_potential, pcm_rbj_build_async(64)") +
                         ", pcm_cg_solve(A q = v, 1e-8, RBJ-64), pcm_fock (solver_ms includes what of the RBJ build is not hidden)",
                 "ms": whole_ms, "potential_ms": mean(pot_ms), "solver_ms": mean(solve_ms), "fock_ms": mean(fock_ms),
                 "cg_iters": int(iters), "cg_converged": bool(ok), "cg_true_resid": rt, "amatvec_ms_per_iteration": mv_ms},
        "roofline": roofline, "setup_s": t_setup, "generate_s": t_gen, "wall_s_timed_region": wall,
    }

    # ---- end to end through the host-buffer C ABI (pinned host memory, copies inside the timed region)
    Ph = torch.as_tensor(w.P, dtype=torch.float64).pin_memory().numpy()
    qh = torch.as_tensor(q.cpu()).pin_memory().numpy()
    vh = torch.empty(M, dtype=torch.float64).pin_memory().numpy()
    Fh = torch.empty((nbf, nbf), dtype=torch.float64).pin_memory().numpy()

    def calls_host():
        pcm.pcm_potential_host(ctx, Ph, vh)
        pcm.pcm_fock_host(ctx, qh, Fh)
    calls_host()
    torch.cuda.synchronize()
    n_e2e = max(2, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        calls_host()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) / n_e2e * 1e3
    line["e2e"] = {"value": world * units_per_step / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms, "steps": n_e2e,
                   "h2d_bytes_per_step": int(info.components * 16 + M * 8), "d2h_bytes_per_step": int(info.components * 16 + M * 8),
                   "dense_matrix_bytes": int(nbf * nbf * 8),
                   "api": ("pcm_potential_host(P -> v) + pcm_fock_host(q -> F) on pinned host buffers, inside the timed region; of the dense "
                           "P and F only the elements of surviving shell pairs cross PCIe (gathered / scattered on the host, F zero-filled there)")}
    del Ph, Fh

    # ---- SURVEY 8(f) rows, timed outside the step: the PCM gradient term (Eq. 14/22) and the glue of Eq. 1/4/13
    if not args.no_extras:
        ge = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
        pcm.pcm_set_nuclei(ctx, w.atom_xyz, synth.nuclear_charges(w.elements))
        pcm.pcm_set_cavity(ctx, synth.cavity_radii(w.elements), w.surface.atom)
        f_eps = (78.39 - 1.0) / 78.39
        gms, glue_ms = [], []
        for k in range(1 + 3):
            flush.zero_()
            ge[0].record(stream)
            pcm.pcm_gradient(ctx, P, q, stream=stream)
            ge[1].record(stream)
            u = pcm.pcm_nuclear_potential(ctx, stream=stream)
            b = pcm.pcm_rhs(ctx, u, v, f_eps, stream=stream)
            ge[2].record(stream)
            en = pcm.pcm_energy(ctx, u, v, q, f_eps, stream=stream)
            ge[3].record(stream)
            pcm.pcm_surface_gradient(ctx, q, f_eps, stream=stream)
            ge[4].record(stream)
            torch.cuda.synchronize()
            if k >= 1:
                gms.append(ge[0].elapsed_time(ge[1]))
                glue_ms.append((ge[1].elapsed_time(ge[2]), ge[2].elapsed_time(ge[3]), ge[3].elapsed_time(ge[4])))
        line["gradient"] = {"ms": min(gms), "ms_median": statistics.median(gms), "prim_pair_point_per_s": info.prim_pair_points / (min(gms) * 1e-3),
                            "note": "pcm_gradient: Fock sweep at Hermite order L+1 and a three-accumulator point sweep; not part of the step"}
        line["glue"] = {"bz_plus_rhs_ms": min(g[0] for g in glue_ms), "energy_ms": min(g[1] for g in glue_ms),
                        "surface_gradient_ms": min(g[2] for g in glue_ms), "energy_hartree": float(en[3])}

    # ---- every config (SURVEY.md 8(d) "Reporting: for every config"): the headline's own entry from the calls timed alone
    per_config = []
    if not args.no_configs:
        meas, _, _ = measure_integrals(pcm, torch, ctx, P, q, flush, reps=3, warm=2)
        head = config_entry(pcm, torch, args.config, w, ctx, info, meas, t_setup, model, peak_tflops)
    pcm.pcm_destroy(ctx)
    del P, F, v
    torch.cuda.empty_cache()
    if not args.no_configs:
        for cfg in range(4):
            if cfg == args.config:
                per_config.append(head)
                continue
            wc = synth.make_workload(cfg)
            t0 = time.perf_counter()
            cc = pcm.setup_from_workload(wc.basis, wc.surface)
            torch.cuda.synchronize()
            ts = time.perf_counter() - t0
            Pc = torch.as_tensor(wc.P, dtype=torch.float64, device=dev)
            qc = torch.as_tensor(wc.q, dtype=torch.float64, device=dev)
            meas, _, _ = measure_integrals(pcm, torch, cc, Pc, qc, flush, reps=10 if cfg < 2 else 5)
            entry = config_entry(pcm, torch, cfg, wc, cc, pcm.pcm_get_info(cc), meas, ts, model, peak_tflops)
            if cfg == 0:
                entry["launch_bound"] = small_config_extras(pcm, torch, wc, cc, Pc, qc, flush)
            per_config.append(entry)
            pcm.pcm_destroy(cc)
            del Pc, qc
        line["per_config"] = per_config

    # ---- A q sweep and the solver on configs[4] (BASELINE metric: A q FP64 fraction; HBM GB/s reported as asked)
    if not args.no_sweep:
        line["amatvec"], line["solver"] = amat_and_solver_sweep(pcm, torch, dev, flush, model, peak_tflops)
        line["amatvec_stored"] = stored_a_comparison(pcm, torch, dev, flush, float(peaks.get("hbm_gbs", 6650.0)))

    # ---- the oracle on the host cores (reported baseline, not the target)
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline_block(w, M, int(info.prim_pairs_total))
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_kernels(args):
    """--mode kernels: only the three hot calls (potential and Fock of --config, A q at --amat-m points), W warm-up and K timed
    rounds, no solver and no oracle.  This is the command the ncu captures under profiles/ are taken with."""
    import torch
    import paper_1505_07851_b200 as pcm
    torch.cuda.set_device(0)
    pcm.lib(build=True)
    w = synth.make_workload(args.config)
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=args.with_gradient)
    s4, q4, _ = synth.make_solver_points(args.amat_m)
    c4 = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0), s4.xyz, s4.zeta, s4.switch)
    dev = torch.device("cuda", 0)
    P = torch.as_tensor(w.P, dtype=torch.float64, device=dev)
    q = torch.as_tensor(w.q, dtype=torch.float64, device=dev)
    qd = torch.as_tensor(q4, dtype=torch.float64, device=dev)
    for c in (ctx, c4):
        pcm.pcm_set_timing(c, True)
    out = {"potential_ms": [], "fock_ms": [], "amatvec_ms": [], "gradient_ms": [], "potential_by_L": None, "fock_by_L": None}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for k in range(args.warmup + args.steps):
        pcm.pcm_potential(ctx, P)
        pcm.pcm_fock(ctx, q)
        pcm.pcm_amatvec(c4, qd)
        e0.record()
        if args.with_gradient:
            pcm.pcm_gradient(ctx, P, q)
        e1.record()
        torch.cuda.synchronize()
        if k >= args.warmup:
            out["gradient_ms"].append(e0.elapsed_time(e1))
            out["potential_ms"].append(sum(pcm.pcm_last_kernel_ms(ctx, pcm.OP_POTENTIAL)[:2]))
            out["fock_ms"].append(sum(pcm.pcm_last_kernel_ms(ctx, pcm.OP_FOCK)[:2]))
            out["amatvec_ms"].append(sum(pcm.pcm_last_kernel_ms(c4, pcm.OP_AMATVEC)[:2]))
            out["potential_by_L"] = pcm.pcm_last_class_ms(ctx, pcm.OP_POTENTIAL)
            out["fock_by_L"] = pcm.pcm_last_class_ms(ctx, pcm.OP_FOCK)
    info = pcm.pcm_get_info(ctx)
    out.update({"mode": "kernels", "config": args.config, "M": ctx.M, "nbf": ctx.nbf, "amat_M": args.amat_m,
                "products_by_L": list(map(int, info.products)), "prim_pairs": int(info.prim_pairs_total)})
    print(json.dumps(out), flush=True)


def run_reference(args):
    """The oracle, as it stands, on the host cores: K steps, each a bounded sample of pcm_potential + pcm_fock on the headline
    workload.  ms_per_step is the MEASURED time of one sample; the full calls are extrapolated in a separate field."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    w = synth.make_workload(args.config)
    table = pair_table(w)
    threads = os.cpu_count() or 1
    npts, npairs = max(threads // 2, 1), 10 * threads
    for _ in range(max(args.warmup, 0)):
        oracle_sample(w, table, n_points=1, n_pairs=threads, threads=threads)
    samples = []
    t0 = time.perf_counter()
    for k in range(args.steps):
        samples.append(oracle_sample(w, table, n_points=npts, n_pairs=npairs, threads=threads, seed=99 + k))
    wall = time.perf_counter() - t0
    last = samples[-1]
    M = w.surface.M
    # throughput of the sampled work (units actually evaluated per second), and of the extrapolated full calls
    value = float(sum(s["sample_units"] for s in samples) / sum(s["sample_s"] for s in samples))
    full_s = float(np.mean([s["full_s_extrapolated"] for s in samples]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": wall / max(args.steps, 1) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": f"synthetic (seeded generator, BASELINE.json configs[{args.config}] recipe; stands in for the paper's PDB proteins at RHF/6-31G(*))",
            "config": base_config(w, world),
            "counts": {"prim_pairs_nominal": int(last["prim_pairs_nominal"])},
            "sample": {"per_step": f"oracle potential on {last['points_sampled']} + {3 * last['points_sampled']} of {M} points (two sizes: the slope "
                                   f"extrapolates), oracle Fock blocks of {last['shell_pairs_sampled']} of {last['shell_pairs_alive']} shell pairs",
                       "units_per_step": last["sample_units"], "full_calls_s_extrapolated": full_s,
                       "full_calls_value_extrapolated": 2.0 * last["prim_pairs_nominal"] * M / full_s},
            "cpu_baseline": {"value": value, "unit": UNIT, "kind": "oracle", "cores": last["threads"],
                             "sample": "the line's own steps (see `sample`); value = sampled units / measured time"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "wall_s": wall}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the configs[4] A q sweep and solver runs")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle timing (cpu_baseline)")
    ap.add_argument("--no-extras", action="store_true", help="skip the gradient / glue timings that follow the timed region")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config table (configs[0..3])")
    ap.add_argument("--mode", default="step", choices=["step", "kernels"], help="kernels: only the three hot calls (for ncu)")
    ap.add_argument("--config", type=int, default=CONFIG_INDEX, help="BASELINE.json config index 0..3 of the headline (default 3)")
    ap.add_argument("--amat-m", type=int, default=50_000, help="--mode kernels: surface points of the A q call")
    ap.add_argument("--with-gradient", action="store_true", help="--mode kernels: also run pcm_gradient")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.mode == "kernels":
        run_kernels(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
