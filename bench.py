#!/usr/bin/env python
"""bench.py -- one C-PCM step per timed iteration on the seeded synthetic workload of BASELINE.json configs[1].

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-sweep] [--no-cpu]

A step is one pass of the whole hot path on device-resident inputs:
    v = pcm_potential(P)  ||  pcm_rbj_build_async(64) on a side stream  ->  pcm_cg_solve(A q = v, tol 1e-8, RBJ)  ->  F = pcm_fock(q)
`value` = primitive-pair x point evaluated per second over the whole step (2 * prim_pair_points / step time: the
potential and the Fock build each evaluate every surviving primitive pair against every surface point; the
solver's time is inside the step, its work is not counted in the units).  The JSON line also carries the
BASELINE.json metric's other clauses: ms per pcm_potential + pcm_fock (`integrals`), the A q sweep of configs[4]
with its FP64 fraction (`amatvec`), the roofline of the dominant kernel, the oracle timed on the host (`cpu_baseline`)
and the same step through the host-buffer C ABI (`e2e`).

`--impl reference` times the CPU oracle (oracle/) on bounded samples of the same workload and prints the same
line with "impl": "reference".  N > 1: the path does not shard (north_star: one GPU) -- every rank runs an
independent replica of the step ("replicas only"), value = N * units / max-over-ranks time.
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
CONFIG_INDEX = 1
RBJ_BLOCK = 64
CG_TOL = 1e-8
SWEEP_M = (10_000, 50_000, 100_000, 200_000)

# Algorithmic fp64 work per (Hermite product, point) in the far field, counted from the kernel's arithmetic
# (DESIGN.md "Roofline"): [FP64-pipe instructions, flops (FMA = 2)] per unit for L = 0..4, potential and Fock.
# geometry 3 DADD + (1 DMUL + 2 DFMA) + rsqrt (2 DMUL + 3 DFMA) = 11 instr / 16 flop, then seeds and recursion.
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the hot kernels on the bench workload, from the ncu --set full
# captures summarised in profiles/r1e_ncu_full_summary.csv (a profiler number cannot be taken live).  The A q launch
# streams its stored near patches (50.3 MB on configs[1]; ncu flushes L2 between replays, in the step they stay in L2).
TRAFFIC = {"amatvec": 50.81e6, "potential": [1715456.0, 2184704.0, 1097216.0, None, None],
           "fock": [1547008.0, 1363712.0, 639232.0, None, None]}
WORK = {
    # A q: the sweep is symmetric -- one evaluation of 1/r_ij serves A_ij and A_ji; unit = one pair evaluation
    # (M^2/2 per call), R = 4 kernel: local-origin geometry 4 + 3/16 (1 DADD + 3 DFMA, the row shift amortised over 32
    # columns), rsqrt 5 (2 DMUL + 3 DFMA), two FMAs, 1/4 DADD of the column reduction = 11.44 instr, 19.4 flop.
    # Below 20 000 points the R = 2 kernel runs: row shift 6/32 per row, half a DADD of column reduction (11.69 instr, 19.75 flop).
    "amatvec": [(11.44, 19.5)],
    "amatvec_small": [(11.69, 19.75)],
    # L = 1, 2, 3: contracted before the seeds, Horner in u = 1/R^2 (pot_far_unit<1..3>); L = 4: generic recursion
    "potential": [(12, 18), (17, 26), (28, 45), (51, 85), (97, 164)],
    "fock": [(12, 18), (17, 27), (28, 44), (51, 81), (90, 146)],   # the charge multiplies the first seed only
}


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
def pair_table(w, radius=30.0):
    """Unordered shell pairs (I <= J) within `radius` bohr and, per pair, the [6 x 6] arrays of |c_i c_j| K_AB and of
    the s-type Schwarz estimate |c_i c_j| (2 pi^{5/2}/(p^2 sqrt(2p)))^{1/2} K_AB (padding entries are 0).  Plain numpy
    bookkeeping used to size and extrapolate the oracle samples; it is not part of either arithmetic path."""
    from scipy.spatial import cKDTree
    b = w.basis
    ns, po = b.nshell, b.prim_offset
    E = np.zeros((ns, 6))
    Cf = np.zeros((ns, 6))
    for sh in range(ns):
        n = int(b.shell_nprim[sh])
        E[sh, :n] = b.prim_exp[po[sh]:po[sh] + n]
        Cf[sh, :n] = np.abs(b.prim_coef[po[sh]:po[sh] + n])
    E[E == 0] = 1.0
    pairs = np.concatenate([cKDTree(b.shell_xyz).query_pairs(radius, output_type="ndarray"), np.stack([np.arange(ns)] * 2, axis=1)])
    I, J = pairs[:, 0], pairs[:, 1]
    a, c = E[I][:, :, None], E[J][:, None, :]
    cc = Cf[I][:, :, None] * Cf[J][:, None, :]
    p = a + c
    r2 = np.sum((b.shell_xyz[I] - b.shell_xyz[J]) ** 2, axis=1)[:, None, None]
    k = cc * np.exp(-a * c / p * r2)
    est = k * np.sqrt(2 * np.pi ** 2.5 / (p * p * np.sqrt(2 * p)))
    return pairs.astype(np.int32), k, est


def oracle_sample(w, info_prim_pairs: int, n_points: int, n_pairs: int, with_solver: bool, table=None, threads: int | None = None):
    """Times the oracle, as it stands, on a bounded sample of the step and extrapolates to one full step.
    potential: n_points of the M surface points x all shell pairs (scaled by M / n_points); Fock: n_pairs unordered
    shell pairs x all points (scaled by the primitive pairs the oracle's 1e-20 cutoff keeps); solver: the full
    RBJ build + PCG with stored A.  Returns a dict."""
    import oracle
    if threads:
        oracle.set_num_threads(threads)
    b, s = w.basis, w.surface
    rng = np.random.default_rng(99)
    M = s.M
    pts = np.sort(rng.choice(M, size=min(n_points, M), replace=False))
    t0 = time.perf_counter()
    oracle.potential(b, s, w.P, points=pts)
    t_pot = time.perf_counter() - t0
    pairs, k, _ = table if table is not None else pair_table(w)
    kept = (k >= 1e-20).sum(axis=(1, 2))
    alive = np.flatnonzero(kept > 0)
    pick = alive[rng.choice(len(alive), size=min(n_pairs, len(alive)), replace=False)]
    sel = np.ascontiguousarray(pairs[pick])
    t0 = time.perf_counter()
    oracle.fock_blocks(b, s, w.q, sel)
    t_fock = time.perf_counter() - t0
    full_pot = t_pot * M / len(pts)
    full_fock = t_fock * float(kept.sum()) / float(kept[pick].sum())
    out = {"potential_s_sample": t_pot, "fock_s_sample": t_fock, "potential_s_full_extrapolated": full_pot,
           "fock_s_full_extrapolated": full_fock, "points_sampled": int(len(pts)), "shell_pairs_sampled": int(len(sel)),
           "shell_pairs_alive": int(len(alive)), "threads": oracle.num_threads()}
    t_solve = 0.0
    if with_solver:
        t0 = time.perf_counter()
        A = oracle.amatrix(s)
        rbj = oracle.rbj_build(s, RBJ_BLOCK, oracle.pivot_order(7, M))
        rhs = np.random.default_rng(5).uniform(1.0, 3.0, M)   # a potential-like right-hand side of the right size
        _, it, rr, _ = oracle.pcg(s, rhs, CG_TOL, 2000, precond=2, rbj=rbj, A=A)
        t_solve = time.perf_counter() - t0
        out.update({"solver_s": t_solve, "solver_iters": int(it)})
    step_s = full_pot + full_fock + t_solve
    out["step_s_extrapolated"] = step_s
    out["value"] = 2.0 * info_prim_pairs * M / step_s
    return out


def nominal_prim_pairs(table, eps=1e-12):
    """Primitive pairs an Eq. 15 screening keeps, estimated without the product library (used by --impl reference only)
    from the s-type bound; unordered, diagonal shell pairs counted i <= j."""
    pairs, _, est = table
    keep = est >= eps
    diag = pairs[:, 0] == pairs[:, 1]
    n = int(keep[~diag].sum())
    n += int(np.triu(np.ones((6, 6), bool))[None, :, :].__and__(keep[diag]).sum())
    return n


# ----------------------------------------------------------------------------- the CUDA arm
def run_ours(args):
    import torch
    import paper_1505_07851_b200 as pcm

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

    t0 = time.perf_counter()
    w = synth.make_workload(CONFIG_INDEX)
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=True)
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
    pcm.pcm_set_timing(ctx, True)
    stream = torch.cuda.current_stream()

    side = torch.cuda.Stream(device=dev, priority=-1)   # the RBJ build depends on the geometry only: it overlaps pcm_potential

    def step():
        pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=side)   # first, so that its one CTA finds a free SM
        pcm.pcm_potential(ctx, P, v, stream=stream)
        _, it, rr, rt, ok = pcm.pcm_cg_solve(ctx, v, q, tol=CG_TOL, max_iter=2000, precond=2, stream=stream)
        pcm.pcm_fock(ctx, q, F, stream=stream)
        return it, rr, rt, ok

    peak_tflops = pcm.pcm_fp64_peak(ctx, 10)
    sampler = ClockSampler(local)
    sampler.start()                          # before the warm-up: its first line takes ~0.1 s
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    cls_pot, cls_fock, main_ms, cg_mv = [], [], [], []
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = pcm.pcm_launch_count(ctx)
    wall0 = time.perf_counter()
    iters = None
    for k in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (not timed)
        ev[k][0].record(stream)
        side.wait_event(ev[k][0])               # the build starts inside the timed region, concurrently with the potential
        pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=side)
        pcm.pcm_potential(ctx, P, v, stream=stream)
        ev[k][1].record(stream)
        _, iters, rr, rt, ok = pcm.pcm_cg_solve(ctx, v, q, tol=CG_TOL, max_iter=2000, precond=2, stream=stream)
        ev[k][2].record(stream)
        pcm.pcm_fock(ctx, q, F, stream=stream)
        ev[k][3].record(stream)
        ev[k][3].synchronize()
        cls_pot.append(pcm.pcm_last_class_ms(ctx, pcm.OP_POTENTIAL))
        cls_fock.append(pcm.pcm_last_class_ms(ctx, pcm.OP_FOCK))
        main_ms.append((pcm.pcm_last_kernel_ms(ctx, pcm.OP_POTENTIAL), pcm.pcm_last_kernel_ms(ctx, pcm.OP_FOCK)))
        cg_mv.append(pcm.pcm_last_cg_matvec_ms(ctx)[0])
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
    total_ms = max_over_ranks(sum(step_ms), dist, dev)
    ms_per_step = total_ms / args.steps
    value = job_value(world, units_per_step, ms_per_step)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peaks, peak_src = load_peaks()
    mean = lambda xs: float(sum(xs) / len(xs))
    cp = [mean([c[L] for c in cls_pot]) for L in range(5)]
    cf = [mean([c[L] for c in cls_fock]) for L in range(5)]
    # dominant kernel = the kernel with the largest share of the step's device time (launch time x launches per step):
    # the A q sweep of the CG iterations (timed per launch inside pcm_cg_solve, main + concurrent near kernel) or one
    # of the integral kernels (one launch per step each)
    mv_ms = mean(cg_mv)
    cands = [("potential", L, cp[L], 1) for L in range(5)] + [("fock", L, cf[L], 1) for L in range(5)]
    cands.append(("amatvec", 0, mv_ms, int(iters) + 1))
    op, Ld, ms_dom, per_step = max(cands, key=lambda c: c[2] * c[3])
    n_units = 0.5 * float(M) * M if op == "amatvec" else float(info.products[Ld]) * M
    wk = lambda o, L: WORK["amatvec_small" if (o == "amatvec" and M < 20000) else o][L]
    instr, flop = wk(op, Ld)
    achieved = n_units * flop / (ms_dom * 1e-3) * 1e-12
    kernels = {f"{o}_L{L}": {"ms_per_launch": ms, "launches_per_step": n,
                             "frac": (0.5 * float(M) * M if o == "amatvec" else float(info.products[L]) * M) * wk(o, L)[1] / (ms * 1e-3) * 1e-12 / peak_tflops}
               for (o, L, ms, n) in cands if ms > 0.01}
    roofline = {"bound": "alu", "kernel": ("amatvec_kernel (CG iteration, M = %d; unit = pair evaluation of the symmetric sweep)" % M)
                if op == "amatvec" else f"{op}_kernel<L={Ld}>", "launches_per_step": per_step,
                "share_of_step": ms_dom * per_step / ms_per_step, "all_hot_kernels": kernels,
                "achieved": achieved, "peak": peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                "traffic": TRAFFIC["amatvec"] if op == "amatvec" else TRAFFIC[op][Ld],
                "traffic_source": "bytes per launch, ncu --set full capture in profiles/r1e_ncu_full_summary.csv",
                "algorithmic_bytes": (48.0 * M + float(info.amat_stored_bytes) if op == "amatvec" else 40.0 * M + (32.0 + 8.0 * [1, 4, 10, 20, 35][Ld]) * float(info.products[Ld])),
                "fp64_pipe_frac": n_units * instr * 2.0 / (ms_dom * 1e-3) * 1e-12 / peak_tflops,
                "units_per_launch": n_units, "flop_per_unit": flop, "fp64_instr_per_unit": instr, "ms_per_launch": ms_dom,
                "peak_source": "measured live: pcm_fp64_peak DFMA chain (nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2)",
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded generator, BASELINE.json configs[1] recipe; stands in for the paper's PDB proteins at RHF/6-31G)",
        "config": {"workload": "configs[1]: 300-atom peptide-like chain, 6-31G-shaped s/sp shells, 110 points/atom",
                   "atoms": len(w.elements), "nbf": int(nbf), "surface_points": int(M),
                   "prim_pairs": int(info.prim_pairs_total), "prim_pairs_by_class": dict(zip(pcm.CLASS_NAMES, map(int, info.prim_pairs))),
                   "products_by_L": list(map(int, info.products)), "prim_pair_points_per_call": info.prim_pair_points,
                   "step": "pcm_potential || pcm_rbj_build_async(64) on a side stream, then pcm_cg_solve(1e-8, RBJ) + pcm_fock",
                   "l2": "flushed between timed steps (256 MiB memset, untimed)", "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "screen_eps": 1e-12},
        "clocks": clocks, "gpu_launches": int(launches),
        "integrals": {"potential_ms": mean(pot_ms), "fock_ms": mean(fock_ms), "potential_plus_fock_ms": mean(pot_ms) + mean(fock_ms),
                      "prim_pair_point_per_s": units_per_step / ((mean(pot_ms) + mean(fock_ms)) * 1e-3),
                      "potential_main_ms_by_L": cp, "fock_main_ms_by_L": cf,
                      "potential_transform_ms": mean([m[0][1] for m in main_ms]), "fock_transform_ms": mean([m[1][1] for m in main_ms])},
        "solver": {"ms": mean(solve_ms), "cg_iters": int(iters), "precond": f"RBJ-{RBJ_BLOCK}", "tol": CG_TOL},
        "roofline": roofline, "setup_s": t_setup, "generate_s": t_gen, "wall_s_timed_region": wall,
    }

    # ---- end to end through the host-buffer C ABI (pinned host memory, copies inside the timed region)
    Ph = torch.as_tensor(w.P, dtype=torch.float64).pin_memory().numpy()
    vh = torch.empty(M, dtype=torch.float64).pin_memory().numpy()
    Fh = torch.empty((nbf, nbf), dtype=torch.float64).pin_memory().numpy()
    def step_host():
        pcm.pcm_rbj_build_async(ctx, RBJ_BLOCK, seed=7, stream=side)
        pcm.pcm_potential_host(ctx, Ph, vh)
        xh, it, _, _, _ = pcm.pcm_cg_solve_host(ctx, vh, tol=CG_TOL, max_iter=2000, precond=2)
        pcm.pcm_fock_host(ctx, xh, Fh)
    step_host()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_host()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) / args.steps * 1e3
    line["e2e"] = {"value": world * units_per_step / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                   "h2d_bytes_per_step": int(nbf * nbf * 8 + 2 * M * 8), "d2h_bytes_per_step": int(nbf * nbf * 8 + 2 * M * 8),
                   "api": "pcm_rbj_build_async || pcm_potential_host, pcm_cg_solve_host, pcm_fock_host"}

    # ---- SURVEY 8(f) rows built so far, timed outside the step: the PCM gradient term (Eq. 14/22) and the glue of Eq. 1/4/13
    ge = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
    pcm.pcm_set_nuclei(ctx, w.atom_xyz, synth.nuclear_charges(w.elements))
    pcm.pcm_set_cavity(ctx, synth.cavity_radii(w.elements), w.surface.atom)
    f_eps = (78.39 - 1.0) / 78.39
    gms, glue_ms = [], []
    for k in range(0 if args.no_extras else 3 + 5):
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
        if k >= 3:
            gms.append(ge[0].elapsed_time(ge[1]))
            glue_ms.append((ge[1].elapsed_time(ge[2]), ge[2].elapsed_time(ge[3]), ge[3].elapsed_time(ge[4])))
    if not args.no_extras:
      line["gradient"] = {"ms": min(gms), "ms_median": statistics.median(gms), "prim_pair_point_per_s": info.prim_pair_points / (min(gms) * 1e-3),
                        "note": "pcm_gradient: Fock sweep at Hermite order L+1 and a three-accumulator point sweep; not part of the step"}
      line["glue"] = {"bz_plus_rhs_ms": min(g[0] for g in glue_ms), "energy_ms": min(g[1] for g in glue_ms),
                    "surface_gradient_ms": min(g[2] for g in glue_ms), "energy_hartree": float(en[3])}

    # ---- A q sweep of configs[4] (BASELINE metric: A q FP64 fraction; HBM GB/s reported as asked)
    if not args.no_sweep:
        sweep = []
        for Ms in SWEEP_M:
            s4, q4, qt4 = synth.make_solver_points(Ms)
            c4 = pcm.pcm_setup(np.zeros(0, np.int32), np.zeros((0, 3)), np.zeros(0, np.int32), np.zeros(0), np.zeros(0),
                               s4.xyz, s4.zeta, s4.switch)
            pcm.pcm_set_timing(c4, True)
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
            instr, flop = WORK["amatvec" if Ms >= 20000 else "amatvec_small"][0]
            pairs = 0.5 * float(Ms) * Ms
            tf = pairs * flop / (ms * 1e-3) * 1e-12
            sweep.append({"M": Ms, "ms": ms, "ms_median": statistics.median(ts), "entries_per_s": float(Ms) * Ms / (ms * 1e-3),
                          "pair_evaluations_per_s": pairs / (ms * 1e-3),
                          "tflops": tf, "frac_of_fp64_peak": tf / peak_tflops,
                          "fp64_pipe_frac": pairs * instr * 2.0 / (ms * 1e-3) * 1e-12 / peak_tflops,
                          "algorithmic_hbm_gbs": (40.0 * Ms + 16.0 * Ms) / (ms * 1e-3) * 1e-9})
            pcm.pcm_destroy(c4)
        line["amatvec"] = sweep

    # ---- the oracle on the host cores (reported baseline, not the target)
    if world == 1 and not args.no_cpu:
        ob = oracle_sample(w, int(info.prim_pairs_total), n_points=192, n_pairs=3000, with_solver=True)
        line["cpu_baseline"] = {"value": ob["value"], "unit": UNIT, "cores": ob["threads"], "kind": "oracle",
                                "sample": (f"potential on {ob['points_sampled']} of {M} points, Fock on {ob['shell_pairs_sampled']} of "
                                           f"{ob['shell_pairs_alive']} shell pairs (both extrapolated to the full step), "
                                           f"full RBJ-{RBJ_BLOCK} PCG with stored A ({ob['solver_iters']} iterations)"),
                                "detail": ob}
    print(json.dumps(line), flush=True)
    pcm.pcm_destroy(ctx)
    if dist is not None:
        dist.destroy_process_group()


def run_kernels(args):
    """--mode kernels: only the three hot calls (configs[1] potential and Fock, configs[4] A q at M = 50k), W warm-up
    and K timed rounds, no solver and no oracle.  This is the command the ncu captures under profiles/ are taken with."""
    import torch
    import paper_1505_07851_b200 as pcm
    torch.cuda.set_device(0)
    pcm.lib(build=True)
    w = synth.make_workload(args.config)
    ctx = pcm.setup_from_workload(w.basis, w.surface, gradient=True)
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
    """The oracle, as it stands, on the host cores: K steps, each a bounded sample of the configs[1] step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    w = synth.make_workload(CONFIG_INDEX)
    table = pair_table(w)
    npp = nominal_prim_pairs(table)
    for _ in range(max(args.warmup, 0)):
        oracle_sample(w, npp, n_points=8, n_pairs=100, with_solver=False, table=table)
    vals, last = [], None
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = oracle_sample(w, npp, n_points=64, n_pairs=1000, with_solver=True, table=table)
        vals.append(last["value"])
    wall = time.perf_counter() - t0
    value = float(len(vals) / sum(1.0 / v for v in vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": last["step_s_extrapolated"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic (seeded generator, BASELINE.json configs[1] recipe)",
            "config": {"workload": "configs[1]: 300-atom peptide-like chain, 6-31G-shaped s/sp shells, 110 points/atom",
                       "surface_points": int(w.surface.M), "nbf": int(w.basis.nbf), "prim_pairs_nominal": int(npp),
                       "step": "oracle potential + RBJ-64 PCG (stored A) + oracle Fock; ms_per_step is extrapolated from the sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "kind": "oracle", "cores": last["threads"],
                             "sample": (f"per step: potential on {last['points_sampled']} of {w.surface.M} points, Fock on "
                                        f"{last['shell_pairs_sampled']} of {last['shell_pairs_alive']} shell pairs "
                                        f"(extrapolated), full RBJ-PCG")},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "wall_s": wall}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the configs[4] A q sweep")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle timing (cpu_baseline)")
    ap.add_argument("--no-extras", action="store_true", help="skip the gradient / glue timings that follow the timed region")
    ap.add_argument("--mode", default="step", choices=["step", "kernels"], help="kernels: only the three hot calls (for ncu)")
    ap.add_argument("--config", type=int, default=CONFIG_INDEX, help="--mode kernels: BASELINE.json config index 0..3")
    ap.add_argument("--amat-m", type=int, default=50_000, help="--mode kernels: surface points of the A q call")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.mode == "kernels":
        run_kernels(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
