"""Work per unit of the hot kernels, taken from a committed ncu counter capture instead of hand counts.

`profiles/<tag>_flops.csv` holds one row per hot kernel: the FP64 instruction counters of one launch
(`sm__sass_thread_inst_executed_op_{dfma,dadd,dmul}_pred_on.sum`, `sm__inst_executed_pipe_fp64.sum`), its DRAM bytes
(`dram__bytes_read.sum + dram__bytes_write.sum`), its duration under ncu and the units that launch processed
(Hermite products of the class x surface points for the integral kernels, M^2/2 pair evaluations for the symmetric
A q sweep).  `load()` turns it into per-unit figures keyed by kernel:

    flop_per_unit        = (2 DFMA + DADD + DMUL) / units
    fp64_instr_per_unit  = (DFMA + DADD + DMUL) / units                  (thread instructions on the FP64 pipe)
    traffic_per_unit     = DRAM bytes / units
    issue_slots_per_unit = (FP64 warp instructions + all warp instructions) / units   (an FP64 instruction takes two issue cycles)

`python -m paper_1505_07851_b200.workmodel RAW.csv KERNELS.json [--no-header] >> profiles/<tag>_flops.csv`
writes its rows from the raw `ncu --csv --page raw --print-units base` output of one `bench.py --mode kernels` run and the
JSON line the same command printed without ncu (it carries M and the products per L, i.e. the units).  No arithmetic of the method lives
here; this is bookkeeping for bench.py's roofline.
"""
from __future__ import annotations

import csv
import glob
import hashlib
import json
import os
import re
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FIELDS = ["key", "kernel", "workload", "units", "time_us", "dfma", "dadd", "dmul", "fp64_warp_inst", "dram_bytes", "regs", "grid",
          "fp64_pipe_pct_elapsed", "warp_inst"]
METRICS = {
    "dfma": "sm__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "dadd": "sm__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "dmul": "sm__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "fp64_warp_inst": "sm__inst_executed_pipe_fp64.sum",
    "dram_read": "dram__bytes_read.sum",
    "dram_write": "dram__bytes_write.sum",
    "time": "gpu__time_duration.sum",
    "regs": "launch__registers_per_thread",
    "pipe": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "warp_inst": "smsp__inst_executed.sum",
}
NCU_METRICS = ",".join(METRICS[k] for k in ("dfma", "dadd", "dmul", "fp64_warp_inst", "dram_read", "dram_write", "time", "regs", "pipe", "warp_inst"))


def kernel_key(name: str) -> str | None:
    """'void pcm::potential_kernel<2, 2, 2>(...)' -> 'potential_L2'; A q kernels -> 'amatvec_R<R>'."""
    m = re.search(r"(potential|fock)_kernel<\s*(\d+)", name)
    if m and "near" not in name:
        return f"{m.group(1)}_L{m.group(2)}"
    m = re.search(r"(potential|fock)_near_kernel<\s*(\d+)", name)
    if m:
        return f"{m.group(1)}_near_L{m.group(2)}"
    m = re.search(r"cgp_matvec_kernel<\s*(\d+)", name)
    if m:
        return "amatvec_cgp" if m.group(1) == "0" else f"amatvec_cgp_mode{m.group(1)}"
    m = re.search(r"amatvec\w*_kernel<\s*(\d+)", name)
    if m:
        return f"amatvec_R{m.group(1)}"
    m = re.search(r"(\w+)_kernel", name)
    return m.group(1) if m else None


def latest_csv() -> str | None:
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "*_flops.csv")))
    return files[-1] if files else None


def load(path: str | None = None) -> dict:
    """{key: {flop_per_unit, fp64_instr_per_unit, traffic_per_unit, ...}, '_source': {file, sha16}}; {} if no capture."""
    path = path or latest_csv()
    if not path or not os.path.exists(path):
        return {}
    out = {}
    with open(path, newline="") as f:
        raw = f.read()
    for row in csv.DictReader(raw.splitlines()):
        try:
            units = float(row["units"])
            dfma, dadd, dmul = float(row["dfma"]), float(row["dadd"]), float(row["dmul"])
        except (KeyError, ValueError):
            continue
        if units <= 0:
            continue
        key = row["key"] + ("@" + row["workload"] if row.get("workload") else "")
        rec = {"flop_per_unit": (2 * dfma + dadd + dmul) / units, "fp64_instr_per_unit": (dfma + dadd + dmul) / units,
               "traffic_per_unit": float(row["dram_bytes"]) / units if row.get("dram_bytes") else None,
               "traffic_per_launch": float(row["dram_bytes"]) if row.get("dram_bytes") else None,
               "units": units, "time_us_under_ncu": float(row["time_us"]) if row.get("time_us") else None,
               "fp64_pipe_pct_elapsed": float(row["fp64_pipe_pct_elapsed"]) if row.get("fp64_pipe_pct_elapsed") else None,
               "workload": row.get("workload", "")}
        # issue slots per unit: on this part an FP64 warp instruction holds its sub-partition's issue port for two cycles, every
        # other instruction for one: (2 fp64 + other) = fp64 + all warp instructions, per unit
        if row.get("warp_inst") and row.get("fp64_warp_inst"):
            try:
                rec["issue_slots_per_unit"] = (float(row["warp_inst"]) + float(row["fp64_warp_inst"])) / units
            except ValueError:
                pass
        out[key] = rec
        out.setdefault(row["key"], rec)      # first row of a key = the default (largest workload first in the file)
    out["_source"] = {"file": os.path.relpath(path, ROOT), "sha16": hashlib.sha256(raw.encode()).hexdigest()[:16]}
    return out


def _summarise(raw_csv: str, kernel_json: str) -> list:
    """Rows of the summary CSV from the `ncu --csv --page raw --print-units base` output of ONE `bench.py --mode kernels`
    run and the JSON line that run printed; the first launch of every kernel is kept."""
    run = None
    for line in open(kernel_json):
        line = line.strip()
        if line.startswith("{") and '"mode": "kernels"' in line:
            run = json.loads(line)
    if run is None:
        raise SystemExit(f"{kernel_json}: no kernels-mode JSON line")
    with open(raw_csv, newline="") as f:
        lines = [ln for ln in f if ln.startswith('"')]
    rd = csv.reader(lines)
    header = next(rd)
    col = {h: i for i, h in enumerate(header)}
    rows, seen = [], set()
    for r in rd:
        if len(r) < len(header) or not r[col["ID"]].strip().isdigit():
            continue   # the units row
        name = r[col["Kernel Name"]]
        key = kernel_key(name)
        if key is None or key in seen:
            continue
        seen.add(key)

        def val(k):
            c = col.get(METRICS[k])
            try:
                return float(r[c].replace(",", "")) if c is not None else 0.0
            except ValueError:
                return 0.0
        if key.startswith("amatvec_cgp_mode"):
            continue     # the fill / stored variants of the one-launch sweep are not part of the work model
        if key.startswith("amatvec"):
            M = run["amat_M"]
            units, workload = 0.5 * M * M, f"configs[4] M={M}"
        elif key[-2] == "L" and key[-1].isdigit():
            units, workload = float(run["products_by_L"][int(key[-1])]) * run["M"], f"configs[{run['config']}]"
        else:
            continue     # not a hot kernel of the work model (transforms, reductions)
        rows.append({"key": key, "kernel": name.split("(")[0].replace("void ", "").strip(), "workload": workload, "units": f"{units:.6g}",
                     "time_us": f"{val('time') / 1e3:.3f}", "dfma": f"{val('dfma'):.0f}", "dadd": f"{val('dadd'):.0f}",
                     "dmul": f"{val('dmul'):.0f}", "fp64_warp_inst": f"{val('fp64_warp_inst'):.0f}",
                     "dram_bytes": f"{val('dram_read') + val('dram_write'):.0f}", "regs": f"{val('regs'):.0f}",
                     "grid": r[col["Grid Size"]] if "Grid Size" in col else "", "fp64_pipe_pct_elapsed": f"{val('pipe'):.2f}",
                     "warp_inst": f"{val('warp_inst'):.0f}"})
    return rows


if __name__ == "__main__":
    if len(sys.argv) < 3:
        sys.exit(__doc__)
    w = csv.DictWriter(sys.stdout, fieldnames=FIELDS)
    if "--no-header" not in sys.argv:
        w.writeheader()
    for row in _summarise(sys.argv[1], sys.argv[2]):
        w.writerow(row)
