"""Roofline bookkeeping for bench.py.  No arithmetic of the method lives here.

The roofline of a kernel (or of the step) is the slower of two ceilings (north_star: "the slower of the two"):

* HBM — the bytes the METHOD must move: u^n read once and u^{n+1} written once, 80 B per cell-update times the
  ghost-shell factor Np/N (SURVEY.md:480).  Every intermediate an implementation sends through HBM (interface
  states, first-pass fluxes) is implementation traffic and is NOT counted here; it is reported separately as the
  `decomposition` figures (what the present split into kernels has to move) and as ncu's measured `traffic`.
* FP64 — FP64 arithmetic instructions (DADD + DMUL + DFMA, thread level) per cell-update divided by the DFMA
  INSTRUCTION rate measured in the same run (ch_fp64_peak_probe: flop/s / 2).  DADD and DMUL take the same issue
  slot as DFMA, so instructions, not flops, are what the pipe is short of.

    roofline time = max(80 B x Np/N x N / hbm_gbs, inst_per_cell x N / dfma_inst_rate),   frac = that / measured.

A second ceiling is stated beside it because the first cannot be reached by this instruction mix: on B200 an FP64
warp instruction holds its scheduler's dispatch port for two cycles, every other instruction for about one, and the
two do not overlap (ch_issue_mix_probe measures both costs in the same run).  A kernel that executes F FP64-pipe and
O other warp instructions therefore needs at least (F t_fp64 + O t_alu) / (148 x 4 schedulers): its ISSUE ceiling.
Half of the instructions of this method are not FP64 arithmetic (selects of the limiters, compares, moves, address
arithmetic), so the issue ceiling sits at about twice the FP64 one; `issue_frac` says how close a kernel is to it.

The per-cell instruction counts are NOT typed in here: they are read from the ncu capture named by CAPTURE (a text
file committed under profiles/, taken at 512^3 with the kernels of the commit being benched), so every roofline
field can be reproduced from that one file and the bench line.  The same file supplies the measured DRAM traffic
per launch and ncu's sm__pipe_fp64_cycles_active, reported beside the fraction.
"""
from __future__ import annotations

import json
import os

CAPTURE = "profiles/r02_full_512_summary.txt"     # `metric | unit | one column per kernel`, see profiles/r02_README.md
CAPTURE_N = 512 ** 3                              # real cells of the captured launch

METHOD_BYTES_PER_CELL = 80.0                      # u^n in, u^{n+1} out: 2 x 5 doubles (SURVEY.md:480)

# What the present decomposition into kernels moves per REAL cell-update (every array a kernel consumes read once,
# every array it produces written once, no halo re-reads): implementation traffic, reported, not the roofline.
DECOMPOSITION_BYTES = {
    "k_pass1_x": 160.0,          # u (5) -> U*_L, U*_R(.,x), F*_x (15)
    "k_pass1_march<y>": 160.0,
    "k_pass1_march<z>": 160.0,
    "k_final3d": 440.0,          # U*_L, U*_R x3 (30) + F* x3 (15) + u (5) -> u (5)
}

SMS = 148
FP64_LANES_PER_SM = 64
HBM_FALLBACK_GBS = 6453.1     # MEASURED_PEAKS.json on this pool (used only if the file is absent)


def nominal_fp64_tflops(sm_mhz: float) -> float:
    return SMS * FP64_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def hbm_peak_gbs(root: str):
    """(GB/s, source) — the driver-written measured copy bandwidth if present."""
    p = os.path.join(root, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst copy bandwidth)"
    except (OSError, KeyError, ValueError):
        return HBM_FALLBACK_GBS, "fallback: MEASURED_PEAKS.json absent, last driver-measured value for this pool"


def kernel_key(ncu_name: str):
    """ch_kernel_name() key of an ncu kernel name (None for kernels that are not part of the step)."""
    n = ncu_name
    if "k_pass1_x" in n:
        return "k_pass1_x"
    if "k_pass1_march<1" in n or "k_pass1_march<(int)1" in n:
        return "k_pass1_march<y>"
    if "k_pass1_march<2" in n or "k_pass1_march<(int)2" in n:
        return "k_pass1_march<z>"
    if "k_final3d" in n:
        return "k_final3d"
    for k in ("k_pass2", "k_update", "k_ghost", "k_eta", "k_dt", "k_reset", "k_pick_dt"):
        if k in n:
            return k
    return None


_UNIT_SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0}


def load_capture(root: str, rel: str = CAPTURE):
    """Parse a profiles/*_summary.txt (`metric | unit | v1 | v2 ...`, header `metric | <kernel names>`) into
    {kernel key: {metric: value in base units}}.  Returns {} if the file is missing."""
    path = os.path.join(root, rel)
    try:
        lines = [l.rstrip("\n") for l in open(path)]
    except OSError:
        return {}
    keys, out = None, {}
    for l in lines:
        cells = [c.strip() for c in l.split("|")]
        if len(cells) < 3:
            continue
        if cells[0] == "metric" and keys is None:
            keys = [kernel_key(c) for c in cells[1:]]
            # the header has no unit column: metric | k1 | k2 ...
            for k in keys:
                if k:
                    out.setdefault(k, {})
            continue
        if keys is None:
            continue
        name, unit, vals = cells[0], cells[1], cells[2:]
        scale = _UNIT_SCALE.get(unit, 1.0)
        for k, v in zip(keys, vals):
            if not k:
                continue
            try:
                out[k][name] = float(v) * scale
            except ValueError:
                pass
    return out


def per_cell_counts(cap: dict):
    """{kernel: dict(inst, flops, fp64_pipe_inst, dram_bytes, pipe_pct, ncu_ms)} per real cell-update / per launch."""
    res = {}
    for k, m in cap.items():
        try:
            dadd = m["sm__sass_thread_inst_executed_op_dadd_pred_on.sum"]
            dmul = m["sm__sass_thread_inst_executed_op_dmul_pred_on.sum"]
            dfma = m["sm__sass_thread_inst_executed_op_dfma_pred_on.sum"]
        except KeyError:
            continue
        res[k] = {
            "inst": (dadd + dmul + dfma) / CAPTURE_N,
            "flops": (dadd + dmul + 2.0 * dfma) / CAPTURE_N,
            "fp64_pipe_inst": 32.0 * m.get("sm__inst_executed_pipe_fp64.sum", float("nan")) / CAPTURE_N,
            "warp_inst": m.get("sm__inst_executed.sum", float("nan")),                 # per launch at CAPTURE_N cells
            "fp64_warp_inst": m.get("sm__inst_executed_pipe_fp64.sum", float("nan")),
            "dram_bytes": m.get("dram__bytes_read.sum", float("nan")) + m.get("dram__bytes_write.sum", float("nan")),
            "pipe_pct": m.get("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
            "ncu_ms": m.get("gpu__time_duration.sum", float("nan")) * 1e3,
        }
    return res
