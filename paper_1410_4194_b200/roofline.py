"""Roofline bookkeeping for bench.py: algorithmic work per cell-update and the peaks.

No arithmetic of the method lives here, only constants derived in DESIGN.md §6 ("Roofline").

Two ceilings bound every kernel of the step (north_star: "the slower of the two"):

* HBM: ALG_BYTES[kernel] = bytes per REAL cell-update the kernel must move given the step's
  decomposition into kernels (every array it consumes read once, every array it produces written
  once, no halo re-reads) — against MEASURED_PEAKS.json's copy bandwidth;
* FP64 ALU: ALG_FLOPS[kernel] = FP64 flops (DADD = DMUL = 1, DFMA = 2) per real cell-update, every
  piece of the method done exactly once per cell / interface it is defined on (no halo
  recomputation) — against the DFMA rate measured in the same run (ch_fp64_peak_probe).

ALG_FLOPS / ALG_INST were frozen from the ncu thread-level counts
(sm__sass_thread_inst_executed_op_{dadd,dmul,dfma}_pred_on.sum) of the kernels that compute each
piece once with the present arithmetic, divided by 512^3: k_pass1_* from
profiles/r01f_full_512_summary.txt, and the unfused k_pass2 + k_update (CH_UNFUSED=1,
profiles/r01f_unfused_counts.csv) for the second half.  k_final3d recomputes halo lanes / rows
(32/30 x 12/10) and is still charged only the unfused count.  Re-freeze whenever ch_hydro.cuh changes.
"""

# bytes per real cell-update (fp64 = 8 B): pass 1 reads u (5) and writes U*_L, U*_R, F* (15);
# the fused second half reads U*_L, U*_R of three directions (30), F* (15) and u (5), writes u (5).
ALG_BYTES = {
    "k_pass1_x": 160.0,
    "k_pass1_march<y>": 160.0,
    "k_pass1_march<z>": 160.0,
    "k_final3d": 440.0,
}

# (DADD + DMUL + 2*DFMA) per real cell-update at 512^3, throughput-sweep workload.
ALG_FLOPS = {
    "k_pass1_x": 580.4,
    "k_pass1_march<y>": 561.4,   # r01f count 586.4 minus the A20 interface value now computed once per interface
    "k_pass1_march<z>": 561.5,   # (5 components x 5 flops), not re-profiled
    "k_final3d": 1030.0,      # k_pass2 (929.0) + k_update (101.0) of the unfused path
}

# FP64-pipe arithmetic instructions (DADD + DMUL + DFMA) per real cell-update, same provenance.
ALG_INST = {
    "k_pass1_x": 442.3,
    "k_pass1_march<y>": 426.9,
    "k_pass1_march<z>": 426.9,
    "k_final3d": 731.4,
}

# B200 plain-FP64 peak: 148 SMs x 64 FP64 lanes x 2 flop (FMA) x SM clock.  At the 1965 MHz
# maximum that is 37.2 TFLOP/s; the measured figure comes from ch_fp64_peak_probe at run time
# (8 independent DFMA chains per thread, 8 CTAs of 256 threads per SM).
SMS = 148
FP64_LANES_PER_SM = 64
HBM_FALLBACK_GBS = 6453.1     # MEASURED_PEAKS.json on this pool (used only if the file is absent)


def nominal_fp64_tflops(sm_mhz: float) -> float:
    return SMS * FP64_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def hbm_peak_gbs(root: str):
    """(GB/s, source) — the driver-written measured copy bandwidth if present."""
    import json
    import os
    p = os.path.join(root, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst copy bandwidth)"
    except (OSError, KeyError, ValueError):
        return HBM_FALLBACK_GBS, "fallback: MEASURED_PEAKS.json absent, last driver-measured value for this pool"
