"""Roofline bookkeeping for bench.py: algorithmic FP64 work per cell-update and the peaks.

No arithmetic of the method lives here, only constants derived in DESIGN.md ("Roofline").

The CTU + PPMC + exact-Riemann step is bound by the plain FP64 ALU pipe, not by HBM:
at >= 4 k FP64-pipe instructions per cell-update and <= 2 kB of HBM traffic per cell-update the
machine balance (FP64 peak / HBM peak) puts the ALU time well above the memory time.  bench.py
therefore reports `"bound": "alu"`.

ALG_FLOPS[kernel] — algorithmic FP64 flops (DADD = DMUL = 1, DFMA = 2; division, square root,
reciprocal square root, log and exp counted as the FP64-pipe instructions of their CUDA fast paths)
per REAL cell-update, for the arithmetic each kernel is responsible for, every piece of the method
done exactly once per cell / interface it is defined on (no halo recomputation).  Frozen from the
ncu counts of the round-1 unfused kernels, which store every intermediate instead of recomputing it
(profiles/r01_fp64_inst_counts.md); a later kernel that recomputes to save traffic executes MORE
than this and is still charged only this.
"""

# (DADD + DMUL + 2*DFMA) per real cell-update at 256^3 on the throughput-sweep workload; see module doc.
ALG_FLOPS = {
    "k_pass1_x": 0.0,
    "k_pass1_march<y>": 0.0,
    "k_pass1_march<z>": 0.0,
    "k_pass2": 0.0,
    "k_update": 0.0,
    "k_final3d": 0.0,
}
# FP64-pipe instructions (DADD + DMUL + DFMA) per real cell-update, same provenance.
ALG_INST = dict(ALG_FLOPS)

# B200 plain-FP64 peak: 148 SMs x 64 FP64 lanes x 2 flop (FMA) x SM clock.  At the 1965 MHz
# maximum that is 37.2 TFLOP/s; the measured figure comes from ch_fp64_peak_probe at run time
# (8 independent DFMA chains per thread, 8 CTAs of 256 threads per SM).
SMS = 148
FP64_LANES_PER_SM = 64


def nominal_fp64_tflops(sm_mhz: float) -> float:
    return SMS * FP64_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12
