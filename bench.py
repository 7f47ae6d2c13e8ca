#!/usr/bin/env python
"""bench.py — cell-updates/s of the full CTU + PPMC + exact-Riemann step (fp64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size 512] [--impl reference]

A "step" is one pass of the whole hot path over the grid: `dt = ch_compute_dt(cfl)` (Eq. 22) then
`ch_step(dt)` (PPMC + exact Riemann in x, y, z; transverse correction; second Riemann pass; update;
ghost fill).  Workload: BASELINE.json's throughput-sweep configuration (periodic box, gamma = 5/3,
seeded sum of 8 random-phase sinusoids) at `--size`^3 (default 512, the largest size the metric is
quoted on; 128^3, 256^3 and 384^3 are reported beside it under "other_sizes").  The state (5.6 GB at 512^3) is far
larger than the 126 MB L2, so no L2 flush is needed between steps.

N > 1 (torchrun): the path does not shard in this build ("replicas only"): every rank
steps its own replica with no data-path collective; value = all ranks' cell-updates / max-over-ranks
time.

`--impl reference`: the oracle (oracle/, plain C++ on the host cores) on a bounded sample of the
same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/sec (fp64 CTU+PPM+exact Riemann)"
UNIT = "cell-updates/s"
CPU_SAMPLE_N = 128          # the oracle is timed on a 128^3 corner of the workload (and on a 256^3 one, all cores)
ORACLE_FLAGS = "g++ -std=c++17 -O2 -ffp-contract=off -fopenmp (oracle/ref.py)"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--size", type=int, default=512)
    ap.add_argument("--other-sizes", type=str, default="128,256,384")
    ap.add_argument("--impl", type=str, default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-workloads", action="store_true")
    ap.add_argument("--solver", type=str, default="exact", choices=["exact", "roe"],
                    help="Riemann solver of the main measured workload (default: the metric's exact solver)")
    ap.add_argument("--recon", type=str, default="ppmc", choices=["ppmc", "plmc", "pcm"],
                    help="reconstruction of the main measured workload (default: the metric's PPM)")
    ap.add_argument("--hcorr", action="store_true",
                    help="main workload with the H correction of Appendix C (implies --solver roe and four ghost layers)")
    return ap.parse_args()


# ---- clocks ---------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, power, reasons = [], [], [], set()
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(power))
        return out


# ---- the oracle arm ---------------------------------------------------------------------------------
def corner_sample(w, m):
    """A bounded sample of the workload: the m^3 corner of its initial state, outflow faces, the
    workload's own cell width."""
    import numpy as np
    return np.ascontiguousarray(w.u[:, :m, :m, :m])


def host_cores():
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def set_oracle_threads(n):
    """Thread count of the oracle's OpenMP loops, set through the OpenMP runtime the oracle library links (the
    oracle itself is untouched).  Returns the count in force."""
    import ctypes
    from oracle import ref
    ref.lib()                                   # make sure libgomp is loaded by the oracle first
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(int(n))
        return int(gomp.omp_get_max_threads())
    except OSError:
        return None


def time_oracle(w, steps, warmup, m=CPU_SAMPLE_N, threads=None):
    from oracle import ref
    from paper_1410_4194_b200 import workloads as wl
    nx = w.shape[0]
    m = min(m, nx)
    u = corner_sample(w, m)
    cores = host_cores()
    omp = os.environ.get("OMP_NUM_THREADS")
    if omp:
        cores = min(cores, int(omp))
    if threads is not None:
        got = set_oracle_threads(threads)
        cores = got if got is not None else cores
    G = ref.RefGrid(m, m, m, 3, w.gamma, (wl.OUTFLOW,) * 6)
    G.set_spacing(1.0 / nx, 1.0 / nx, 1.0 / nx)
    G.set_state(u)
    for _ in range(warmup):
        G.step(G.compute_dt(w.cfl))
    t0 = time.perf_counter()
    for _ in range(steps):
        G.step(G.compute_dt(w.cfl))
    el = time.perf_counter() - t0
    del G
    return dict(value=m ** 3 * steps / el, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{m}^3 corner of the {nx}^3 sweep initial state (outflow faces, dx=1/{nx}), "
                       f"{steps} steps of compute_dt+step after {warmup} warm-up, OpenMP over the outer loops, "
                       f"{cores} thread(s)",
                ms_per_step=el / steps * 1e3, per_core=m ** 3 * steps / el / max(cores, 1))


def oracle_legs(w):
    """SURVEY.md section 8(d) "Oracle timing": (i) one thread, 128^3, 3 steps; (ii) all host cores, 128^3 x 10 steps and
    256^3 x 2 steps.  The oracle as it stands; bit-identical at any thread count (no floating-point reduction)."""
    n_all = host_cores()
    legs = []
    for label, m, steps, warm, thr in (("single thread 128^3 x 3", 128, 3, 0, 1),
                                       ("all cores 128^3 x 10", 128, 10, 1, n_all),
                                       ("all cores 256^3 x 2", 256, 2, 0, n_all)):
        if m > w.shape[0]:
            continue
        r = time_oracle(w, steps, warm, m=m, threads=thr)
        legs.append({"leg": label, "value": r["value"], "unit": UNIT, "per_core": r["per_core"], "cores": r["cores"],
                     "ms_per_step": r["ms_per_step"], "sample": r["sample"]})
    set_oracle_threads(n_all)
    return legs


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1410_4194_b200 import workloads as wl
    w = wl.sweep(args.size)
    r = time_oracle(w, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"throughput sweep (BASELINE.json config 5), {CPU_SAMPLE_N}^3 corner sample per step",
                       "gamma": w.gamma, "cfl": w.cfl, "bc": "outflow (sample faces)"},
            "cpu_baseline": dict({k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
                                 cpu_model=cpu_model(), nproc=host_cores(), build=ORACLE_FLAGS),
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- the CUDA arm -----------------------------------------------------------------------------------
def timed_steps(G, cfl, steps, stream_events):
    """K steps of compute_dt + step, timed with CUDA events on the library's stream."""
    import torch
    e0, e1 = stream_events
    torch.cuda.synchronize()
    e0.record(G.cuda_stream)
    for _ in range(steps):
        G.step(G.compute_dt(cfl))
    e1.record(G.cuda_stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3


def bench_size(pkg, wl, n, steps, warmup, device, dist=None, profile=True, e2e=True, solver=0, recon=0, hcorr=False):
    import numpy as np
    import torch
    from paper_1410_4194_b200.driver import max_over_ranks
    w = wl.sweep(n)
    N = n ** 3
    G = pkg.Grid(n, n, n, 4 if hcorr else 3, w.gamma, w.bc, device=device)
    G.set_solver(solver)
    G.set_reconstruction(recon)
    if hcorr:
        G.set_hcorrection(True)
    u_dev = torch.from_numpy(w.u).to(device)
    G.set_state(u_dev)
    ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    for _ in range(max(warmup, 3)):
        G.step(G.compute_dt(w.cfl))
    n0 = G.kernel_launches
    if dist is not None:
        dist.barrier()
    el = timed_steps(G, w.cfl, steps, ev)
    launches = G.kernel_launches - n0
    if dist is not None:
        el = max_over_ranks(el, dist, device)
        dist.barrier()
    out = dict(n=n, seconds=el, launches=launches, cells=N, gamma=w.gamma, cfl=w.cfl)
    # the same steps queued through ch_step_cfl (dt stays on the device, the kernels of a step replayed as one graph)
    for _ in range(3):
        G.step_cfl(w.cfl)
    torch.cuda.synchronize()
    ev[0].record(G.cuda_stream)
    for _ in range(steps):
        G.step_cfl(w.cfl)
    ev[1].record(G.cuda_stream)
    torch.cuda.synchronize()
    out["step_cfl_seconds"] = ev[0].elapsed_time(ev[1]) * 1e-3
    if profile:
        # same K steps again with an event pair around every kernel (ch_profile): per-kernel durations
        G.profile(True)
        for _ in range(steps):
            G.step(G.compute_dt(w.cfl))
        prof = G.profile_read()
        G.profile(False)
        out["kernels"] = {k: {"ms_avg": ms / c, "launches_per_step": c / steps}
                          for k, (ms, c) in prof.items() if c}
        out["kernel_ms_per_step"] = sum(ms for ms, c in prof.values()) / steps
    if e2e:
        # the user's call sequence with HOST buffers: H2D of the state, dt, step, D2H of the result
        k_e2e = max(1, min(steps, 5))
        h_in = torch.from_numpy(w.u).pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        G.set_state(h_in); G.step(G.compute_dt(w.cfl)); G.get_state(h_out)       # warm-up
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            G.set_state(h_in)
            G.step(G.compute_dt(w.cfl))
            G.get_state(h_out)                                                  # synchronises
        t_e2e = time.perf_counter() - t0
        if dist is not None:
            t_e2e = max_over_ranks(t_e2e, dist, device)
        out["e2e"] = dict(seconds=t_e2e, steps=k_e2e, h2d=h_in.numel() * 8, d2h=h_out.numel() * 8)
        assert bool(torch.isfinite(h_out).all())
        del h_in, h_out
    G.close()
    del G, u_dev
    torch.cuda.empty_cache()
    return out, w


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_1410_4194_b200 as pkg
    from paper_1410_4194_b200 import roofline as rf
    from paper_1410_4194_b200 import workloads as wl
    from paper_1410_4194_b200.binding import fp64_peak_probe, issue_mix_probe

    pkg.load_library()                      # no CPU fallback: raises if the CUDA library is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    device = f"cuda:{local}"

    sampler = ClockSampler(local) if rank == 0 else None
    peak_tf, _ = fp64_peak_probe(device=device)                 # measured DFMA rate, burst
    mix = issue_mix_probe(device=device)                        # scheduler time per FP64 / per other warp instruction
    if args.hcorr:
        args.solver = "roe"
    solver = {"exact": 0, "roe": 1}[args.solver]
    recon = {"ppmc": 0, "plmc": 1, "pcm": 2}[args.recon]
    default_method = solver == 0 and recon == 0 and not args.hcorr
    main_res, w = bench_size(pkg, wl, args.size, args.steps, args.warmup, device, dist,
                             profile=True, e2e=not args.no_e2e, solver=solver, recon=recon, hcorr=args.hcorr)
    clocks = sampler.stop() if sampler else None
    others = {}
    if world == 1:
        for s in [int(x) for x in args.other_sizes.split(",") if x]:
            if s != args.size:
                r, _ = bench_size(pkg, wl, s, args.steps, args.warmup, device, None, profile=False, e2e=False,
                                  solver=solver, recon=recon, hcorr=args.hcorr)
                others[str(s)] = {"value": r["cells"] * args.steps / r["seconds"], "unit": UNIT,
                                  "ms_per_step": r["seconds"] / args.steps * 1e3,
                                  "ch_step_cfl": {"value": r["cells"] * args.steps / r["step_cfl_seconds"], "unit": UNIT,
                                                  "ms_per_step": r["step_cfl_seconds"] / args.steps * 1e3}}
    other_wl = {}
    if world == 1 and not args.no_other_workloads:
        # strong shocks change Newton iteration counts and warp divergence: the smooth sweep alone flatters the
        # solver, so configs 3 and 4 are timed beside it (state after `pre` steps)
        for name, make, pre, k in (("kelvin_helmholtz_256x256 (config 2)", lambda: wl.kelvin_helmholtz(256), 20, 50),
                                   ("sedov_128 (config 3)", lambda: wl.sedov(128), 20, 20),
                                   ("shock_cloud_256 (config 4)", lambda: wl.shock_cloud(256), 10, 10)):
            ww = make()
            G = pkg.Grid(*ww.shape, 3, ww.gamma, ww.bc, device=device)
            G.set_state(torch.from_numpy(ww.u).to(device))
            for _ in range(pre):
                G.step(G.compute_dt(ww.cfl))
            ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            sec = timed_steps(G, ww.cfl, k, ev)
            other_wl[name] = {"value": ww.u[0].size * k / sec, "unit": UNIT, "ms_per_step": sec / k * 1e3,
                              "steps": k, "after_steps": pre}
            # the same steps queued through ch_step_cfl (dt stays on the device: no per-step read-back; graph replay
            # from the third call on, so three untimed calls first)
            for _ in range(3):
                G.step_cfl(ww.cfl)
            torch.cuda.synchronize()
            ev[0].record(G.cuda_stream)
            for _ in range(k):
                G.step_cfl(ww.cfl)
            ev[1].record(G.cuda_stream)
            torch.cuda.synchronize()
            sec2 = ev[0].elapsed_time(ev[1]) * 1e-3
            other_wl[name]["ch_step_cfl"] = {"value": ww.u[0].size * k / sec2, "unit": UNIT, "ms_per_step": sec2 / k * 1e3}
            G.close()
            del G
            torch.cuda.empty_cache()
    if world == 1 and not args.no_other_workloads:
        # the paper's other method choices on the same workload and size: the Roe + HLLE solver (B.2)
        # with PPMC, and the second-order pair PLMC + Roe the paper quotes its 2-D figure for
        for label, solver, recon, hc in ((f"sweep_{args.size} PPMC + Roe/HLLE", 1, 0, False),
                                         (f"sweep_{args.size} PLMC + Roe/HLLE", 1, 1, False),
                                         (f"sweep_{args.size} PPMC + Roe/HLLE + H correction (4 ghost layers, k_eta + fused second half)", 1, 0, True),
                                         (f"sweep_{args.size} PPMP + exact (4 ghost layers)", 0, 3, False),
                                         (f"sweep_{args.size} PLMP + exact", 0, 4, False)):
            G = pkg.Grid(args.size, args.size, args.size, 4 if (hc or recon == 3) else 3, w.gamma, w.bc, device=device)
            G.set_solver(solver)
            G.set_reconstruction(recon)
            G.set_hcorrection(hc)
            G.set_state(torch.from_numpy(w.u).to(device))
            for _ in range(3):
                G.step(G.compute_dt(w.cfl))
            ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            k = max(1, min(args.steps, 10))
            sec = timed_steps(G, w.cfl, k, ev)
            other_wl[label] = {"value": args.size ** 3 * k / sec, "unit": UNIT, "ms_per_step": sec / k * 1e3, "steps": k}
            G.close()
            del G
            torch.cuda.empty_cache()
    if world == 1 and not args.no_other_workloads:
        # the same box cut into 2 x 2 x 2 blocks, all on this GPU: eight contexts, halo slabs through
        # ch_halo_pack / ch_halo_unpack in x -> y -> z order, dt = min over the blocks; what the decomposition costs
        # before any link is involved (results bitwise equal to the undivided grid: tests/test_gpu_decomp.py)
        from paper_1410_4194_b200 import decomp
        B = decomp.BlockGrid((args.size,) * 3, (2, 2, 2), 3, w.gamma, w.bc,
                             lambda nx, ny, nz, g, gamma, bc, dev: pkg.Grid(nx, ny, nz, g, gamma, bc, device=dev), devices=device)
        B.set_spacing(1.0 / args.size, 1.0 / args.size, 1.0 / args.size)
        B.set_state(w.u)
        for _ in range(3):
            B.step(B.compute_dt(w.cfl))
        k = max(1, min(args.steps, 10))
        ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
        torch.cuda.synchronize()
        ev[0].record(B.grids[0].cuda_stream)
        for _ in range(k):
            B.step(B.compute_dt(w.cfl))
        ev[1].record(B.grids[0].cuda_stream)
        torch.cuda.synchronize()
        sec = ev[0].elapsed_time(ev[1]) * 1e-3
        other_wl[f"sweep_{args.size} as 2x2x2 blocks on one GPU (block decomposition, halo exchange on the device)"] = {
            "value": args.size ** 3 * k / sec, "unit": UNIT, "ms_per_step": sec / k * 1e3, "steps": k,
            "halo_messages_per_step": 48}
        B.close()
        del B
        torch.cuda.empty_cache()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    N, K = main_res["cells"], args.steps
    value = world * N * K / main_res["seconds"]
    # Rooflines as SURVEY.md section 8(d) defines them (paper_1410_4194_b200/roofline.py): the slower of the METHOD's
    # bytes (80 B x ghost factor per cell-update) over the measured copy bandwidth and the FP64 arithmetic
    # instructions (from the committed ncu capture) over the DFMA instruction rate measured in this run.
    kern = main_res["kernels"]
    hbm_gbs, hbm_src = rf.hbm_peak_gbs(ROOT)
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    cap = rf.per_cell_counts(rf.load_capture(ROOT)) if default_method else {}
    ghost = (args.size + 6) ** 3 / args.size ** 3
    dfma_rate = peak_tf * 1e12 / 2.0                                    # FP64 instructions / s
    method_bytes = rf.METHOD_BYTES_PER_CELL * ghost
    capture_applies = default_method and args.size == 512 and bool(cap)
    per_kernel, inst_step, issue_step = {}, 0.0, 0.0
    for k, v in kern.items():
        if k not in rf.DECOMPOSITION_BYTES:
            continue
        t = v["ms_avg"] * 1e-3
        c = cap.get(k)
        # bytes of the method this kernel touches: pass 1 reads u^n; the last kernel reads u^n and writes u^{n+1}
        mb = method_bytes if k == "k_final3d" else 0.5 * method_bytes
        t_h = mb * N / (hbm_gbs * 1e9)
        t_a = c["inst"] * N / dfma_rate if c else 0.0
        inst_step += (c["inst"] if c else 0.0) * v["launches_per_step"]
        dec = rf.DECOMPOSITION_BYTES[k]
        # issue ceiling of this kernel's own instruction mix (counts from the capture, scaled to this grid)
        t_i = None
        if c and c["warp_inst"] == c["warp_inst"]:
            scale = N / rf.CAPTURE_N
            t_i = scale * (c["fp64_warp_inst"] * mix["t_fp64"] + (c["warp_inst"] - c["fp64_warp_inst"]) * mix["t_alu"]) / (rf.SMS * 4)
            issue_step += t_i * v["launches_per_step"]
        per_kernel[k] = {"ms": v["ms_avg"], "bound": "hbm" if t_h >= t_a else "alu",
                         "roofline_ms": max(t_h, t_a) * 1e3, "frac": max(t_h, t_a) / t,
                         "method_bytes_per_cell": mb, "fp64_inst_per_cell": c["inst"] if c else None,
                         "fp64_flops_per_cell": c["flops"] if c else None,
                         "fp64_TFLOPs": c["flops"] * N / t / 1e12 if c else None,
                         "fp64_pipe_inst_per_cell_incl_compares": c["fp64_pipe_inst"] if c else None,
                         "ncu_sm__pipe_fp64_cycles_active_pct": c["pipe_pct"] if c else None,
                         "ncu_ms": c["ncu_ms"] if c else None,
                         "issue_ceiling_ms": t_i * 1e3 if t_i else None, "issue_frac": t_i / t if t_i else None,
                         "decomposition_bytes_per_cell": dec,
                         "hbm_utilisation_of_decomposition": dec * N / t / 1e9 / hbm_gbs,
                         "traffic": c["dram_bytes"] if (c and capture_applies) else None}
    top = max(per_kernel, key=lambda k: kern[k]["ms_avg"] * kern[k]["launches_per_step"])
    pk = per_kernel[top]
    step_ms = main_res["seconds"] / K * 1e3
    t_h_step, t_a_step = method_bytes * N / (hbm_gbs * 1e9), inst_step * N / dfma_rate
    if pk["bound"] == "hbm":
        ach, peak, unit, psrc = pk["method_bytes_per_cell"] * N / (pk["ms"] * 1e-3) / 1e9, hbm_gbs, "GB/s", hbm_src
    else:
        # every FP64 instruction counted as one FMA slot (2 flop), exactly as the DFMA peak counts its own
        ach, peak, unit = 2.0 * pk["fp64_inst_per_cell"] * N / (pk["ms"] * 1e-3) / 1e12, peak_tf, "TFLOP/s"
        psrc = ("measured: ch_fp64_peak_probe DFMA chains in this run (burst); nominal 148 SM x 64 lanes x 2 x "
                f"{sm_mhz:.0f} MHz = {rf.nominal_fp64_tflops(sm_mhz):.1f}")
    roofline = {"bound": pk["bound"], "kernel": top, "achieved": ach, "peak": peak, "unit": unit,
                "frac": ach / peak, "traffic": pk["traffic"],
                "definition": "SURVEY.md 8(d): max(80 B x Np/N per cell-update / hbm_gbs, FP64 arithmetic instructions per "
                              "cell-update / measured DFMA instruction rate) / measured kernel time; 'achieved' counts "
                              "every FP64 instruction as one FMA slot (2 flop) as the DFMA peak does",
                "capture": rf.CAPTURE if cap else None,
                "capture_note": "per-cell instruction counts, DRAM traffic and pipe utilisation are read from this ncu "
                                "--set full capture (512^3, kernels of this commit); traffic only when this run is the "
                                "captured configuration",
                "peak_source": psrc,
                "kernel_ms": kern[top]["ms_avg"],
                "kernel_share_of_step": kern[top]["ms_avg"] * kern[top]["launches_per_step"] / main_res["kernel_ms_per_step"],
                "issue_mix_probe": {"t_fp64_scheduler_ns": mix["t_fp64"] * 1e9, "t_other_scheduler_ns": mix["t_alu"] * 1e9,
                                    "t_other_16_scheduler_ns": mix["t_alu_16"] * 1e9, "ms": mix["ms"],
                                    "note": "loops of 8 DFMA + {0,16,32} integer ops on 16 warps per scheduler (ch_issue_mix_probe): "
                                            "an FP64 warp instruction costs t_fp64 of its scheduler, every other one t_other ON TOP "
                                            "(no overlap); issue_ceiling = (F t_fp64 + O t_other) / 592 with F, O from the capture"},
                "issue_ceiling_ms": pk["issue_ceiling_ms"], "issue_frac": pk["issue_frac"],
                "fp64_peak_TFLOPs_measured": peak_tf, "fp64_inst_rate_measured": dfma_rate, "hbm_peak_GBps": hbm_gbs,
                "ghost_factor": ghost,
                "step": {"method_bytes_per_cell": method_bytes, "fp64_inst_per_cell": inst_step or None,
                         "hbm_ms": t_h_step * 1e3, "fp64_ms": t_a_step * 1e3,
                         "bound": "hbm" if t_h_step >= t_a_step else "alu",
                         "roofline_ms": max(t_h_step, t_a_step) * 1e3, "measured_ms": step_ms,
                         "frac": max(t_h_step, t_a_step) * 1e3 / step_ms,
                         "issue_ceiling_ms": issue_step * 1e3 or None, "issue_frac": issue_step * 1e3 / step_ms if issue_step else None,
                         "decomposition_bytes_per_cell": sum(rf.DECOMPOSITION_BYTES[k] for k in per_kernel),
                         "hbm_utilisation_of_decomposition":
                             sum(rf.DECOMPOSITION_BYTES[k] for k in per_kernel) * N / (step_ms * 1e-3) / 1e9 / hbm_gbs},
                "kernels": per_kernel, "kernel_times": kern}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": main_res["seconds"] / K * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"throughput sweep (BASELINE.json config 5) {args.size}^3 periodic, "
                                   "sum of 8 seeded sinusoids, 1 replica per GPU",
                       "gamma": w.gamma, "cfl": w.cfl, "nghost": 4 if args.hcorr else 3, "h_correction": bool(args.hcorr), "l2": "state (5 fields) larger than L2, no flush",
                       "reconstruction": args.recon, "riemann_solver": args.solver,
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "gpu_launches": main_res["launches"], "clocks": clocks, "roofline": roofline}
    line["ch_step_cfl"] = {"value": world * N * K / main_res["step_cfl_seconds"], "unit": UNIT,
                           "ms_per_step": main_res["step_cfl_seconds"] / K * 1e3,
                           "note": "optional sixth call: Eq. 22 finished on the device, steps queued without the read-back, graph replay"}
    if others:
        line["other_sizes"] = others
    if other_wl:
        line["other_workloads"] = other_wl
    if "e2e" in main_res:
        e = main_res["e2e"]
        line["e2e"] = {"value": world * N * e["steps"] / e["seconds"], "unit": UNIT,
                       "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"], "steps": e["steps"],
                       "how": "ch_set_state(pinned host) + ch_compute_dt + ch_step + ch_get_state(pinned host) per step"}
    if world == 1 and not args.no_cpu_baseline:
        legs = oracle_legs(w)
        head = next(l for l in legs if l["leg"].startswith("all cores 128"))
        line["cpu_baseline"] = {"value": head["value"], "unit": UNIT, "cores": head["cores"], "kind": "oracle",
                                "sample": head["sample"], "cpu_model": cpu_model(), "nproc": host_cores(),
                                "build": ORACLE_FLAGS, "legs": legs}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
