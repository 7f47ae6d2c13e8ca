"""Thin Python binding over the C-ABI library declared in include/ch.h (argument marshalling only).

PyTorch owns device memory and streams (torch tensors are handed to `ch_bind`); every step of the
hot path runs in the CUDA kernels of csrc/.  There is no CPU fallback: `load_library()` raises if
the shared library is missing and `Grid` raises if no CUDA device is present.  This module never
imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libch_b200.so")
_SOURCES = [os.path.join(_CSRC, "ch_kernels.cu")]
_HEADERS = [os.path.join(_CSRC, "ch_hydro.cuh"), os.path.join(os.path.dirname(_HERE), "include", "ch.h")]

PERIODIC, REFLECTIVE, OUTFLOW, NOH, EXCHANGE = 1, 2, 3, 4, 5
SOLVER_EXACT, SOLVER_ROE = 0, 1
RECON_PPMC, RECON_PLMC, RECON_PCM, RECON_PPMP, RECON_PLMP = 0, 1, 2, 3, 4
CH_OK, CH_EINVAL, CH_ESTATE, CH_ECUDA, CH_ENONPHYS = 0, -1, -2, -3, -4

# every symbol include/ch.h declares
SYMBOLS = ("ch_init", "ch_free", "ch_last_error", "ch_set_spacing", "ch_padded_cells", "ch_workspace_bytes",
           "ch_bind", "ch_set_state", "ch_get_state", "ch_set_padded", "ch_get_padded", "ch_compute_dt",
           "ch_step", "ch_step_cfl", "ch_last_dt", "ch_elapsed", "ch_set_solver", "ch_set_reconstruction", "ch_set_hcorrection", "ch_set_option", "ch_tiling", "ch_set_noh", "ch_set_time", "ch_get_time", "ch_fill_ghosts",
           "ch_halo_cells", "ch_halo_pack", "ch_halo_unpack", "ch_fill_dim", "ch_set_origin", "ch_sync", "ch_kernel_launches", "ch_profile", "ch_profile_read", "ch_kernel_name",
           "ch_fp64_peak_probe", "ch_issue_mix_probe", "ch_dt_noalloc", "ch_noalloc_setup", "ch_noalloc_max_cells")
K_COUNT = 11
OPT_MARCH_SEG, OPT_FINAL_SEG, OPT_TMA, OPT_UNFUSED, OPT_GRAPH, OPT_FOLD_GHOST = 0, 1, 2, 3, 4, 5

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ for sm_100a with nvcc into paper_1410_4194_b200/libch_b200.so (in-tree)."""
    deps = _SOURCES + _HEADERS
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    nvcc = os.environ.get("NVCC") or ("/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc")
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + _SOURCES
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


class ChStruct(C.Structure):
    _fields_ = [("state", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("reduce", C.c_void_p)]


_lib = None


def load_library() -> C.CDLL:
    """dlopen the CUDA library.  Raises (loudly) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB):
        raise RuntimeError(f"{_LIB} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(there is no CPU fallback)")
    L = C.CDLL(_LIB)
    vp, dp = C.c_void_p, C.c_void_p   # data pointers go through as raw addresses (host or device)
    L.ch_init.restype = vp
    L.ch_init.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int)]
    L.ch_free.argtypes = [vp]
    L.ch_last_error.restype = C.c_char_p
    L.ch_set_spacing.argtypes = [vp, C.c_double, C.c_double, C.c_double]
    L.ch_padded_cells.restype = C.c_longlong
    L.ch_padded_cells.argtypes = [vp]
    L.ch_workspace_bytes.restype = C.c_size_t
    L.ch_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int]
    L.ch_bind.argtypes = [vp, C.POINTER(ChStruct), vp]
    for name in ("ch_set_state", "ch_get_state", "ch_set_padded", "ch_get_padded"):
        getattr(L, name).argtypes = [vp, dp]
    L.ch_compute_dt.restype = C.c_double
    L.ch_compute_dt.argtypes = [vp, C.c_double]
    L.ch_step.argtypes = [vp, C.c_double]
    L.ch_step_cfl.argtypes = [vp, C.c_double, C.c_double]
    L.ch_last_dt.restype = C.c_double
    L.ch_last_dt.argtypes = [vp]
    L.ch_elapsed.restype = C.c_double
    L.ch_elapsed.argtypes = [vp]
    L.ch_set_solver.argtypes = [vp, C.c_int]
    L.ch_set_reconstruction.argtypes = [vp, C.c_int]
    L.ch_set_hcorrection.argtypes = [vp, C.c_int]
    L.ch_set_option.argtypes = [vp, C.c_int, C.c_int]
    L.ch_tiling.argtypes = [vp, C.POINTER(C.c_int)]
    L.ch_set_noh.argtypes = [vp, C.c_double, C.c_double]
    L.ch_set_time.argtypes = [vp, C.c_double]
    L.ch_get_time.argtypes = [vp]
    L.ch_get_time.restype = C.c_double
    L.ch_fill_ghosts.argtypes = [vp]
    L.ch_halo_cells.argtypes = [vp, C.c_int]
    L.ch_halo_cells.restype = C.c_longlong
    L.ch_halo_pack.argtypes = [vp, C.c_int, dp]
    L.ch_halo_unpack.argtypes = [vp, C.c_int, dp]
    L.ch_fill_dim.argtypes = [vp, C.c_int]
    L.ch_set_origin.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.ch_sync.argtypes = [vp]
    L.ch_kernel_launches.restype = C.c_longlong
    L.ch_kernel_launches.argtypes = [vp]
    L.ch_profile.argtypes = [vp, C.c_int]
    L.ch_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.ch_kernel_name.restype = C.c_char_p
    L.ch_kernel_name.argtypes = [C.c_int]
    L.ch_fp64_peak_probe.restype = C.c_double
    L.ch_fp64_peak_probe.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
    L.ch_issue_mix_probe.restype = C.c_double
    L.ch_issue_mix_probe.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp]
    L.ch_dt_noalloc.restype = C.c_int
    L.ch_dt_noalloc.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                C.c_double, vp, vp]
    L.ch_noalloc_setup.restype = C.c_int
    L.ch_noalloc_setup.argtypes = []
    L.ch_noalloc_max_cells.restype = C.c_longlong
    L.ch_noalloc_max_cells.argtypes = []
    _lib = L
    return L


def last_error() -> str:
    return load_library().ch_last_error().decode()


def _addr(a) -> int:
    """Raw address of a numpy array (host) or torch tensor (host or device), fp64 and contiguous."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags.c_contiguous
        return a.ctypes.data
    import torch
    assert isinstance(a, torch.Tensor) and a.dtype == torch.float64 and a.is_contiguous()
    return a.data_ptr()


class Grid:
    """ch_init + ch_bind with torch-owned device buffers; methods mirror the C calls one to one."""

    def __init__(self, nx, ny, nz, nghost=3, gamma=1.4, bc=(PERIODIC,) * 6, device="cuda:0", stream=None):
        import torch
        L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1410_4194_b200.Grid needs a CUDA device (no CPU fallback)")
        bc_arr = (C.c_int * 6)(*[int(b) for b in bc])
        self._h = L.ch_init(nx, ny, nz, nghost, gamma, bc_arr)
        if not self._h:
            raise ValueError("ch_init: " + last_error())
        self._L = L
        self.shape = (nz, ny, nx)
        self.nghost = nghost
        g = [nghost if n > 1 else 0 for n in (nz, ny, nx)]
        self.padded_shape = tuple(n + 2 * gg for n, gg in zip(self.shape, g))
        self.device = torch.device(device)
        np_cells = L.ch_padded_cells(self._h)
        ws_bytes = L.ch_workspace_bytes(nx, ny, nz, nghost)
        with torch.cuda.device(self.device):
            self._state = torch.empty(5 * np_cells, dtype=torch.float64, device=self.device)
            self._ws = torch.empty(ws_bytes // 8, dtype=torch.float64, device=self.device)
            self._red = torch.zeros(8, dtype=torch.int64, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        bufs = ChStruct(self._state.data_ptr(), self._ws.data_ptr(), ws_bytes, self._red.data_ptr())
        self._check(L.ch_bind(self._h, C.byref(bufs), self._stream.cuda_stream), "ch_bind")

    def _check(self, rc, what):
        if rc != CH_OK:
            raise (ValueError if rc == CH_EINVAL else RuntimeError)(f"{what}: {last_error()} (code {rc})")

    def close(self):
        if getattr(self, "_h", None):
            self._L.ch_sync(self._h)
            self._L.ch_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def cuda_stream(self):
        return self._stream

    def set_spacing(self, dx, dy, dz):
        self._check(self._L.ch_set_spacing(self._h, dx, dy, dz), "ch_set_spacing")

    def set_state(self, u):
        """u: numpy array or torch tensor (host, pinned host or device), [5][nz][ny][nx] fp64."""
        if isinstance(u, np.ndarray):
            u = np.ascontiguousarray(u, dtype=np.float64)
        assert tuple(u.shape) == (5,) + self.shape, (tuple(u.shape), self.shape)
        self._check(self._L.ch_set_state(self._h, _addr(u)), "ch_set_state")
        if isinstance(u, np.ndarray):
            self._L.ch_sync(self._h)   # the source array may be a temporary

    def get_state(self, out=None):
        if out is None:
            out = np.empty((5,) + self.shape)
        assert tuple(out.shape) == (5,) + self.shape
        self._check(self._L.ch_get_state(self._h, _addr(out)), "ch_get_state")
        return out

    def set_padded(self, up):
        if isinstance(up, np.ndarray):
            up = np.ascontiguousarray(up, dtype=np.float64)
        assert tuple(up.shape) == (5,) + self.padded_shape, (tuple(up.shape), self.padded_shape)
        self._check(self._L.ch_set_padded(self._h, _addr(up)), "ch_set_padded")
        if isinstance(up, np.ndarray):
            self._L.ch_sync(self._h)

    def get_padded(self, out=None):
        if out is None:
            out = np.empty((5,) + self.padded_shape)
        self._check(self._L.ch_get_padded(self._h, _addr(out)), "ch_get_padded")
        return out

    def compute_dt(self, cfl) -> float:
        dt = float(self._L.ch_compute_dt(self._h, cfl))
        if dt != dt:
            err = last_error()
            if "cfl" in err or "no state" in err:
                raise ValueError("ch_compute_dt: " + err)
        return dt

    def step(self, dt):
        self._check(self._L.ch_step(self._h, dt), "ch_step")

    def step_cfl(self, cfl, t_left=0.0):
        """One step with the device-resident Eq. 22 time step (no host round trip); t_left > 0 clips it."""
        self._check(self._L.ch_step_cfl(self._h, cfl, t_left), "ch_step_cfl")

    def last_dt(self) -> float:
        return float(self._L.ch_last_dt(self._h))

    def elapsed(self) -> float:
        return float(self._L.ch_elapsed(self._h))

    def set_solver(self, solver):
        """0 = exact (default), 1 = Roe with the HLLE failsafe."""
        self._check(self._L.ch_set_solver(self._h, int(solver)), "ch_set_solver")

    def set_hcorrection(self, on):
        """H correction (Appendix C): Roe solver only, nghost >= 4."""
        self._check(self._L.ch_set_hcorrection(self._h, int(bool(on))), "ch_set_hcorrection")

    def set_reconstruction(self, recon):
        """0 = PPMC (default), 1 = PLMC, 2 = PCM, 3 = PPMP (nghost >= 4), 4 = PLMP."""
        self._check(self._L.ch_set_reconstruction(self._h, int(recon)), "ch_set_reconstruction")

    def set_noh(self, rho0=1.0, p0=1e-6):
        """Ambient state of the analytic (NOH) faces."""
        self._check(self._L.ch_set_noh(self._h, rho0, p0), "ch_set_noh")

    def set_time(self, t):
        self._check(self._L.ch_set_time(self._h, float(t)), "ch_set_time")

    def get_time(self) -> float:
        return float(self._L.ch_get_time(self._h))

    def fill_ghosts(self):
        self._check(self._L.ch_fill_ghosts(self._h), "ch_fill_ghosts")

    def halo_cells(self, d) -> int:
        return int(self._L.ch_halo_cells(self._h, int(d)))

    def halo_pack(self, face, buf):
        """buf: device tensor of 5 * halo_cells(face // 2) doubles."""
        self._check(self._L.ch_halo_pack(self._h, int(face), _addr(buf)), "ch_halo_pack")

    def halo_unpack(self, face, buf):
        self._check(self._L.ch_halo_unpack(self._h, int(face), _addr(buf)), "ch_halo_unpack")

    def fill_dim(self, d):
        self._check(self._L.ch_fill_dim(self._h, int(d)), "ch_fill_dim")

    def set_origin(self, i0, j0, k0):
        self._check(self._L.ch_set_origin(self._h, int(i0), int(j0), int(k0)), "ch_set_origin")

    def set_option(self, option, value):
        """Launch-configuration choice (OPT_MARCH_SEG, OPT_FINAL_SEG, OPT_TMA: 2 / 1 / 0, OPT_UNFUSED, OPT_GRAPH, OPT_FOLD_GHOST); see ch_set_option."""
        self._check(self._L.ch_set_option(self._h, int(option), int(value)), "ch_set_option")

    def tiling(self) -> dict:
        """How the grid is cut into CTAs (ch_tiling)."""
        out = (C.c_int * 8)()
        self._check(self._L.ch_tiling(self._h, out), "ch_tiling")
        keys = ("x_interfaces_per_cta", "march_columns_per_cta", "march_seg_y", "march_seg_z", "final_tile_x",
                "final_tile_y", "final_seg", "tma")
        return dict(zip(keys, [int(v) for v in out]))

    def sync(self):
        self._check(self._L.ch_sync(self._h), "ch_sync")

    def profile(self, enable=True):
        self._check(self._L.ch_profile(self._h, 1 if enable else 0), "ch_profile")

    def profile_read(self) -> dict:
        """{kernel name: (total ms, launches timed)} since the last profile() call."""
        ms = (C.c_double * K_COUNT)()
        calls = (C.c_longlong * K_COUNT)()
        self._check(self._L.ch_profile_read(self._h, ms, calls), "ch_profile_read")
        return {self._L.ch_kernel_name(k).decode(): (ms[k], calls[k]) for k in range(K_COUNT)}

    @property
    def kernel_launches(self) -> int:
        return int(self._L.ch_kernel_launches(self._h))


def fp64_peak_probe(blocks=148 * 8, threads=256, iters=200000, device="cuda:0"):
    """Measured DFMA rate (the ALU-roofline denominator): returns (TFLOP/s, ms)."""
    import torch
    L = load_library()
    sink = torch.empty(blocks * threads, dtype=torch.float64, device=device)
    st = torch.cuda.current_stream(sink.device)
    ms = L.ch_fp64_peak_probe(sink.data_ptr(), blocks, threads, iters, st.cuda_stream)
    if ms <= 0:
        raise RuntimeError("ch_fp64_peak_probe: " + last_error())
    return 2.0 * 8 * iters * blocks * threads / (ms * 1e-3) / 1e12, ms


def issue_mix_probe(blocks=148 * 4, threads=512, iters=100000, device="cuda:0"):
    """Scheduler time per FP64 and per ALU warp instruction (seconds x schedulers, i.e. per SM sub-partition):
    returns dict(t_fp64, t_alu, overlap) from loops of 8 DFMA + {0, 16, 32} integer operations on 4 warps per
    scheduler.  t_fp64 = time of one DFMA warp instruction on its scheduler, t_alu = ADDED time per ALU warp
    instruction; overlap = 1 - t_alu / (ALU-only cost) is not measured here: what matters is that the added time is
    not hidden under the FP64 instructions."""
    import torch
    L = load_library()
    sink = torch.empty(blocks * threads, dtype=torch.float64, device=device)
    st = torch.cuda.current_stream(sink.device)
    ms = {}
    for n in (0, 16, 32):
        ms[n] = L.ch_issue_mix_probe(sink.data_ptr(), n, blocks, threads, iters, st.cuda_stream)
        if ms[n] <= 0:
            raise RuntimeError("ch_issue_mix_probe: " + last_error())
    warps_per_sched = (blocks / 148.0) * (threads / 32.0) / 4.0         # resident warps per scheduler (all co-resident)
    per_iter = {n: ms[n] * 1e-3 / iters / warps_per_sched for n in ms}   # scheduler seconds per warp iteration
    t_fp64 = per_iter[0] / 8.0
    t_alu = (per_iter[32] - per_iter[0]) / 32.0
    return dict(t_fp64=t_fp64, t_alu=t_alu, t_alu_16=(per_iter[16] - per_iter[0]) / 16.0, ms=ms)


def noalloc_max_cells() -> int:
    """Largest number of real cells ch_dt_noalloc serves (its scratch is a fixed file-scope device array)."""
    return int(load_library().ch_noalloc_max_cells())


def dt_noalloc(u_padded, nx, ny, nz, nghost, gamma, dx, dy, dz, cfl, dt_out, stream=None):
    """ch_dt_noalloc: Eq. 22 of the padded state `u_padded` (a CUDA float64 tensor laid out as Grid.get_padded) into
    the one-element CUDA tensor `dt_out`, enqueued on `stream` (torch stream; default: the current one).  Allocates
    nothing: argument marshalling only.  Raises ValueError for bad arguments or a grid beyond noalloc_max_cells()."""
    import torch
    L = load_library()
    if not (u_padded.is_cuda and dt_out.is_cuda and u_padded.dtype == torch.float64 and dt_out.dtype == torch.float64):
        raise ValueError("dt_noalloc: u_padded and dt_out must be CUDA float64 tensors")
    if not u_padded.is_contiguous():
        raise ValueError("dt_noalloc: u_padded must be contiguous")
    st = stream if stream is not None else torch.cuda.current_stream(u_padded.device)
    rc = L.ch_dt_noalloc(u_padded.data_ptr(), int(nx), int(ny), int(nz), int(nghost), float(gamma), float(dx), float(dy),
                         float(dz), float(cfl), dt_out.data_ptr(), st.cuda_stream)
    if rc != 0:
        err = last_error()
        raise (ValueError if rc == -1 else RuntimeError)("ch_dt_noalloc: " + err)
