"""Thin Python binding of the C-ABI library (include/ising.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C entry points; this module
turns numpy arrays (host memory) and torch CUDA tensors (device memory) into pointers and
sizes, provides the workspace as a torch uint8 tensor, and passes torch's current stream.
The function names are those of the C ABI.  There is no CPU fallback: a missing library or a
missing B200 raises.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

from . import build as _build

ISING_MODE_GS, ISING_MODE_JACOBI, ISING_MODE_RACY, ISING_MODE_EXACT_N = 0, 1, 2, 3
ISING_TIE_MINUS, ISING_TIE_KEEP = 0, 1
ISING_INIT_PHILOX, ISING_INIT_GIVEN, ISING_INIT_CONTINUE = 0, 1, 2
ISING_W_INT8, ISING_W_INT32 = 1, 4
ISING_LOAD_DEFAULT, ISING_LOAD_NO_DENSE = 0, 1
ISING_LOAD_NO_SMALL, ISING_LOAD_NO_CLUSTER, ISING_LOAD_NO_TAIL_CHAIN, ISING_LOAD_NO_OVERLAP = 2, 4, 8, 16
# ising_problem_info(13): the Gauss-Seidel engine of a loaded problem
ENGINE_PER_PHASE, ENGINE_GRID, ENGINE_CLUSTER, ENGINE_GRID_TAIL_CHAIN, ENGINE_SMALL = 0, 1, 2, 3, 4

STATUS_NAMES = {
    0: "ISING_OK", 1: "ISING_ERR_NULL_ARG", 2: "ISING_ERR_BAD_SHAPE", 3: "ISING_ERR_UNSORTED_OR_DUP",
    4: "ISING_ERR_SELF_LOOP", 5: "ISING_ERR_ASYMMETRIC", 6: "ISING_ERR_BAD_COLOURING",
    7: "ISING_ERR_FIELD_OVERFLOW", 8: "ISING_ERR_TOO_MANY_REPLICAS", 9: "ISING_ERR_WORKSPACE_TOO_SMALL",
    10: "ISING_ERR_NO_COLOURING_FOR_GS", 11: "ISING_ERR_UNSUPPORTED_DEVICE", 12: "ISING_ERR_CUDA",
    13: "ISING_ERR_BAD_SPINS", 14: "ISING_ERR_NO_STATE",
}

_vp, _i32, _i64, _u64, _sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64, ctypes.c_size_t
_lib = None


class IsingError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        msg = lib().ising_status_string(status).decode()
        super().__init__("%s: %s (%s)" % (where, STATUS_NAMES.get(self.status, self.status), msg))


def lib():
    """Load libising_b200.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    if _build.is_stale():
        if _build.nvcc_path() is None:
            import os
            if not os.path.exists(_build.LIB):
                raise RuntimeError("libising_b200.so is not built and nvcc is unavailable; "
                                   "run __graft_entry__.build() where nvcc exists. There is no CPU fallback.")
        else:
            _build.build_library()
    L = ctypes.CDLL(_build.LIB)
    L.ising_status_string.restype = ctypes.c_char_p
    L.ising_status_string.argtypes = [_i32]
    L.ising_workspace_bytes.restype = _i32
    L.ising_workspace_bytes.argtypes = [_i32, _i64, _i32, _i32, _i32, ctypes.POINTER(_sz)]
    L.ising_load_csr.restype = _i32
    L.ising_load_csr.argtypes = [_i32, _i64, _vp, _vp, _vp, _i32, _vp, _i32, _i32, _vp, _sz, _i32, _vp,
                                 ctypes.POINTER(_vp)]
    L.ising_anneal.restype = _i32
    L.ising_anneal.argtypes = [_vp, _i32, _i32, _i32, _i32, _u64, _vp, _i32, _i32, _i32, _vp, _vp, _vp]
    L.ising_energy_cut.restype = _i32
    L.ising_energy_cut.argtypes = [_vp, _vp, _i32, _vp, _vp, _vp]
    L.ising_best_state.restype = _i32
    L.ising_best_state.argtypes = [_vp, _i32, _vp, ctypes.POINTER(_i64), ctypes.POINTER(_i32),
                                   ctypes.POINTER(_i32), _vp]
    L.ising_current_state.restype = _i32
    L.ising_current_state.argtypes = [_vp, _vp, _i32, _vp]
    L.ising_problem_info.restype = _i32
    L.ising_problem_info.argtypes = [_vp, _i32, ctypes.POINTER(_i64)]
    L.ising_debug_phase_timing.restype = _i32
    L.ising_debug_phase_timing.argtypes = [_vp, _vp, _i32]
    L.ising_debug_probe_l2.restype = _i32
    L.ising_debug_probe_l2.argtypes = [_vp, _sz, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                       ctypes.POINTER(ctypes.c_double), _vp]
    L.ising_free.restype = _i32
    L.ising_free.argtypes = [_vp]
    L.ising_energy_cut_noalloc.restype = _i32
    L.ising_energy_cut_noalloc.argtypes = [_i32, _i64, _vp, _vp, _vp, _i32, _vp, _i32, _vp, _vp, _vp]
    _lib = L
    return L


def _torch():
    import torch
    return torch


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def _ptr(x):
    """Raw pointer of a numpy array (host) or torch tensor (device or host)."""
    if x is None:
        return None
    if _is_torch(x):
        assert x.is_contiguous()
        return x.data_ptr()
    assert x.flags["C_CONTIGUOUS"]
    return x.ctypes.data


def _stream(stream):
    if stream is not None:
        return int(stream)
    return int(_torch().cuda.current_stream().cuda_stream)


def _check(status: int, where: str):
    if status != 0:
        raise IsingError(status, where)


def _as(x, np_dtype, torch_dtype_name):
    if x is None:
        return None
    if _is_torch(x):
        t = _torch()
        want = getattr(t, torch_dtype_name)
        return x.to(want).contiguous() if x.dtype != want or not x.is_contiguous() else x
    return np.ascontiguousarray(x, dtype=np_dtype)


@dataclass
class Problem:
    """Handle of a loaded graph; owns the device workspace (a torch uint8 tensor)."""
    handle: int
    workspace: object
    n: int
    nnz: int
    n_colours: int
    max_replicas: int
    _keep: list = field(default_factory=list)

    def info(self, what: int) -> int:
        v = _i64(0)
        _check(lib().ising_problem_info(self.handle, what, ctypes.byref(v)), "ising_problem_info")
        return int(v.value)

    @property
    def w_total(self) -> int:
        return self.info(4)

    @property
    def has_dense_engine(self) -> bool:
        return bool(self.info(5))

    @property
    def launches(self) -> int:
        return self.info(6)

    @property
    def engine(self) -> int:
        """ENGINE_* : which Gauss-Seidel kernel ising_anneal will use for this problem."""
        return self.info(13)

    def phase_timing(self, sweep: int = 0):
        """Diagnostics (include/ising_debug.h): record SM clocks of sweep `sweep` of the next GS anneal (per virtual
        phase and CTA: 0/1 barrier arrive / leave).  Returns the int64 device tensor [virtual phases + 1][n_cta][8]."""
        t = _torch()
        buf = t.zeros((self.info(15) + 1, self.info(12), 8), dtype=t.int64, device="cuda")
        _check(lib().ising_debug_phase_timing(self.handle, buf.data_ptr(), sweep), "ising_debug_phase_timing")
        self._keep.append(buf)
        return buf

    def free(self):
        if self.handle:
            lib().ising_free(self.handle)
            self.handle = 0
            self.workspace = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def ising_workspace_bytes(n: int, nnz: int, wtype: int, max_replicas: int, n_colours: int) -> int:
    out = _sz(0)
    _check(lib().ising_workspace_bytes(n, nnz, wtype, max_replicas, n_colours, ctypes.byref(out)),
           "ising_workspace_bytes")
    return int(out.value)


def ising_load_csr(row_ptr, col_idx, weights, colour=None, n_colours: int = 0, max_replicas: int = 1,
                   flags: int = 0, stream=None, workspace_bytes: Optional[int] = None,
                   n: Optional[int] = None) -> Problem:
    """Arrays may be numpy (host) or torch CUDA tensors (device).  weights: int8 or int32."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise RuntimeError("ising_load_csr needs a CUDA device (B200); there is no CPU fallback")
    row_ptr = _as(row_ptr, np.int64, "int64")
    col_idx = _as(col_idx, np.int32, "int32")
    if _is_torch(weights):
        wtype = ISING_W_INT8 if weights.dtype == torch.int8 else ISING_W_INT32
        weights = _as(weights, None, "int8" if wtype == 1 else "int32")
    else:
        weights = np.ascontiguousarray(weights)
        if weights.dtype == np.int8:
            wtype = ISING_W_INT8
        elif weights.dtype == np.int32:
            wtype = ISING_W_INT32
        else:
            raise TypeError("weights must be int8 or int32")
    colour = _as(colour, np.int32, "int32")
    if n is None:
        n = int(row_ptr.shape[0]) - 1
    nnz = int(col_idx.shape[0])
    if workspace_bytes is None:
        workspace_bytes = ising_workspace_bytes(n, nnz, wtype, max_replicas, n_colours)
    ws = torch.empty(int(workspace_bytes) + 256, dtype=torch.uint8, device="cuda")
    base = ws.data_ptr()
    off = (-base) % 256
    h = _vp(0)
    st = lib().ising_load_csr(n, nnz, _ptr(row_ptr), _ptr(col_idx), _ptr(weights), wtype, _ptr(colour),
                              n_colours, max_replicas, base + off, int(workspace_bytes), flags,
                              _stream(stream), ctypes.byref(h))
    _check(st, "ising_load_csr")
    return Problem(handle=h.value, workspace=ws, n=n, nnz=nnz, n_colours=n_colours, max_replicas=max_replicas)


def ising_anneal(p: Problem, thresholds, *, mode: int = ISING_MODE_GS, tie_rule: int = ISING_TIE_MINUS,
                 n_replicas: int = 1, first_replica: int = 0, seed: int = 0, sweep_offset: int = 0,
                 init_mode: int = ISING_INIT_PHILOX, init_spins=None, cut_trace=None, stream=None):
    """Enqueue n_sweeps = len(thresholds) sweeps.  cut_trace: torch int64 CUDA tensor [M][R], True to
    allocate one, or None.  Returns the trace tensor (or None)."""
    torch = _torch()
    thr = np.ascontiguousarray(thresholds, dtype=np.uint32)
    M = int(thr.shape[0])
    if cut_trace is True:
        cut_trace = torch.zeros((max(M, 1), n_replicas), dtype=torch.int64, device="cuda")
    if init_spins is not None:
        init_spins = _as(init_spins, np.int8, "int8")
    st = lib().ising_anneal(p.handle, mode, tie_rule, n_replicas, first_replica, _u64(int(seed)),
                            _ptr(thr) if M else None, M, sweep_offset, init_mode, _ptr(init_spins),
                            _ptr(cut_trace), _stream(stream))
    _check(st, "ising_anneal")
    return cut_trace


def ising_energy_cut(p: Problem, spins=None, n_replicas: Optional[int] = None, stream=None):
    """Returns (energy, cut) as torch int64 CUDA tensors [n_replicas]."""
    torch = _torch()
    if spins is not None:
        spins = _as(spins, np.int8, "int8")
        if n_replicas is None:
            n_replicas = int(spins.shape[0]) if spins.ndim == 2 else 1
    assert n_replicas is not None
    e = torch.zeros(n_replicas, dtype=torch.int64, device="cuda")
    c = torch.zeros(n_replicas, dtype=torch.int64, device="cuda")
    _check(lib().ising_energy_cut(p.handle, _ptr(spins), n_replicas, _ptr(e), _ptr(c), _stream(stream)),
           "ising_energy_cut")
    return e, c


NOALLOC_MAX_REPLICAS = 1024


def ising_energy_cut_noalloc(row_ptr, col_idx, weights, spins, energy_out, cut_out, stream=None):
    """include/ising_noalloc.h: energy / cut straight from a DEVICE CSR, nothing allocated (the library's static
    scratch; at most NOALLOC_MAX_REPLICAS replicas; calls that overlap on the GPU race).  Every argument is a CUDA
    tensor the caller owns: row_ptr int64 [n+1], col_idx int32 [nnz], weights int8 | int32 [nnz], spins int8 [R][n],
    energy_out / cut_out int64 [R] (either may be None).  Marshals only: no tensor is created here."""
    torch = _torch()
    for t in (row_ptr, col_idx, weights, spins, energy_out, cut_out):
        if t is not None and not (t.is_cuda and t.is_contiguous()):
            raise ValueError("ising_energy_cut_noalloc takes contiguous CUDA tensors")
    if row_ptr.dtype != torch.int64 or col_idx.dtype != torch.int32 or spins.dtype != torch.int8:
        raise ValueError("row_ptr int64, col_idx int32, spins int8")
    wtype = {torch.int8: ISING_W_INT8, torch.int32: ISING_W_INT32}[weights.dtype]
    n = int(row_ptr.numel()) - 1
    n_replicas = int(spins.shape[0]) if spins.ndim == 2 else 1
    _check(lib().ising_energy_cut_noalloc(n, int(col_idx.numel()), _ptr(row_ptr), _ptr(col_idx), _ptr(weights), wtype,
                                          _ptr(spins), n_replicas, _ptr(energy_out), _ptr(cut_out), _stream(stream)),
           "ising_energy_cut_noalloc")


def ising_best_state(p: Problem, replica: int = -1, want_spins: bool = True, stream=None):
    """Returns (spins torch int8 CUDA [n] or None, cut, sweep, replica)."""
    torch = _torch()
    s = torch.zeros(p.n, dtype=torch.int8, device="cuda") if want_spins else None
    cut, sweep, rep = _i64(0), _i32(0), _i32(0)
    _check(lib().ising_best_state(p.handle, replica, _ptr(s), ctypes.byref(cut), ctypes.byref(sweep),
                                  ctypes.byref(rep), _stream(stream)), "ising_best_state")
    return s, int(cut.value), int(sweep.value), int(rep.value)


def ising_current_state(p: Problem, n_replicas: int, out=None, stream=None):
    """Current spins as a torch int8 CUDA tensor [n_replicas][n] (or written into `out`)."""
    torch = _torch()
    if out is None:
        out = torch.zeros((n_replicas, p.n), dtype=torch.int8, device="cuda")
    _check(lib().ising_current_state(p.handle, _ptr(out), n_replicas, _stream(stream)), "ising_current_state")
    return out


def probe_l2(nbytes: int = 32 << 20, stream=None):
    """include/ising_debug.h: (random 32-byte sector gather GB/s with the best access shape, the same with the sweep's
    16-byte lane-pair shape, streaming read GB/s) of an nbytes buffer on this GPU."""
    t = _torch()
    buf = t.zeros(nbytes, dtype=t.uint8, device="cuda")
    g, g16, s_ = ctypes.c_double(0), ctypes.c_double(0), ctypes.c_double(0)
    _check(lib().ising_debug_probe_l2(buf.data_ptr(), nbytes, ctypes.byref(g), ctypes.byref(g16), ctypes.byref(s_),
                                      _stream(stream)), "ising_debug_probe_l2")
    return float(g.value), float(g16.value), float(s_.value)


def ising_free(p: Problem):
    p.free()


def load_workload(wl, max_replicas: Optional[int] = None, flags: int = 0, device_inputs: bool = False) -> Problem:
    """Convenience: ising_load_csr on a workloads.Workload."""
    torch = _torch()
    arrs = [wl.row_ptr, wl.col, wl.w, wl.colour]
    if device_inputs:
        arrs = [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]
    return ising_load_csr(arrs[0], arrs[1], arrs[2], arrs[3], wl.n_colours,
                          max_replicas or wl.n_replicas, flags=flags)


def anneal_workload(p: Problem, wl, **kw):
    """Convenience: ising_anneal with the workload's mode / seed / replicas / thresholds."""
    args = dict(mode=ISING_MODE_GS if wl.mode == "gs" else ISING_MODE_JACOBI, tie_rule=wl.tie_rule,
                n_replicas=wl.n_replicas, first_replica=wl.first_replica, seed=wl.seed)
    thr = kw.pop("thr", wl.thr)
    args.update(kw)
    return ising_anneal(p, thr, **args)
