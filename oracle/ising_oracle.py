"""ctypes loader for the CPU oracle (oracle/ising_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It holds
no arithmetic of its own: it compiles ising_oracle.cpp with g++ on first use and
marshals numpy arrays into the `oracle_*` C functions.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ising_oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None

_vp = ctypes.c_void_p
_i32 = ctypes.c_int32
_u64 = ctypes.c_uint64


def build(force: bool = False) -> str:
    """Compile the oracle shared library (g++ -O2, no CUDA anywhere)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread",
                               "-o", _SO, _SRC])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.oracle_philox4x32_10.restype = None
        L.oracle_philox4x32_10.argtypes = [_vp, _vp, _vp]
        L.oracle_energy_cut.restype = _i32
        L.oracle_energy_cut.argtypes = [_i32, _vp, _vp, _vp, _i32, _vp, _i32, _vp, _vp]
        L.oracle_local_fields.restype = _i32
        L.oracle_local_fields.argtypes = [_i32, _vp, _vp, _vp, _i32, _vp, _vp]
        L.oracle_anneal.restype = _i32
        L.oracle_anneal.argtypes = [_i32, _vp, _vp, _vp, _i32, _vp, _i32, _i32, _i32, _i32, _u64,
                                    _vp, _i32, _i32, _vp, _vp, _vp, _vp, _vp, _vp, _i32]
        L.oracle_bruteforce_maxcut.restype = _i32
        L.oracle_bruteforce_maxcut.argtypes = [_i32, _vp, _vp, _vp, _i32, _vp, _vp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data


def _wtype(w: np.ndarray) -> int:
    if w.dtype == np.int8:
        return 1
    if w.dtype == np.int32:
        return 4
    raise TypeError("weights must be int8 or int32")


def _graph(row_ptr, col, w):
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col = np.ascontiguousarray(col, dtype=np.int32)
    w = np.ascontiguousarray(w)
    return row_ptr, col, w, _wtype(w)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def energy_cut(n, row_ptr, col, w, spins):
    """spins int8 [R][n] -> (E int64[R], cut int64[R])."""
    row_ptr, col, w, wt = _graph(row_ptr, col, w)
    spins = np.ascontiguousarray(spins, dtype=np.int8).reshape(-1, n)
    R = spins.shape[0]
    E = np.zeros(R, dtype=np.int64)
    cut = np.zeros(R, dtype=np.int64)
    rc = lib().oracle_energy_cut(n, _p(row_ptr), _p(col), _p(w), wt, _p(spins), R, _p(E), _p(cut))
    assert rc == 0
    return E, cut


def local_fields(n, row_ptr, col, w, spins):
    row_ptr, col, w, wt = _graph(row_ptr, col, w)
    spins = np.ascontiguousarray(spins, dtype=np.int8).reshape(n)
    h = np.zeros(n, dtype=np.int64)
    rc = lib().oracle_local_fields(n, _p(row_ptr), _p(col), _p(w), wt, _p(spins), _p(h))
    assert rc == 0
    return h


def order_from_colour(colour: np.ndarray) -> np.ndarray:
    """Visiting order of the colour-class Gauss-Seidel sweep: (colour asc, id asc)."""
    n = colour.shape[0]
    return np.lexsort((np.arange(n), colour)).astype(np.int32)


def anneal(n, row_ptr, col, w, *, order=None, mode=0, tie_rule=0, n_replicas=1, first_replica=0,
           seed=0, thr=None, sweep_offset=0, init_spins=None, n_threads=1):
    """Run the oracle annealer.  Returns dict(final, trace, best_cut, best_sweep, best_spins)."""
    row_ptr, col, w, wt = _graph(row_ptr, col, w)
    thr = np.ascontiguousarray(thr, dtype=np.uint32)
    M = int(thr.shape[0])
    R = int(n_replicas)
    if order is not None:
        order = np.ascontiguousarray(order, dtype=np.int32)
    if init_spins is not None:
        init_spins = np.ascontiguousarray(init_spins, dtype=np.int8).reshape(R, n)
    final = np.zeros((R, n), dtype=np.int8)
    trace = np.zeros((M, R), dtype=np.int64)
    best_cut = np.zeros(R, dtype=np.int64)
    best_sweep = np.full(R, -1, dtype=np.int32)
    best_spins = np.zeros((R, n), dtype=np.int8)
    rc = lib().oracle_anneal(n, _p(row_ptr), _p(col), _p(w), wt, _p(order), int(mode), int(tie_rule),
                             R, int(first_replica), ctypes.c_uint64(int(seed)), _p(thr), M,
                             int(sweep_offset), _p(init_spins), _p(final), _p(trace), _p(best_cut),
                             _p(best_sweep), _p(best_spins), int(n_threads))
    assert rc == 0, rc
    return dict(final=final, trace=trace, best_cut=best_cut, best_sweep=best_sweep,
                best_spins=best_spins)


def bruteforce_maxcut(n, row_ptr, col, w):
    row_ptr, col, w, wt = _graph(row_ptr, col, w)
    mc = np.zeros(1, dtype=np.int64)
    arg = np.zeros(n, dtype=np.int8)
    rc = lib().oracle_bruteforce_maxcut(n, _p(row_ptr), _p(col), _p(w), wt, _p(mc), _p(arg))
    assert rc == 0
    return int(mc[0]), arg


def anneal_workload(wl, **kw):
    """Convenience: run a paper_1807_10750_b200.workloads.Workload through the oracle."""
    args = dict(order=order_from_colour(wl.colour) if wl.colour is not None else None,
                mode=0 if wl.mode == "gs" else 1, tie_rule=wl.tie_rule, n_replicas=wl.n_replicas,
                first_replica=wl.first_replica, seed=wl.seed, thr=wl.thr)
    args.update(kw)
    return anneal(wl.n, wl.row_ptr, wl.col, wl.w, **args)
