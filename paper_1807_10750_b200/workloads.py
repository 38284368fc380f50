"""Seeded synthetic workload generators (graphs, weights, colourings, schedules).

This module is the ONE piece shared by the CPU oracle tests and the CUDA path.
It holds none of the method's arithmetic (no field, no update rule, no Philox,
no energy): it only produces *inputs* -- a symmetric integer-weighted CSR
graph, a proper colouring, per-sweep uint32 flip thresholds -- with the shapes
of the paper's workloads (G-set benchmark + custom random graphs,
Table III).  Neither the G-set files nor the paper's custom graphs are
reproduced; these synthetic graphs stand in for them.

All randomness is an integer counter-based generator (splitmix64 finaliser over
seed + index), so the inputs do not depend on numpy's RNG implementation.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_GOLD = np.uint64(0x9E3779B97F4A7C15)


# --------------------------------------------------------------------------
# integer RNG
# --------------------------------------------------------------------------
def splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 output function applied to uint64 state(s) `x` (vectorised)."""
    with np.errstate(over="ignore"):
        z = np.asarray(x, dtype=np.uint64) + _GOLD
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def rand_u64(seed: int, stream: int, count: int, offset: int = 0) -> np.ndarray:
    """`count` uint64 words of stream `stream` of generator `seed` (counter based)."""
    with np.errstate(over="ignore"):
        base = splitmix64(np.array([seed], dtype=np.uint64) * np.uint64(0xD1342543DE82EF95)
                          + np.uint64(stream) * np.uint64(0xDA942042E4DD58B5))[0]
        idx = np.arange(offset, offset + count, dtype=np.uint64)
        return splitmix64(base + idx * _GOLD)


def rand_unit(seed: int, stream: int, count: int) -> np.ndarray:
    """Uniform doubles in [0,1) with 53 random bits."""
    return (rand_u64(seed, stream, count) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))


def hash_pairs(seed: int, a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Order-sensitive 64-bit hash of integer pairs (used with a<b for edge weights)."""
    with np.errstate(over="ignore"):
        k = (a.astype(np.uint64) << np.uint64(32)) | b.astype(np.uint64)
        s = splitmix64(np.array([seed], dtype=np.uint64) * np.uint64(0xD1342543DE82EF95))[0]
        return splitmix64(splitmix64(k ^ s))


# --------------------------------------------------------------------------
# workload container
# --------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    n: int
    row_ptr: np.ndarray            # int64 [n+1]
    col: np.ndarray                # int32 [nnz], rows sorted by column, symmetric
    w: np.ndarray                  # int8 or int32 [nnz]
    colour: Optional[np.ndarray]   # int32 [n] proper colouring, or None (Jacobi only)
    n_colours: int
    n_replicas: int
    first_replica: int
    seed: int                      # Philox seed
    thr: np.ndarray                # uint32 [M] per-sweep flip thresholds
    mode: str                      # "gs" | "jacobi"
    tie_rule: int = 0              # 0 MINUS, 1 KEEP
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    @property
    def n_sweeps(self) -> int:
        return int(self.thr.shape[0])

    @property
    def w_total(self) -> int:
        """W = sum_{i<j} w_ij = half the sum over directed entries."""
        return int(self.w.astype(np.int64).sum()) // 2


# --------------------------------------------------------------------------
# CSR assembly from an undirected edge list
# --------------------------------------------------------------------------
def csr_from_edges(n: int, u: np.ndarray, v: np.ndarray, wt: np.ndarray, wdtype):
    """Symmetric CSR (both directions, rows sorted by column) from unique pairs u<v."""
    u = u.astype(np.int64)
    v = v.astype(np.int64)
    src = np.concatenate([u, v])
    dst = np.concatenate([v, u])
    ww = np.concatenate([wt, wt])
    key = src * np.int64(n) + dst
    order = np.argsort(key, kind="stable")
    src = src[order]
    col = dst[order].astype(np.int32)
    w = ww[order].astype(wdtype)
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    row_ptr[1:] = np.cumsum(np.bincount(src, minlength=n), dtype=np.int64)
    return row_ptr, col, w


def weights_from_hash(h: np.ndarray, kind: str) -> np.ndarray:
    """Map 64-bit hashes to integer weights.
    kind: "+1" | "pm1" | "pm4" ([-4,4] minus 0) | "pm8" ([-8,8] minus 0)."""
    if kind == "+1":
        return np.ones(h.shape, dtype=np.int64)
    if kind == "pm1":
        return np.where((h >> np.uint64(17)) & np.uint64(1), 1, -1).astype(np.int64)
    if kind in ("pm4", "pm8"):
        m = 4 if kind == "pm4" else 8
        k = ((h >> np.uint64(20)) % np.uint64(2 * m)).astype(np.int64)  # 0..2m-1
        return np.where(k < m, k - m, k - m + 1)
    raise ValueError(kind)


# --------------------------------------------------------------------------
# graph families
# --------------------------------------------------------------------------
def erdos_renyi_edges(n: int, p: float, seed: int):
    """Each pair i<j kept with probability p (pairs enumerated row by row)."""
    iu, ju = np.triu_indices(n, k=1)
    keep = rand_unit(seed, 1, iu.size) < p
    return iu[keep].astype(np.int64), ju[keep].astype(np.int64)


def torus_edges(L: int):
    """L x L toroidal grid, id = L*y + x; each undirected edge once (u<v)."""
    y, x = np.divmod(np.arange(L * L, dtype=np.int64), L)
    right = L * y + (x + 1) % L
    down = L * ((y + 1) % L) + x
    me = np.arange(L * L, dtype=np.int64)
    a = np.concatenate([me, me])
    b = np.concatenate([right, down])
    u = np.minimum(a, b)
    v = np.maximum(a, b)
    key = np.unique(u * (L * L) + v)      # L=2 would duplicate; unique keeps it simple
    u, v = np.divmod(key, L * L)
    keep = u != v
    return u[keep], v[keep]


def complete_edges(n: int):
    iu, ju = np.triu_indices(n, k=1)
    return iu.astype(np.int64), ju.astype(np.int64)


def powerlaw_edges(n: int, seed: int, exponent: float = 2.5, dmin: int = 6, dmax: int = 4096):
    """Configuration model with i.i.d. degrees P(d) ~ d^-exponent on [dmin, dmax];
    stubs matched by a seeded shuffle; self-loops and multi-edges dropped."""
    dmax = int(min(dmax, max(dmin, n // 4)))
    d = np.arange(dmin, dmax + 1, dtype=np.float64)
    pmf = d ** (-exponent)
    cdf = np.cumsum(pmf / pmf.sum())
    deg = dmin + np.searchsorted(cdf, rand_unit(seed, 1, n), side="right")
    deg = np.minimum(deg, dmax).astype(np.int64)
    if int(deg.sum()) & 1:
        deg[-1] += 1
    stubs = np.repeat(np.arange(n, dtype=np.int64), deg)
    perm = np.argsort(rand_u64(seed, 2, stubs.size), kind="stable")
    stubs = stubs[perm]
    a = stubs[0::2]
    b = stubs[1::2]
    u = np.minimum(a, b)
    v = np.maximum(a, b)
    keep = u != v
    key = np.unique(u[keep] * np.int64(n) + v[keep])
    u, v = np.divmod(key, np.int64(n))
    return u, v


# --------------------------------------------------------------------------
# colouring (native helper)
# --------------------------------------------------------------------------
_wl_lib = None


def _load_native():
    global _wl_lib
    if _wl_lib is not None:
        return _wl_lib
    so = os.path.join(_HERE, "_wlgen.so")
    src = os.path.join(_HERE, "_wlgen.c")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", so, src])
    lib = ctypes.CDLL(so)
    lib.wl_greedy_colour.restype = ctypes.c_int32
    lib.wl_greedy_colour.argtypes = [ctypes.c_int32] + [ctypes.c_void_p] * 4
    _wl_lib = lib
    return lib


def greedy_colouring(n: int, row_ptr: np.ndarray, col: np.ndarray, order: str = "index"):
    """Sequential greedy colouring.  order: "index" (smallest index first) or
    "ldf" (largest degree first, ties by index).  Returns (colour int32[n], n_colours)."""
    lib = _load_native()
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col = np.ascontiguousarray(col, dtype=np.int32)
    if order == "index":
        visit = np.arange(n, dtype=np.int32)
    elif order == "ldf":
        deg = np.diff(row_ptr)
        visit = np.lexsort((np.arange(n), -deg)).astype(np.int32)
    else:
        raise ValueError(order)
    colour = np.empty(n, dtype=np.int32)
    nc = lib.wl_greedy_colour(n, row_ptr.ctypes.data, col.ctypes.data,
                              visit.ctypes.data, colour.ctypes.data)
    if nc < 0:
        raise MemoryError("wl_greedy_colour")
    return colour, int(nc)


# --------------------------------------------------------------------------
# schedules -> uint32 thresholds  (schedules are inputs)
# --------------------------------------------------------------------------
def thresholds_from_probs(p: np.ndarray) -> np.ndarray:
    """thr[t] = min(floor(p_t * 2^32), 2^32 - 1), computed once in IEEE double."""
    t = np.floor(np.asarray(p, dtype=np.float64) * 4294967296.0)
    t = np.clip(t, 0.0, 4294967295.0)
    return t.astype(np.uint64).astype(np.uint32)


def linear_schedule(p0: float, p_end: float, m: int) -> np.ndarray:
    if m == 1:
        return thresholds_from_probs(np.array([p0]))
    t = np.arange(m, dtype=np.float64)
    return thresholds_from_probs(p0 + (p_end - p0) * t / (m - 1))


def exponential_schedule(p0: float, p_end: float, m: int) -> np.ndarray:
    if m == 1:
        return thresholds_from_probs(np.array([p0]))
    t = np.arange(m, dtype=np.float64)
    return thresholds_from_probs(p0 * (p_end / p0) ** (t / (m - 1)))


# --------------------------------------------------------------------------
# the five BASELINE.json configurations (and scaled-down variants)
# --------------------------------------------------------------------------
def exact_n_schedule(n0: int, m: int, kind: str = "linear", factor: float = 0.01) -> np.ndarray:
    """Numbers of spins to flip per sweep for Algorithm 1 (ISING_MODE_EXACT_N).  The paper's setting "set to 200
    which decays linearly each sweep by a factor of 0.01" is ambiguous (reading Q6): "linear"
    subtracts factor * n0 per sweep (N_t = max(0, round(n0 (1 - factor t))), zero after 1 / factor sweeps),
    "geometric" multiplies by (1 - factor) per sweep."""
    t = np.arange(m, dtype=np.float64)
    if kind == "linear":
        v = n0 * (1.0 - factor * t)
    elif kind == "geometric":
        v = n0 * (1.0 - factor) ** t
    else:
        raise ValueError(kind)
    return np.maximum(0, np.rint(v)).astype(np.uint32)


def _finish(name, n, u, v, wkind, wdtype, wseed, colouring, R, first, seed, thr, mode, note,
            torus_L=None):
    wt = weights_from_hash(hash_pairs(wseed, u, v), wkind)
    row_ptr, col, w = csr_from_edges(n, u, v, wt, wdtype)
    if colouring is None:
        colour, nc = None, 0
    elif colouring == "checker":
        y, x = np.divmod(np.arange(n), torus_L)
        colour = ((x + y) & 1).astype(np.int32)
        nc = 2
    else:
        colour, nc = greedy_colouring(n, row_ptr, col, colouring)
    return Workload(name=name, n=n, row_ptr=row_ptr, col=col, w=w, colour=colour, n_colours=nc,
                    n_replicas=R, first_replica=first, seed=seed, thr=thr, mode=mode, note=note)


def config1(n: int = 800, p: float = 0.06, sweeps: int = 1000, replicas: int = 1) -> Workload:
    """ER(800, 0.06), all weights +1 passed as int32, 1 replica, smallest-index greedy
    colouring, 1000 sweeps, linear 0.10 -> 0.0, Philox seed 1.  Stands in for the G-set
    800-vertex 6%-density family (Table III row G9, L279)."""
    u, v = erdos_renyi_edges(n, p, 1001)
    return _finish("cfg1_er800", n, u, v, "+1", np.int32, 1001, "index", replicas, 0, 1,
                   linear_schedule(0.10, 0.0, sweeps), "gs", "ER graph, w=+1 (int32)")


def config2(n: int = 2000, p: float = 0.005, sweeps: int = 2000, replicas: int = 64) -> Workload:
    """G(2000, 0.005), weights +-1 int8, 64 replicas, 2000 sweeps, linear 0.10 -> 0.0,
    colour-class Gauss-Seidel.  Stands in for the G-set 2000-vertex sparse +-1 family."""
    u, v = erdos_renyi_edges(n, p, 1002)
    return _finish("cfg2_g2000", n, u, v, "pm1", np.int8, 1002, "index", replicas, 0, 0,
                   linear_schedule(0.10, 0.0, sweeps), "gs", "random graph, w=+-1 (int8)")


def config3(L: int = 100, sweeps: int = 5000, replicas: int = 256, all_plus: bool = False) -> Workload:
    """L x L toroidal grid (degree 4), weights +-1 int8 (or all +1), 256 replicas,
    5000 sweeps, checkerboard 2-colouring.  Stands in for the G-set toroidal family
    (Table III row G67, L281).  all_plus: known max cut = #E = 2 L^2 (L even)."""
    u, v = torus_edges(L)
    return _finish("cfg3_torus%d%s" % (L, "_plus" if all_plus else ""), L * L, u, v,
                   "+1" if all_plus else "pm1", np.int8, 1003, "checker", replicas, 0, 0,
                   linear_schedule(0.10, 0.0, sweeps), "gs", "2D torus", torus_L=L)


def config4(n: int = 4096, sweeps: int = 1000, replicas: int = 1024) -> Workload:
    """Fully connected K_n, weights uniform int8 in [-8,8] minus 0, symmetric, zero diagonal,
    1024 replicas, synchronous Jacobi, 1000 sweeps, linear 0.10 -> 0.0.  Not in the paper
    (general connectivity only); exercises the dense tcgen05 field path."""
    u, v = complete_edges(n)
    return _finish("cfg4_k%d" % n, n, u, v, "pm8", np.int8, 1004, None, replicas, 0, 0,
                   linear_schedule(0.10, 0.0, sweeps), "jacobi", "K_n dense int8")


def config5(n: int = 1_000_000, sweeps: int = 500, replicas: int = 32,
            colouring: str = "ldf") -> Workload:
    """Sparse power-law graph (exponent 2.5, degrees in [6,4096], mean ~16), weights uniform
    int8 in [-4,4] minus 0, 32 replicas, 500 sweeps, greedy colouring shipped with the input
    (largest-degree-first by default), exponential schedule 0.2 -> 1e-4.  Stands in for the
    paper's large custom random graphs C6/C7, scaled to 1M vertices."""
    u, v = powerlaw_edges(n, 1005)
    return _finish("cfg5_powerlaw%d" % n, n, u, v, "pm4", np.int8, 1005, colouring, replicas, 0, 0,
                   exponential_schedule(0.2, 1e-4, sweeps), "gs", "power-law sparse, %s colouring" % colouring)


def load_edge_list(path: str, replicas: int = 32, sweeps: int = 1000, p0: float = 0.10, p_end: float = 0.0,
                   colouring: str = "ldf", seed: int = 0, name: Optional[str] = None) -> Workload:
    """Weighted graph from a text file in the edge-list layout the paper's benchmark files use (PAPER.md L190,
    SURVEY 8(f) rank 4; the files themselves are not in this repo): first line `n m`, then m lines `i j w` with
    1-based vertex ids and an integer weight.  Duplicate pairs are summed, self loops dropped, zero weights dropped.
    Returns a Gauss-Seidel workload with a greedy colouring and a linear flip schedule p0 -> p_end."""
    with open(path, "r") as f:
        head = f.readline().split()
        n, m = int(head[0]), int(head[1])
        data = np.loadtxt(f, dtype=np.int64, ndmin=2) if m > 0 else np.zeros((0, 3), dtype=np.int64)
    if data.shape[0] != m or (m > 0 and data.shape[1] != 3):
        raise ValueError("%s: expected %d lines 'i j w'" % (path, m))
    i, j, w = data[:, 0] - 1, data[:, 1] - 1, data[:, 2]
    if m > 0 and (i.min() < 0 or j.min() < 0 or i.max() >= n or j.max() >= n):
        raise ValueError("%s: vertex id out of range 1..%d" % (path, n))
    keep = i != j
    i, j, w = i[keep], j[keep], w[keep]
    u, v = np.minimum(i, j), np.maximum(i, j)
    key, inv = np.unique(u * n + v, return_inverse=True)
    wsum = np.zeros(key.shape[0], dtype=np.int64)
    np.add.at(wsum, inv, w)
    nz = wsum != 0
    key, wsum = key[nz], wsum[nz]
    u, v = key // n, key % n
    wdtype = np.int8 if (wsum.size == 0 or np.abs(wsum).max() <= 127) else np.int32
    row_ptr, col, wt = csr_from_edges(n, u, v, wsum, wdtype)
    colour, nc = greedy_colouring(n, row_ptr, col, colouring)
    return Workload(name=name or os.path.basename(path), n=n, row_ptr=row_ptr, col=col, w=wt, colour=colour,
                    n_colours=nc, n_replicas=replicas, first_replica=0, seed=seed,
                    thr=linear_schedule(p0, p_end, sweeps), mode="gs", note="edge-list file %s" % path)


def build_config(k: int, **kw) -> Workload:
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[k](**kw)


def random_spins(seed: int, n_replicas: int, n: int) -> np.ndarray:
    """Seeded +-1 int8 spins [R][n] for energy/cut parity tests (an input, not Philox)."""
    bits = (rand_u64(seed, 7, n_replicas * n) >> np.uint64(33)) & np.uint64(1)
    return (bits.astype(np.int8) * 2 - 1).reshape(n_replicas, n)
