"""General Ising / QUBO front door (eq. (1)-(3), L39-53).

The hot path minimises the pair energy  E(s) = sum_{i<j} w_ij s_i s_j  (max-cut form, external field zero,
L126).  An external field  sum_i f_i s_i  is brought into that form by the standard gauge reduction: one
auxiliary spin s_n with couplings w_in = f_i gives  E'(s, s_n) = sum_{i<j} w_ij s_i s_j + s_n sum_i f_i s_i,
E' is invariant under the global flip, and  E'(s, s_n) = E_field(s * s_n).  So the library, the oracle and the
parity tests run unchanged on the augmented graph; `decode_field_solution` maps a state back.
Nothing here runs on the device and nothing here is used by the oracle.
"""
from __future__ import annotations

from typing import Tuple

import numpy as np

from . import workloads as W


def ising_with_field(n: int, u: np.ndarray, v: np.ndarray, w: np.ndarray, f: np.ndarray):
    """Edges (u < v, integer weights w) plus an integer field f[n]  ->  edges of the augmented graph on n + 1
    vertices (vertex n = the auxiliary spin).  Returns (n + 1, u', v', w')."""
    f = np.asarray(f, dtype=np.int64)
    if f.shape != (n,):
        raise ValueError("field must have one entry per vertex")
    idx = np.nonzero(f)[0].astype(np.int64)
    u2 = np.concatenate([np.asarray(u, dtype=np.int64), idx])
    v2 = np.concatenate([np.asarray(v, dtype=np.int64), np.full(idx.size, n, dtype=np.int64)])
    w2 = np.concatenate([np.asarray(w, dtype=np.int64), f[idx]])
    order = np.argsort(u2 * (n + 1) + v2, kind="stable")
    return n + 1, u2[order], v2[order], w2[order]


def decode_field_solution(spins: np.ndarray) -> np.ndarray:
    """State(s) of the augmented graph [..., n + 1] -> state(s) of the original problem [..., n] (gauge s * s_n)."""
    spins = np.asarray(spins)
    return (spins[..., :-1] * spins[..., -1:]).astype(np.int8)


def field_energy(n: int, u, v, w, f, s) -> int:
    """E_field(s) = sum_{i<j} w_ij s_i s_j + sum_i f_i s_i (for checks on small instances)."""
    s = np.asarray(s, dtype=np.int64)
    return int((np.asarray(w, dtype=np.int64) * s[np.asarray(u)] * s[np.asarray(v)]).sum() + (np.asarray(f, dtype=np.int64) * s).sum())


def qubo_to_ising(Q: np.ndarray) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray, int]:
    """Minimise x^T Q x over x in {0,1}^n (Q integer, any square matrix; only Q + Q^T matters off the diagonal).
    With x = (1 + s) / 2:  4 x^T Q x = const + sum_i f_i s_i + sum_{i<j} w_ij s_i s_j  with
    w_ij = Q_ij + Q_ji,  f_i = 2 Q_ii + sum_{j != i} (Q_ij + Q_ji),  const = 2 tr Q + sum_{i<j} (Q_ij + Q_ji).
    Returns (u, v, w, f, const) with u < v and zero couplings dropped."""
    Q = np.asarray(Q, dtype=np.int64)
    n = Q.shape[0]
    if Q.shape != (n, n):
        raise ValueError("Q must be square")
    S = Q + Q.T
    iu, ju = np.triu_indices(n, k=1)
    w = S[iu, ju]
    f = 2 * np.diag(Q) + S.sum(axis=1) - np.diag(S)
    const = int(2 * np.trace(Q) + w.sum())
    keep = w != 0
    return iu[keep].astype(np.int64), ju[keep].astype(np.int64), w[keep], f.astype(np.int64), const


def field_workload(n: int, u, v, w, f, replicas: int = 32, sweeps: int = 1000, p0: float = 0.10, p_end: float = 0.0,
                   colouring: str = "ldf", seed: int = 0, name: str = "ising_with_field") -> W.Workload:
    """Gauss-Seidel workload of the augmented graph (greedy colouring, linear flip schedule)."""
    n2, u2, v2, w2 = ising_with_field(n, u, v, w, f)
    wdtype = np.int8 if (w2.size == 0 or np.abs(w2).max() <= 127) else np.int32
    row_ptr, col, wt = W.csr_from_edges(n2, u2, v2, w2, wdtype)
    colour, nc = W.greedy_colouring(n2, row_ptr, col, colouring)
    return W.Workload(name=name, n=n2, row_ptr=row_ptr, col=col, w=wt, colour=colour, n_colours=nc, n_replicas=replicas,
                      first_replica=0, seed=seed, thr=W.linear_schedule(p0, p_end, sweeps), mode="gs",
                      note="external field through one auxiliary spin (vertex %d)" % n)
