"""Helpers of the `-m gpu` parity tests: run the CUDA path through the binding (C ABI) and
compare with the CPU oracle element by element."""
import numpy as np

import paper_1807_10750_b200 as P
from oracle import ising_oracle as O


def gpu_anneal(wl, *, thr=None, n_replicas=None, first_replica=None, mode=None, tie_rule=None, seed=None,
               sweep_offset=0, init_spins=None, flags=0, device_inputs=False, problem=None, init_mode=None,
               want_best_spins=True):
    """Returns a dict shaped like oracle.anneal(): final, trace, best_cut, best_sweep, best_spins."""
    import torch
    thr = wl.thr if thr is None else thr
    R = wl.n_replicas if n_replicas is None else n_replicas
    p = problem or P.load_workload(wl, max_replicas=max(R, wl.n_replicas), flags=flags, device_inputs=device_inputs)
    kw = dict(thr=thr, n_replicas=R, sweep_offset=sweep_offset, cut_trace=True)
    if first_replica is not None:
        kw["first_replica"] = first_replica
    if mode is not None:
        kw["mode"] = mode
    if tie_rule is not None:
        kw["tie_rule"] = tie_rule
    if seed is not None:
        kw["seed"] = seed
    if init_spins is not None:
        kw["init_mode"] = P.ISING_INIT_GIVEN
        kw["init_spins"] = init_spins
    if init_mode is not None:
        kw["init_mode"] = init_mode
    trace = P.anneal_workload(p, wl, **kw)
    final = P.ising_current_state(p, R)
    torch.cuda.synchronize()
    out = dict(final=final.cpu().numpy(), trace=trace.cpu().numpy()[: len(thr)])
    bc = np.zeros(R, dtype=np.int64)
    bs = np.zeros(R, dtype=np.int32)
    bsp = np.zeros((R, wl.n), dtype=np.int8)
    if len(thr) > 0:
        for r in range(R):
            s, cut, sweep, rep = P.ising_best_state(p, r, want_spins=want_best_spins)
            assert rep == r
            bc[r], bs[r] = cut, sweep
            if want_best_spins:
                bsp[r] = s.cpu().numpy()
    out.update(best_cut=bc, best_sweep=bs, best_spins=bsp, problem=p)
    return out


def oracle_anneal(wl, *, thr=None, n_replicas=None, first_replica=None, mode=None, tie_rule=None, seed=None,
                  sweep_offset=0, init_spins=None, n_threads=8):
    kw = dict(n_threads=n_threads, sweep_offset=sweep_offset)
    if thr is not None:
        kw["thr"] = thr
    if n_replicas is not None:
        kw["n_replicas"] = n_replicas
    if first_replica is not None:
        kw["first_replica"] = first_replica
    if mode is not None:
        kw["mode"] = mode
        if mode == 0 and wl.colour is not None:
            kw["order"] = O.order_from_colour(wl.colour)
    if tie_rule is not None:
        kw["tie_rule"] = tie_rule
    if seed is not None:
        kw["seed"] = seed
    if init_spins is not None:
        kw["init_spins"] = init_spins
    return O.anneal_workload(wl, **kw)


def assert_same(g, o, best_spins=True):
    """Bit-exact: every cut of the trace, final spins, best cut / sweep / spins, all replicas."""
    np.testing.assert_array_equal(g["trace"], o["trace"])
    np.testing.assert_array_equal(g["final"], o["final"])
    if o["trace"].shape[0] > 0:
        np.testing.assert_array_equal(g["best_cut"], o["best_cut"])
        np.testing.assert_array_equal(g["best_sweep"], o["best_sweep"])
        if best_spins:
            np.testing.assert_array_equal(g["best_spins"], o["best_spins"])
