"""`-m gpu`: parity at BASELINE.json's full size for the workload bench.py times (config 5:
1M-spin power-law graph, 32 replicas), in the same launch configuration, on what the oracle can
compute in bounded time: every replica for the first sweeps, and a subset of replicas for longer.
Replicas are independent, so any subset is an exact check (SURVEY 8(c) sampling plan)."""
import numpy as np
import pytest

import paper_1807_10750_b200 as P
from paper_1807_10750_b200 import workloads as W

from gpu_util import assert_same, gpu_anneal, oracle_anneal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cfg5():
    return W.config5()


def test_config5_full_size_all_replicas_first_sweeps(cfg5):
    wl = cfg5
    M = 40
    g = gpu_anneal(wl, thr=wl.thr[:M], want_best_spins=False)
    o = oracle_anneal(wl, thr=wl.thr[:M], n_threads=16)
    assert_same(g, o, best_spins=False)
    # best state of one replica, full vector
    s, cut, sweep, rep = P.ising_best_state(g["problem"], 17)
    np.testing.assert_array_equal(s.cpu().numpy(), o["best_spins"][17])
    # the cold end of the schedule (sweeps 460..499, flip probability ~2e-4) from the oracle's state, all replicas
    g3 = gpu_anneal(wl, thr=wl.thr[460:], sweep_offset=460, init_spins=o["final"], want_best_spins=False,
                    problem=g["problem"])
    o3 = oracle_anneal(wl, thr=wl.thr[460:], sweep_offset=460, init_spins=o["final"], n_threads=16)
    assert_same(g3, o3, best_spins=False)
    # a replica subset straddling the Philox groups, run longer, same problem handle
    for first in (3,):
        g2 = gpu_anneal(wl, thr=wl.thr[:120], n_replicas=2, first_replica=first, problem=g["problem"],
                        want_best_spins=False)
        o2 = oracle_anneal(wl, thr=wl.thr[:120], n_replicas=2, first_replica=first)
        assert_same(g2, o2, best_spins=False)


def test_config5_energy_cut_of_final_state(cfg5):
    wl = cfg5
    p = P.load_workload(wl)
    trace = P.anneal_workload(p, wl, thr=wl.thr[:3], cut_trace=True)
    E, cut = P.ising_energy_cut(p, None, wl.n_replicas)     # from the definition, current state
    np.testing.assert_array_equal(cut.cpu().numpy(), trace.cpu().numpy()[2])


def test_config4_full_size_dense_engine_all_replicas_first_sweeps():
    """K_4096 x 1024 replicas on the tcgen05 engine in the launch configuration bench.py times (32 x 4 tiles): every
    replica for the first sweeps, and replicas straddling the 256-replica tile edges for longer (SURVEY 8(c) plan)."""
    wl = W.config4()
    g = gpu_anneal(wl, thr=wl.thr[:2], want_best_spins=False)
    assert g["problem"].has_dense_engine
    o = oracle_anneal(wl, thr=wl.thr[:2], n_threads=16)
    assert_same(g, o, best_spins=False)
    for first in (254, 1020):
        g2 = gpu_anneal(wl, thr=wl.thr[:12], n_replicas=4, first_replica=first, problem=g["problem"], want_best_spins=False)
        o2 = oracle_anneal(wl, thr=wl.thr[:12], n_replicas=4, first_replica=first, n_threads=4)
        assert_same(g2, o2, best_spins=False)


def test_config3_full_schedule_on_a_replica_subset():
    """100 x 100 torus, the complete 5000-sweep schedule for 16 replicas straddling a tile edge (ids 120..135)."""
    wl = W.config3()
    g = gpu_anneal(wl, n_replicas=16, first_replica=120)
    o = oracle_anneal(wl, n_replicas=16, first_replica=120, n_threads=16)
    assert_same(g, o)


def _oracle_replica_groups(wl, groups, thr, n_threads):
    """Oracle runs of contiguous replica ranges [(first, count), ...] -> {replica: (trace column, final spins, best cut, best sweep)}."""
    out = {}
    for first, count in groups:
        o = oracle_anneal(wl, thr=thr, n_replicas=count, first_replica=first, n_threads=min(n_threads, count))
        for k in range(count):
            out[first + k] = (o["trace"][:, k], o["final"][k], int(o["best_cut"][k]), int(o["best_sweep"][k]))
    return out


def test_config5_bench_configuration_full_schedule_sampled_replicas(cfg5):
    """SURVEY 8(c) sampling plan: the run bench.py times (all 32 replicas x all 500 sweeps, one ising_anneal call) compared
    with the oracle on replicas {0, 3, 4, 31}: every cut of the trace, the final spins, best cut and sweep."""
    import concurrent.futures as cf
    import torch
    wl = cfg5
    p = P.load_workload(wl)
    assert p.engine == P.ENGINE_GRID_TAIL_CHAIN
    trace = P.anneal_workload(p, wl, cut_trace=True)
    final = P.ising_current_state(p, wl.n_replicas)
    torch.cuda.synchronize()
    trace, final = trace.cpu().numpy(), final.cpu().numpy()
    reps = (0, 3, 4, 31)
    with cf.ThreadPoolExecutor(len(reps)) as ex:     # four single-thread oracle runs side by side (ctypes drops the GIL)
        res = list(ex.map(lambda r: _oracle_replica_groups(wl, [(r, 1)], wl.thr, 1)[r], reps))
    for r, (tr, fin, bc, bs) in zip(reps, res):
        np.testing.assert_array_equal(trace[:, r], tr)
        np.testing.assert_array_equal(final[r], fin)
        s, cut, sweep, rep = P.ising_best_state(p, r, want_spins=False)
        assert (cut, sweep) == (bc, bs)


def test_config4_bench_configuration_full_schedule_sampled_replicas():
    """K_4096 x 1024 replicas x 1000 Jacobi sweeps on the tcgen05 engine exactly as bench.py runs it (one cooperative launch):
    every replica for the first 3 sweeps, and replicas {0-7, 127, 128, 255, 256, 511, 512, 1016-1023} (tile and Philox-group
    edges) for the complete schedule (SURVEY 8(c) plan)."""
    import torch
    wl = W.config4()
    g3 = gpu_anneal(wl, thr=wl.thr[:3], want_best_spins=False)
    assert g3["problem"].has_dense_engine
    assert_same(g3, oracle_anneal(wl, thr=wl.thr[:3], n_threads=16), best_spins=False)
    p = g3["problem"]
    trace = P.anneal_workload(p, wl, cut_trace=True)
    final = P.ising_current_state(p, wl.n_replicas)
    torch.cuda.synchronize()
    trace, final = trace.cpu().numpy(), final.cpu().numpy()
    groups = [(0, 8), (127, 2), (255, 2), (511, 2), (1016, 8)]
    res = _oracle_replica_groups(wl, groups, wl.thr, 16)
    for r, (tr, fin, bc, bs) in res.items():
        np.testing.assert_array_equal(trace[:, r], tr)
        np.testing.assert_array_equal(final[r], fin)
        s, cut, sweep, rep = P.ising_best_state(p, r, want_spins=(r in (0, 1023)))
        assert (cut, sweep) == (bc, bs)
