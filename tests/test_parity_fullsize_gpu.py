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
