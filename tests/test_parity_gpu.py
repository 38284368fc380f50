"""`-m gpu` parity tests: the CUDA path, called through the C ABI (binding.py), against the CPU
oracle on the same seeded inputs.  All quantities are integers, so the bar is BIT-EXACT:
the cut of every replica after every sweep, the final spin vectors, and the best cut / sweep /
state per replica (SURVEY 8(c) "Whole trajectory")."""
import ctypes

import numpy as np
import pytest

import paper_1807_10750_b200 as P
from paper_1807_10750_b200 import binding
from paper_1807_10750_b200 import workloads as W
from oracle import ising_oracle as O

from gpu_util import assert_same, gpu_anneal, oracle_anneal

pytestmark = pytest.mark.gpu


def wl_from_csr(n, csr, colour, nc, R, thr, mode="gs", seed=0, name="custom"):
    row_ptr, col, w = csr
    return W.Workload(name=name, n=n, row_ptr=row_ptr, col=col, w=w, colour=colour, n_colours=nc, n_replicas=R,
                      first_replica=0, seed=seed, thr=thr, mode=mode)


def er_workload(n, p, gseed, wkind, wdtype, R, M, colouring="index", mode="gs", seed=0, p0=0.1):
    u, v = W.erdos_renyi_edges(n, p, gseed)
    wt = W.weights_from_hash(W.hash_pairs(gseed, u, v), wkind)
    csr = W.csr_from_edges(n, u, v, wt, wdtype)
    if colouring:
        colour, nc = W.greedy_colouring(n, csr[0], csr[1], colouring)
    else:
        colour, nc = None, 0
    return wl_from_csr(n, csr, colour, nc, R, W.linear_schedule(p0, 0.0, M), mode=mode, seed=seed)


# ---------------------------------------------------------------------------------------------
# energy / cut reduction (a7) from the definition
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("device_inputs", [False, True])
def test_energy_cut_matches_oracle(device_inputs):
    import torch
    wl = er_workload(1500, 0.02, 11, "pm4", np.int8, 40, 4)
    p = P.load_workload(wl, max_replicas=40, device_inputs=device_inputs)
    spins = W.random_spins(5, 40, wl.n)
    E, cut = P.ising_energy_cut(p, torch.from_numpy(spins).cuda() if device_inputs else spins)
    oE, ocut = O.energy_cut(wl.n, wl.row_ptr, wl.col, wl.w, spins)
    np.testing.assert_array_equal(E.cpu().numpy(), oE)
    np.testing.assert_array_equal(cut.cpu().numpy(), ocut)
    assert p.w_total == wl.w_total
    # host output pointers
    e_h = np.zeros(40, dtype=np.int64)
    c_h = np.zeros(40, dtype=np.int64)
    st = binding.lib().ising_energy_cut(p.handle, spins.ctypes.data, 40, e_h.ctypes.data, c_h.ctypes.data, None)
    assert st == 0
    np.testing.assert_array_equal(e_h, oE)
    np.testing.assert_array_equal(c_h, ocut)


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs 1-3 (and a cut-down 5) : colour-class Gauss-Seidel
# ---------------------------------------------------------------------------------------------
def test_config1_full():
    wl = W.config1()
    g = gpu_anneal(wl)
    o = oracle_anneal(wl, n_threads=1)
    assert_same(g, o)
    assert g["trace"].shape == (1000, 1)


def test_config2_full():
    wl = W.config2()
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)


def test_config3_all_replicas_first_sweeps_and_some_replicas_longer():
    wl = W.config3()
    g = gpu_anneal(wl, thr=wl.thr[:150])
    o = oracle_anneal(wl, thr=wl.thr[:150])
    assert_same(g, o)
    # replicas straddling Philox groups / tiles, longer run (first_replica offsets, R = 3: ragged tile)
    for first in (0, 31, 126, 253):
        g = gpu_anneal(wl, thr=wl.thr[:1500], n_replicas=3, first_replica=first, problem=g["problem"])
        o = oracle_anneal(wl, thr=wl.thr[:1500], n_replicas=3, first_replica=first)
        assert_same(g, o)


def test_config3_all_plus_torus_reaches_known_max_cut():
    """Even torus with all weights +1: max cut = #E = 2 L^2 = 20000 (SURVEY 8(c) closed forms)."""
    wl = W.config3(all_plus=True)
    p = P.load_workload(wl)
    P.anneal_workload(p, wl)
    s, cut, sweep, rep = P.ising_best_state(p, -1)
    assert cut == 20000
    E, c = P.ising_energy_cut(p, s.reshape(1, -1))
    assert int(c[0]) == 20000 and int(E[0]) == wl.w_total - 2 * 20000
    # the recorded best must be the checkerboard (or its negation)
    s = s.cpu().numpy()
    assert np.all(s == s[0] * np.where(wl.colour == wl.colour[0], 1, -1))
    # first sweeps agree with the oracle for every replica
    g = gpu_anneal(wl, thr=wl.thr[:40], problem=p)
    o = oracle_anneal(wl, thr=wl.thr[:40])
    assert_same(g, o)


@pytest.mark.parametrize("colouring", ["ldf", "index"])
def test_config5_cutdown(colouring):
    wl = W.config5(n=30000, sweeps=40, replicas=32, colouring=colouring)
    assert np.diff(wl.row_ptr).max() > 1024     # hub rows: warp-per-row slices
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)


# ---------------------------------------------------------------------------------------------
# Jacobi on the sparse path (dense engine disabled), racy mode invariants
# ---------------------------------------------------------------------------------------------
def test_jacobi_sparse_path():
    wl = er_workload(3000, 0.004, 21, "pm4", np.int8, 40, 60, colouring=None, mode="jacobi", seed=3)
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)
    wl = W.config4(n=200, sweeps=30, replicas=37)
    g = gpu_anneal(wl, flags=P.ISING_LOAD_NO_DENSE)
    o = oracle_anneal(wl)
    assert_same(g, o)
    assert not g["problem"].has_dense_engine


def test_jacobi_two_cycle_on_all_plus_bipartite():
    """Zero-temperature Jacobi from all +1 on a bipartite all-(+1) graph oscillates with cut 0."""
    wl = W.config3(L=20, sweeps=6, replicas=2, all_plus=True)
    init = np.ones((2, wl.n), dtype=np.int8)
    g = gpu_anneal(wl, thr=np.zeros(6, dtype=np.uint32), mode=P.ISING_MODE_JACOBI, init_spins=init)
    assert np.all(g["trace"] == 0)
    assert np.all(g["final"] == 1)      # even number of sweeps: back to all +1


def test_racy_mode_invariants():
    wl = W.config2(sweeps=200, replicas=8)
    p = P.load_workload(wl)
    trace = P.anneal_workload(p, wl, mode=P.ISING_MODE_RACY, cut_trace=True)
    final = P.ising_current_state(p, 8).cpu().numpy()
    assert set(np.unique(final)) <= {-1, 1}
    E, cut = P.ising_energy_cut(p, final)
    np.testing.assert_array_equal(cut.cpu().numpy(), trace.cpu().numpy()[-1])
    for r in range(8):
        s, c, sw, _ = P.ising_best_state(p, r)
        _, c2 = P.ising_energy_cut(p, s.reshape(1, -1))
        assert int(c2[0]) == c == int(trace[:, r].max())


# ---------------------------------------------------------------------------------------------
# semantics: tie rule, replica / sweep split, given init, wide weights, degenerate graphs
# ---------------------------------------------------------------------------------------------
def test_tie_rule_keep():
    wl = W.config3(L=30, sweeps=80, replicas=5, all_plus=True)
    g = gpu_anneal(wl, tie_rule=1)
    o = oracle_anneal(wl, tie_rule=1)
    assert_same(g, o)
    assert not np.array_equal(g["final"], gpu_anneal(wl, tie_rule=0)["final"])


@pytest.mark.parametrize("first", [1, 2, 3, 6, 33])
def test_first_replica_not_multiple_of_four(first):
    wl = er_workload(600, 0.03, 31, "pm1", np.int8, 7, 50)
    g = gpu_anneal(wl, first_replica=first)
    o = oracle_anneal(wl, first_replica=first)
    assert_same(g, o)


def test_batch_split_and_sweep_split_invariance():
    wl = er_workload(900, 0.02, 41, "pm4", np.int8, 35, 60)
    full = gpu_anneal(wl)
    p = full["problem"]
    # R batch == R singles with first_replica = r
    for r in (0, 5, 34):
        one = gpu_anneal(wl, n_replicas=1, first_replica=r, problem=p)
        np.testing.assert_array_equal(one["final"][0], full["final"][r])
        np.testing.assert_array_equal(one["trace"][:, 0], full["trace"][:, r])
    # 0..M == 0..k then k..M with init continue and sweep_offset
    k = 23
    a = gpu_anneal(wl, thr=wl.thr[:k], problem=p)
    b = gpu_anneal(wl, thr=wl.thr[k:], sweep_offset=k, init_mode=P.ISING_INIT_CONTINUE, problem=p)
    np.testing.assert_array_equal(np.vstack([a["trace"], b["trace"]]), full["trace"])
    np.testing.assert_array_equal(b["final"], full["final"])
    o = oracle_anneal(wl)
    assert_same(full, o)


def test_given_init_host_and_device():
    import torch
    wl = er_workload(700, 0.02, 51, "pm4", np.int8, 9, 30)
    init = W.random_spins(9, 9, wl.n)
    o = oracle_anneal(wl, init_spins=init)
    assert_same(gpu_anneal(wl, init_spins=init), o)
    assert_same(gpu_anneal(wl, init_spins=torch.from_numpy(init).cuda()), o)
    bad = init.copy()
    bad[3, 17] = 0
    with pytest.raises(P.IsingError) as e:
        gpu_anneal(wl, init_spins=bad)
    assert e.value.status == 13


def test_wide_int32_weights():
    n = 500
    u, v = W.erdos_renyi_edges(n, 0.05, 61)
    h = W.hash_pairs(61, u, v)
    wt = ((h >> np.uint64(8)) % np.uint64(200001)).astype(np.int64) - 100000     # |w| up to 1e5
    csr = W.csr_from_edges(n, u, v, wt, np.int32)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "index")
    wl = wl_from_csr(n, csr, colour, nc, 6, W.linear_schedule(0.2, 0.0, 40), seed=9)
    assert_same(gpu_anneal(wl), oracle_anneal(wl))
    wlj = wl_from_csr(n, csr, None, 0, 6, W.linear_schedule(0.2, 0.0, 20), mode="jacobi", seed=9)
    assert_same(gpu_anneal(wlj), oracle_anneal(wlj))


def test_isolated_vertices_and_empty_graph():
    n = 70
    u = np.array([0, 3, 3], dtype=np.int64)
    v = np.array([3, 5, 69], dtype=np.int64)
    csr = W.csr_from_edges(n, u, v, np.array([2, -3, 1]), np.int8)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "index")
    wl = wl_from_csr(n, csr, colour, nc, 3, W.linear_schedule(0.3, 0.0, 12), seed=4)
    assert_same(gpu_anneal(wl), oracle_anneal(wl))
    empty = (np.zeros(n + 1, dtype=np.int64), np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.int8))
    wl = wl_from_csr(n, empty, np.zeros(n, dtype=np.int32), 1, 2, W.linear_schedule(0.3, 0.0, 5), seed=4)
    g = gpu_anneal(wl)
    assert_same(g, oracle_anneal(wl))
    assert np.all(g["trace"] == 0)


def test_device_relabelling_with_more_degree_runs_than_the_first_read_back():
    """a1 relabels on the device (radix sort of the rows by colour, degree) and reads back only the runs of equal
    (colour, degree); more than 32 768 runs take a second copy.  A ring in which every vertex has a colour of its own
    (a proper colouring) has one run per vertex; also a load from device-resident inputs."""
    n = 40000
    u = np.arange(n, dtype=np.int64)
    v = (u + 1) % n
    wt = W.weights_from_hash(W.hash_pairs(5, np.minimum(u, v), np.maximum(u, v)), "pm4")
    csr = W.csr_from_edges(n, u, v, wt, np.int8)
    colour = np.random.default_rng(1).permutation(n).astype(np.int32)
    wl = wl_from_csr(n, csr, colour, n, 2, W.linear_schedule(0.2, 0.0, 2), seed=8)
    o = oracle_anneal(wl)
    assert_same(gpu_anneal(wl), o)
    assert_same(gpu_anneal(wl, device_inputs=True), o)


def test_n_sweeps_zero_only_initialises():
    wl = er_workload(300, 0.05, 71, "pm1", np.int8, 4, 0)
    g = gpu_anneal(wl, thr=np.zeros(0, dtype=np.uint32))
    o = oracle_anneal(wl, thr=np.zeros(0, dtype=np.uint32))
    np.testing.assert_array_equal(g["final"], o["final"])


# ---------------------------------------------------------------------------------------------
# error behaviour of ising_load_csr / ising_anneal
# ---------------------------------------------------------------------------------------------
def _load_status(row_ptr, col, w, colour=None, nc=0, R=1, ws=None):
    try:
        P.ising_load_csr(row_ptr, col, w, colour, nc, R, workspace_bytes=ws)
    except P.IsingError as e:
        return e.status
    return 0


def test_load_errors():
    n = 6
    u = np.array([0, 1, 2], dtype=np.int64)
    v = np.array([1, 2, 3], dtype=np.int64)
    rp, col, w = W.csr_from_edges(n, u, v, np.array([1, 2, 3]), np.int8)
    assert _load_status(rp, col, w) == 0
    a = w.copy(); a[0] = 5
    assert _load_status(rp, col, a) == 5                      # asymmetric weight
    c2 = col.copy(); c2[0] = 0
    assert _load_status(rp, c2, w) in (4, 5)                  # self loop
    rp2 = rp.copy(); rp2[2] = rp2[3] + 1
    assert _load_status(rp2, col, w) == 2                     # row_ptr not monotone
    c3 = col.copy(); c3[1], c3[2] = c3[2], c3[1]              # row 1 = (0, 2) -> (2, 0)
    assert _load_status(rp, c3, w) == 3
    c4 = col.copy(); c4[0] = 99
    assert _load_status(rp, c4, w) == 2
    good = np.array([0, 1, 0, 1, 0, 0], dtype=np.int32)
    assert _load_status(rp, col, w, good, 2) == 0
    bad = np.array([0, 0, 1, 0, 0, 0], dtype=np.int32)
    assert _load_status(rp, col, w, bad, 2) == 6              # neighbours share a colour
    assert _load_status(rp, col, w, good, 1) == 6             # colour out of range
    assert _load_status(rp, col, w, ws=64) == 9               # workspace too small
    assert _load_status(rp, col, w, R=0) == 8
    big = np.full(col.shape, 2**30, dtype=np.int32)
    assert _load_status(rp, col, big) == 7                    # sum_j |w_ij| >= 2^31
    p = P.ising_load_csr(rp, col, w)
    with pytest.raises(P.IsingError) as e:
        P.ising_anneal(p, np.zeros(3, dtype=np.uint32), mode=P.ISING_MODE_GS)
    assert e.value.status == 10
    with pytest.raises(P.IsingError) as e:
        P.ising_anneal(p, np.zeros(3, dtype=np.uint32), mode=P.ISING_MODE_JACOBI, n_replicas=2)
    assert e.value.status == 8
    with pytest.raises(P.IsingError) as e:
        P.ising_best_state(p, 0)
    assert e.value.status == 14


def _drop_entry(rp, col, w, i, j):
    """CSR without the directed entry (i, j)."""
    at = int(rp[i]) + int(np.searchsorted(col[rp[i]:rp[i + 1]], j))
    assert col[at] == j
    rp2 = rp.copy(); rp2[i + 1:] -= 1
    return rp2, np.delete(col, at), np.delete(w, at)


def test_asymmetry_is_found_whichever_row_is_longer():
    """k_validate looks an entry (i, j) up only in rows j that are not longer than row i and counts the entries of the two
    other kinds against each other (builder.cuh): a missing mirror must be reported from either side, also between rows
    of equal length, and so must a mirror with another weight."""
    n = 40
    u = np.concatenate([np.zeros(30, dtype=np.int64), np.array([31, 32, 33, 34])])      # a hub (0 - 1..30), a path 31-32-33-34-35
    v = np.concatenate([np.arange(1, 31, dtype=np.int64), np.array([32, 33, 34, 35])])
    wt = np.arange(1, 35) % 7 + 1
    rp, col, w = W.csr_from_edges(n, u, v, wt, np.int8)
    assert _load_status(rp, col, w) == 0
    assert _load_status(*_drop_entry(rp, col, w, 0, 7)) == 5       # the entry in the LONG row is missing
    assert _load_status(*_drop_entry(rp, col, w, 7, 0)) == 5       # the entry in the SHORT row is missing
    assert _load_status(*_drop_entry(rp, col, w, 32, 33)) == 5     # rows of equal length (the path's inner vertices)
    assert _load_status(*_drop_entry(rp, col, w, 33, 32)) == 5
    for (i, j) in [(0, 7), (7, 0), (32, 33)]:
        a = w.copy()
        a[int(rp[i]) + int(np.searchsorted(col[rp[i]:rp[i + 1]], j))] += 1
        assert _load_status(rp, col, a) == 5


def test_run_twice_is_bit_identical():
    wl = W.config5(n=20000, sweeps=25, replicas=32)
    a = gpu_anneal(wl)
    b = gpu_anneal(wl, problem=a["problem"])
    assert_same(a, b)


# ---------------------------------------------------------------------------------------------
# persistent-kernel corner cases: hub rows x several replica tiles x ragged replica count, more
# replicas than one persistent launch holds (1024), schedules longer than one threshold chunk
# ---------------------------------------------------------------------------------------------
def test_hub_rows_with_several_tiles_and_ragged_replicas():
    wl = W.config5(n=12000, sweeps=12, replicas=75)
    deg = np.diff(wl.row_ptr)
    assert (deg > 256).sum() > 5 and deg.max() > 1024     # hub rows cut into several parts each
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)
    # Jacobi and evaluation share the part logic
    g = gpu_anneal(wl, mode=P.ISING_MODE_JACOBI, thr=wl.thr[:5], n_replicas=40)
    o = oracle_anneal(wl, mode=1, thr=wl.thr[:5], n_replicas=40)
    assert_same(g, o)


def hub_graph(n, p, gseed, hub_degrees):
    """Sparse Erdos-Renyi background plus a few hub vertices (ids 0, 1, ...) of the given degrees."""
    u, v = W.erdos_renyi_edges(n, p, gseed)
    us, vs = [u], [v]
    for hid, d in enumerate(hub_degrees):
        others = np.arange(len(hub_degrees), n, dtype=np.int64)
        order = np.argsort(W.hash_pairs(gseed + 7 * hid + 1, np.full(others.size, hid, dtype=np.int64), others), kind="stable")
        us.append(np.full(d, hid, dtype=np.int64))
        vs.append(np.sort(others[order[:d]]))
    key = np.unique(np.concatenate(us) * n + np.concatenate(vs))
    return key // n, key % n


def test_hub_parts_with_wide_weights_gs_and_jacobi():
    """Hub rows cut into parts on the int32-weight path (32-bit RED + arrival counter instead of the packed
    64-bit atomic of the int8 path), Gauss-Seidel (launch per phase) and Jacobi, three replica tiles."""
    n = 4000
    u, v = hub_graph(n, 0.002, 71, [1500, 700, 300, 130])
    h = W.hash_pairs(71, u, v)
    wt = ((h >> np.uint64(8)) % np.uint64(60001)).astype(np.int64) - 30000
    wt[wt == 0] = 1
    csr = W.csr_from_edges(n, u, v, wt, np.int32)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "ldf")
    wl = wl_from_csr(n, csr, colour, nc, 70, W.linear_schedule(0.2, 0.0, 12), seed=5)
    assert_same(gpu_anneal(wl), oracle_anneal(wl))
    wlj = wl_from_csr(n, csr, None, 0, 70, W.linear_schedule(0.2, 0.0, 8), mode="jacobi", seed=5)
    assert_same(gpu_anneal(wlj), oracle_anneal(wlj))


@pytest.mark.parametrize("sign", [1, -1])
def test_hub_parts_extreme_int8_partial_sums(sign):
    """All weights +-127 and all spins +1: every hub part adds the largest partial sum the packed arrival
    word has to hold (128 edges x 127 in latency-bound phases); zero-temperature sweeps from there."""
    n = 3000
    u, v = hub_graph(n, 0.001, 73, [2900, 2000, 515, 129])
    wt = np.full(u.size, 127 * sign, dtype=np.int64)
    csr = W.csr_from_edges(n, u, v, wt, np.int8)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "index")
    thr = np.zeros(4, dtype=np.uint32)
    wl = wl_from_csr(n, csr, colour, nc, 33, thr, seed=2)
    init = np.ones((33, n), dtype=np.int8)
    g = gpu_anneal(wl, init_spins=init)
    o = oracle_anneal(wl, init_spins=init)
    assert_same(g, o)


def test_config5_midsize_uses_both_sub_row_lengths():
    """300k spins: the big colour phases take 16-edge sub-rows with tail cells and 256-edge hub parts, the small
    ones 8-edge sub-rows and 128-edge parts (chosen per phase at load)."""
    wl = W.config5(n=300000, sweeps=5, replicas=32)
    g = gpu_anneal(wl, want_best_spins=False)
    assert g["problem"].info(9) > 148 * 16            # more slice units than warps on the GPU
    o = oracle_anneal(wl)
    assert_same(g, o, best_spins=False)


ENGINE_FLAGS = {
    "small": 0,                                                     # whole graph inside one CTA per four replicas
    "cluster": P.ISING_LOAD_NO_SMALL,                                # one thread-block cluster per replica tile
    "grid": P.ISING_LOAD_NO_SMALL | P.ISING_LOAD_NO_CLUSTER | P.ISING_LOAD_NO_TAIL_CHAIN,   # cooperative grid, every class a phase
    "grid+tail": P.ISING_LOAD_NO_SMALL | P.ISING_LOAD_NO_CLUSTER,    # cooperative grid, last classes as a shared-memory chain
    # ... and without the chain overlap (class 0 in one piece, the chain step on its own)
    "grid+tail-overlap": P.ISING_LOAD_NO_SMALL | P.ISING_LOAD_NO_CLUSTER | P.ISING_LOAD_NO_OVERLAP,
}
ENGINE_CODE = {"small": P.ENGINE_SMALL, "cluster": P.ENGINE_CLUSTER, "grid": P.ENGINE_GRID, "grid+tail": P.ENGINE_GRID_TAIL_CHAIN,
               "grid+tail-overlap": P.ENGINE_GRID_TAIL_CHAIN}


@pytest.mark.parametrize("engine", ["small", "cluster", "grid"])
def test_small_graph_through_every_gauss_seidel_engine(engine):
    """A small graph runs wholly inside one CTA per four replicas (shared-memory chain); load flags force the
    cluster and the cooperative-grid variants of the persistent kernel.  All must match the oracle, also with several
    tiles, a ragged replica count, KEEP ties and a continued run."""
    wl = er_workload(900, 0.015, 67, "pm4", np.int8, 75, 40, seed=6, p0=0.2)
    g = gpu_anneal(wl, tie_rule=1, flags=ENGINE_FLAGS[engine])
    assert g["problem"].engine == ENGINE_CODE[engine]
    o = oracle_anneal(wl, tie_rule=1)
    assert_same(g, o)
    g1 = gpu_anneal(wl, thr=wl.thr[:15], problem=g["problem"])
    g2 = gpu_anneal(wl, thr=wl.thr[15:], sweep_offset=15, init_mode=P.ISING_INIT_CONTINUE, problem=g["problem"])
    np.testing.assert_array_equal(g2["final"], oracle_anneal(wl)["final"])


@pytest.mark.parametrize("engine", ["grid", "grid+tail", "grid+tail-overlap"])
@pytest.mark.parametrize("replicas,first", [(32, 0), (70, 5)])
def test_power_law_graph_with_and_without_tail_chain(engine, replicas, first):
    """Config-5-shaped graph: the last colour classes (few hub rows each) run as a shared-memory chain after one bulk
    pseudo-phase (with the chain-free rows of class 0 of the next sweep updated beside the chain, or without that
    overlap), or as grid-wide phases.  Ragged replica count over several tiles, a first replica that is not a
    multiple of four (two Philox calls per word), KEEP ties, trace / best state, and a continued run."""
    wl = W.config5(n=120000, sweeps=9, replicas=replicas)
    g = gpu_anneal(wl, first_replica=first, tie_rule=1, flags=ENGINE_FLAGS[engine])
    assert g["problem"].engine == ENGINE_CODE[engine]
    if engine.startswith("grid+tail"):
        assert 0 < g["problem"].info(14) <= 12288 and g["problem"].info(15) < wl.n_colours
        assert (g["problem"].info(19) > 0) == (engine == "grid+tail")   # rows of the overlapped part of class 0
    o = oracle_anneal(wl, first_replica=first, tie_rule=1, n_threads=16)
    assert_same(g, o)
    g1 = gpu_anneal(wl, thr=wl.thr[:4], first_replica=first, problem=g["problem"], want_best_spins=False)
    g2 = gpu_anneal(wl, thr=wl.thr[4:], sweep_offset=4, first_replica=first, init_mode=P.ISING_INIT_CONTINUE,
                    problem=g["problem"], want_best_spins=False)
    np.testing.assert_array_equal(g2["final"], oracle_anneal(wl, first_replica=first, n_threads=16)["final"])


def test_chain_overlap_layout_with_more_tiles_than_the_overlap_takes():
    """The overlap split of class 0 is part of the loaded layout, but a launch overlaps only while the chain CTAs are at
    most half the grid (8 per tile): 10 tiles run the split layout with the chain step on its own, and a later call with
    few replicas on the same handle overlaps again.  Both must match the oracle."""
    wl = W.config5(n=70000, sweeps=4, replicas=300)
    g = gpu_anneal(wl, want_best_spins=False)
    assert g["problem"].engine == P.ENGINE_GRID_TAIL_CHAIN and g["problem"].info(19) > 0
    o = oracle_anneal(wl, n_threads=16)
    assert_same(g, o, best_spins=False)
    g2 = gpu_anneal(wl, n_replicas=40, problem=g["problem"])
    o2 = oracle_anneal(wl, n_replicas=40, n_threads=16)
    assert_same(g2, o2)


@pytest.mark.parametrize("flags", [0, P.ISING_LOAD_NO_CLUSTER])
def test_small_graph_flip_producer_with_zero_threshold_sweeps(flags):
    """Small-graph engine as a cluster of two CTAs per word (levels + flip producer) and as one CTA per word: sweeps
    whose threshold is 0 draw nothing and hand no buffer over (both CTAs must keep the same count), a first replica
    that is not a multiple of four takes two Philox calls per word, and a call continues where the last one stopped."""
    wl = er_workload(700, 0.02, 91, "pm4", np.int8, 7, 24, seed=3, p0=0.3)
    thr = wl.thr.copy()
    thr[[0, 3, 4, 9, 10, 11, 17, 23]] = 0
    g = gpu_anneal(wl, thr=thr, first_replica=5, flags=flags)
    assert g["problem"].engine == P.ENGINE_SMALL and g["problem"].info(18) == (1 if flags else 2)
    o = oracle_anneal(wl, thr=thr, first_replica=5)
    assert_same(g, o)
    g1 = gpu_anneal(wl, thr=thr[:10], first_replica=5, problem=g["problem"])
    g2 = gpu_anneal(wl, thr=thr[10:], sweep_offset=10, first_replica=5, init_mode=P.ISING_INIT_CONTINUE, problem=g["problem"])
    np.testing.assert_array_equal(g2["final"], o["final"])


def test_small_graph_with_more_than_16k_rows_keeps_local_ids_in_its_cells():
    """Chains of at most 16 384 rows keep byte offsets (id x 4) in their 16-bit cells; longer ones (the paper's largest
    benchmark graphs have 20 000 vertices, Table III) keep local ids: the other instance of the kernel."""
    wl = er_workload(20000, 0.0002, 13, "pm4", np.int8, 6, 10, seed=2, p0=0.2)
    g = gpu_anneal(wl)
    assert g["problem"].engine == P.ENGINE_SMALL
    o = oracle_anneal(wl, n_threads=8)
    assert_same(g, o)


def test_small_graph_streamed_through_shared_memory():
    """A graph whose packed edges do not fit one CTA's shared memory but whose spins do: the chain engine streams the
    edge chunks through two buffers every sweep (several chunks, levels cut across chunks)."""
    wl = er_workload(6000, 0.008, 71, "pm4", np.int8, 8, 12, seed=9, p0=0.2)    # ~290k directed edges: ~0.9 MB of cells
    g = gpu_anneal(wl)
    assert g["problem"].engine == P.ENGINE_SMALL and g["problem"].info(17) == 0 and g["problem"].info(16) > 2
    o = oracle_anneal(wl, n_threads=8)
    assert_same(g, o)


def test_more_replicas_than_one_persistent_launch():
    wl = er_workload(300, 0.05, 23, "pm4", np.int8, 1100, 6, p0=0.3)
    g = gpu_anneal(wl, want_best_spins=False)
    o = oracle_anneal(wl)
    assert_same(g, o, best_spins=False)
    s, cut, sweep, rep = P.ising_best_state(g["problem"], 1077)
    np.testing.assert_array_equal(s.cpu().numpy(), o["best_spins"][1077])


def test_schedule_longer_than_one_threshold_chunk():
    wl = er_workload(24, 0.3, 29, "pm1", np.int8, 3, 70000, p0=0.05)
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)


def test_phase_timing_diagnostics_do_not_change_results():
    wl = W.config5(n=8000, sweeps=6, replicas=32)
    p = P.load_workload(wl, flags=ENGINE_FLAGS["grid+tail"])
    stamps = p.phase_timing(2)
    g = gpu_anneal(wl, problem=p)
    o = oracle_anneal(wl)
    assert_same(g, o)
    t = stamps.cpu().numpy()
    assert t.shape == (p.info(15) + 1, p.info(12), 8)   # 0/1: barrier arrive / leave, per virtual phase (+ the chain)
    rows = p.info(15) + (1 if p.engine == P.ENGINE_GRID_TAIL_CHAIN else 0)
    assert (t[:rows, :, 1] >= t[:rows, :, 0]).all() and (t[:rows, :, 0] > 0).all()


def test_edge_list_file_workload(tmp_path):
    """a graph read from an edge-list text file (synthetic content) through the same path."""
    n = 700
    u, v = hub_graph(n, 0.01, 97, [300])
    wt = W.weights_from_hash(W.hash_pairs(97, u, v), "pm8")
    path = tmp_path / "graph.txt"
    path.write_text("%d %d\n" % (n, u.size) + "".join("%d %d %d\n" % (a + 1, b + 1, c) for a, b, c in zip(u, v, wt)))
    wl = W.load_edge_list(str(path), replicas=36, sweeps=30, p0=0.15)
    assert_same(gpu_anneal(wl), oracle_anneal(wl))


def test_external_field_through_the_auxiliary_spin():
    """an external field (eq. (1)-(3)) enters as one auxiliary vertex coupled to every spin with a
    non-zero field (a hub of degree ~n); the augmented graph runs through the unchanged path."""
    from paper_1807_10750_b200 import frontdoor as F
    n = 3000
    u, v = W.erdos_renyi_edges(n, 0.004, 101)
    w = W.weights_from_hash(W.hash_pairs(101, u, v), "pm4")
    f = (W.rand_u64(101, 3, n) % np.uint64(9)).astype(np.int64) - 4
    wl = F.field_workload(n, u, v, w, f, replicas=33, sweeps=25, p0=0.2)
    g = gpu_anneal(wl)
    o = oracle_anneal(wl)
    assert_same(g, o)
    r = int(np.argmax(g["best_cut"]))
    s = F.decode_field_solution(g["best_spins"][r])
    assert F.field_energy(n, u, v, w, f, s) == wl.w_total - 2 * int(g["best_cut"][r])


# ---------------------------------------------------------------------------------------------
# Algorithm 1: minimisation sweep + exactly N distinct flips per replica
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("R", [5, 70])
def test_exact_n_mode_matches_oracle(R):
    wl = er_workload(1200, 0.01, 53, "pm4", np.int8, R, 1, seed=4)
    counts = np.array([200, 150, 100, 64, 33, 7, 1, 0, 0, 4096], dtype=np.uint32)    # the last one is clamped to n
    g = gpu_anneal(wl, thr=counts, mode=P.ISING_MODE_EXACT_N)
    o = oracle_anneal(wl, thr=counts, mode=2)
    assert_same(g, o)
    # sweep split and first_replica: the draws are keyed on (draw index, absolute sweep, replica)
    g1 = gpu_anneal(wl, thr=counts[:4], mode=P.ISING_MODE_EXACT_N, n_replicas=3, first_replica=2)
    g2 = gpu_anneal(wl, thr=counts[4:], mode=P.ISING_MODE_EXACT_N, n_replicas=3, first_replica=2, sweep_offset=4,
                    init_mode=P.ISING_INIT_CONTINUE, problem=g1["problem"])
    np.testing.assert_array_equal(g2["final"], o["final"][2:5])


def test_exact_n_mode_on_a_hub_graph():
    wl = W.config5(n=20000, sweeps=1, replicas=32)
    counts = np.array([300, 100, 10, 0], dtype=np.uint32)
    g = gpu_anneal(wl, thr=counts, mode=P.ISING_MODE_EXACT_N)
    o = oracle_anneal(wl, thr=counts, mode=2)
    assert_same(g, o)
    with pytest.raises(P.IsingError):
        gpu_anneal(wl, thr=np.array([5000], dtype=np.uint32), mode=P.ISING_MODE_EXACT_N, problem=g["problem"])


# ---------------------------------------------------------------------------------------------
# dense tcgen05 engine (a8): K_n instances in Jacobi mode, J.S on the int8 tensor cores
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,R,M", [(192, 40, 10), (300, 300, 6), (128, 256, 4), (520, 70, 5)])
def test_dense_engine_matches_oracle(n, R, M):
    wl = W.config4(n=n, sweeps=M, replicas=R)
    g = gpu_anneal(wl)
    assert g["problem"].has_dense_engine
    o = oracle_anneal(wl)
    assert_same(g, o)
    # the dense state is readable through the definition-based energy / cut as well
    E, cut = P.ising_energy_cut(g["problem"], None, n_replicas=R)
    np.testing.assert_array_equal(cut.cpu().numpy(), o["trace"][-1])


def test_dense_engine_equals_sparse_jacobi_path():
    wl = W.config4(n=260, sweeps=8, replicas=48)
    g = gpu_anneal(wl, first_replica=5, tie_rule=P.ISING_TIE_KEEP)
    s = gpu_anneal(wl, first_replica=5, tie_rule=P.ISING_TIE_KEEP, flags=P.ISING_LOAD_NO_DENSE)
    assert g["problem"].has_dense_engine and not s["problem"].has_dense_engine
    assert_same(g, s)
    o = oracle_anneal(wl, first_replica=5, tie_rule=1)
    assert_same(g, o)


def test_dense_engine_continue_and_mode_switch():
    wl = W.config4(n=200, sweeps=9, replicas=33)
    p = P.load_workload(wl)
    a = gpu_anneal(wl, thr=wl.thr[:4], problem=p)
    b = gpu_anneal(wl, thr=wl.thr[4:], sweep_offset=4, problem=p, init_mode=P.ISING_INIT_CONTINUE)
    o = oracle_anneal(wl)
    np.testing.assert_array_equal(np.concatenate([a["trace"], b["trace"]]), o["trace"])
    np.testing.assert_array_equal(b["final"], o["final"])
