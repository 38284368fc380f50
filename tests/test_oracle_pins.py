"""Pins for the CPU oracle (oracle/ising_oracle.cpp) -- `-m "not gpu"`.

Every test checks the oracle against something OTHER than itself: published
known-answer vectors, the definition of the cut written independently in numpy,
brute force over all 2^n states, closed forms (torus, K_n, bipartite), and the
invariants the method's definition implies (SURVEY.md 8(c) "What pins each part").
Citations are PAPER.md lines.
"""
import itertools
import os

import numpy as np
import pytest

from paper_1807_10750_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------
# helpers written independently of the oracle (numpy only)
# ----------------------------------------------------------------------------
def edges_of(wl_or_tuple):
    """(u, v, w) for u<v from a symmetric CSR."""
    row_ptr, col, w = wl_or_tuple
    n = row_ptr.shape[0] - 1
    src = np.repeat(np.arange(n), np.diff(row_ptr))
    m = src < col
    return src[m], col[m].astype(np.int64), w[m].astype(np.int64)


def cut_by_definition(csr, s):
    """eq. (4) read as 'total weight of edges whose endpoints are on different sides' (L117)."""
    u, v, w = edges_of(csr)
    s = np.asarray(s, dtype=np.int64)
    return int(w[s[u] != s[v]].sum())


def small_graph(n, p, seed, wkind="pm4", wdtype=np.int8):
    u, v = W.erdos_renyi_edges(n, p, seed)
    wt = W.weights_from_hash(W.hash_pairs(seed, u, v), wkind)
    return W.csr_from_edges(n, u, v, wt, wdtype)


def all_states(n):
    codes = np.arange(1 << n, dtype=np.int64)
    return (((codes[:, None] >> np.arange(n)[None, :]) & 1) * 2 - 1).astype(np.int8)


# ----------------------------------------------------------------------------
# Philox4x32-10 (reading Q11; "cuRAND")
# ----------------------------------------------------------------------------
def test_philox_known_answers(oracle):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_is_a_bijection_of_the_counter(oracle):
    # distinct counters under one key never collide (Philox is a keyed permutation)
    outs = {tuple(int(x) for x in oracle.philox4x32_10([c, 7, 1, 0], [5, 9])) for c in range(2000)}
    assert len(outs) == 2000


# ----------------------------------------------------------------------------
# energy / cut: eq. (3)-(5) L51, L119, L128; reading Q1, Q9
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("wkind,wdtype", [("pm4", np.int8), ("pm8", np.int32), ("+1", np.int32)])
def test_cut_identity_against_definition(oracle, wkind, wdtype):
    n = 60
    csr = small_graph(n, 0.2, 11, wkind, wdtype)
    spins = W.random_spins(3, 5, n)
    E, cut = oracle.energy_cut(n, *csr, spins)
    u, v, w = edges_of(csr)
    Wtot = int(w.sum())
    for r in range(5):
        c_def = cut_by_definition(csr, spins[r])
        assert int(cut[r]) == c_def
        assert 2 * c_def == Wtot - int(E[r])                      # cut = (W - E)/2
        assert int(E[r]) == int((w * spins[r][u].astype(np.int64) * spins[r][v]).sum())
    # global spin flip symmetry
    E2, cut2 = oracle.energy_cut(n, *csr, -spins)
    assert (E2 == E).all() and (cut2 == cut).all()


@pytest.mark.parametrize("n,seed", [(10, 1), (14, 2), (16, 3)])
def test_bruteforce_against_numpy_enumeration(oracle, n, seed):
    csr = small_graph(n, 0.45, seed, "pm4")
    u, v, w = edges_of(csr)
    S = all_states(n).astype(np.int64)
    cuts = ((S[:, u] != S[:, v]) * w[None, :]).sum(axis=1)
    mc, arg = oracle.bruteforce_maxcut(n, *csr)
    assert mc == int(cuts.max())
    assert cut_by_definition(csr, arg) == mc
    # the annealer never reports more than the true maximum, and what it reports is the cut of its state
    colour, nc = W.greedy_colouring(n, csr[0], csr[1])
    res = oracle.anneal(n, *csr, order=oracle.order_from_colour(colour), n_replicas=6, seed=seed,
                        thr=W.linear_schedule(0.3, 0.0, 60))
    assert (res["trace"] <= mc).all()
    for r in range(6):
        assert cut_by_definition(csr, res["best_spins"][r]) == int(res["best_cut"][r])
        assert cut_by_definition(csr, res["final"][r]) == int(res["trace"][-1, r])


def test_annealer_finds_small_optimum(oracle):
    # heuristic, but on 12 vertices with 32 replicas and 200 sweeps the optimum is always found
    n = 12
    csr = small_graph(n, 0.5, 5, "pm4")
    mc, _ = oracle.bruteforce_maxcut(n, *csr)
    colour, _ = W.greedy_colouring(n, csr[0], csr[1])
    res = oracle.anneal(n, *csr, order=oracle.order_from_colour(colour), n_replicas=32, seed=1,
                        thr=W.linear_schedule(0.3, 0.0, 200))
    assert int(res["best_cut"].max()) == mc


# ----------------------------------------------------------------------------
# local update, eq. (2) L45-49 with reading Q1/Q3, on hand-made graphs
# ----------------------------------------------------------------------------
def _csr(n, edges):
    u = np.array([e[0] for e in edges], dtype=np.int64)
    v = np.array([e[1] for e in edges], dtype=np.int64)
    w = np.array([e[2] for e in edges], dtype=np.int64)
    return W.csr_from_edges(n, u, v, w, np.int32)


def test_single_edge_update_rule(oracle):
    zero = np.zeros(1, dtype=np.uint32)
    order = np.array([0, 1], dtype=np.int32)
    # w=+1: from (+,+): vertex 0 sees h=+1 -> -1; vertex 1 then sees h=-1 -> +1: edge is cut
    res = oracle.anneal(2, *_csr(2, [(0, 1, 1)]), order=order, thr=zero, init_spins=[[1, 1]])
    assert res["final"].tolist() == [[-1, 1]] and res["trace"].tolist() == [[1]]
    # w=-1 (cutting it costs): from (+,-): vertex 0 sees h=+1 -> -1; vertex 1 sees h=+1 -> -1: aligned, cut 0
    res = oracle.anneal(2, *_csr(2, [(0, 1, -1)]), order=order, thr=zero, init_spins=[[1, -1]])
    assert res["final"].tolist() == [[-1, -1]] and res["trace"].tolist() == [[0]]
    # Jacobi on w=+1 from (+,+): both see h=+1 -> both -1 (the synchronous 2-cycle), cut stays 0
    res = oracle.anneal(2, *_csr(2, [(0, 1, 1)]), mode=1, thr=zero, init_spins=[[1, 1]])
    assert res["final"].tolist() == [[-1, -1]] and res["trace"].tolist() == [[0]]


def test_tie_rule(oracle):
    # path 0-1-2 with weights +1,-1 and s0=s2=+1: h_1 = 0.  Only vertex 1 is visited first.
    csr = _csr(3, [(0, 1, 1), (1, 2, -1)])
    order = np.array([1, 0, 2], dtype=np.int32)
    zero = np.zeros(1, dtype=np.uint32)
    h = oracle.local_fields(3, *csr, [1, 1, 1])
    assert h.tolist() == [1, 0, -1]
    minus = oracle.anneal(3, *csr, order=order, thr=zero, init_spins=[[1, 1, 1]], tie_rule=0)
    keep = oracle.anneal(3, *csr, order=order, thr=zero, init_spins=[[1, 1, 1]], tie_rule=1)
    assert minus["final"][0, 1] == -1          # "otherwise sigma_i = -1" (L49)
    assert keep["final"][0, 1] == 1            # S=0 "can take any value": unchanged


def test_local_fields_match_dense_matvec(oracle):
    n = 40
    csr = small_graph(n, 0.3, 21, "pm8", np.int32)
    J = np.zeros((n, n), dtype=np.int64)
    src = np.repeat(np.arange(n), np.diff(csr[0]))
    J[src, csr[1]] = csr[2]
    assert (J == J.T).all()
    s = W.random_spins(9, 1, n)[0]
    assert (oracle.local_fields(n, *csr, s) == J @ s.astype(np.int64)).all()


# ----------------------------------------------------------------------------
# zero-temperature invariants (L63: "minimise the local energy ... minimise the global energy")
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("wkind", ["pm4", "+1"])
def test_zero_temperature_gs_is_monotone_and_ends_in_local_optimum(oracle, wkind):
    n = 300
    csr = small_graph(n, 0.04, 31, wkind)
    colour, _ = W.greedy_colouring(n, csr[0], csr[1])
    res = oracle.anneal(n, *csr, order=oracle.order_from_colour(colour), n_replicas=8, seed=4,
                        thr=np.zeros(200, dtype=np.uint32))
    tr = res["trace"]
    assert (np.diff(tr, axis=0) >= 0).all()            # E never increases <=> cut never decreases
    u, v, w = edges_of(csr)
    Wtot = int(w.sum())
    for r in range(8):
        s = res["final"][r]
        h = oracle.local_fields(n, *csr, s)
        assert (s.astype(np.int64) * h <= 0).all()     # 1-flip local optimum
        assert 2 * int(tr[-1, r]) >= Wtot              # local-search bound cut >= W/2


def test_jacobi_two_cycle_on_bipartite_all_plus(oracle):
    wl = W.config3(L=6, sweeps=6, replicas=1, all_plus=True)
    wl.thr[:] = 0
    res = oracle.anneal(wl.n, wl.row_ptr, wl.col, wl.w, mode=1, thr=wl.thr,
                        init_spins=np.ones((1, wl.n), dtype=np.int8))
    assert (res["trace"] == 0).all()                   # all(+1) <-> all(-1), cut 0 forever
    assert (res["final"] == 1).all()                   # even number of sweeps -> back to all(+1)


# ----------------------------------------------------------------------------
# closed forms
# ----------------------------------------------------------------------------
def test_even_torus_all_plus_reaches_number_of_edges(oracle):
    wl = W.config3(L=10, sweeps=300, replicas=8, all_plus=True)
    n_edges = wl.nnz // 2
    assert n_edges == 2 * 10 * 10
    res = oracle.anneal_workload(wl)
    assert (res["best_cut"] == n_edges).all()          # bipartite: max cut = #E (Table III torus rows)
    # the checkerboard state is a fixed point of zero-temperature sweeps with cut #E
    chk = (wl.colour * 2 - 1).astype(np.int8)[None, :]
    res = oracle.anneal_workload(wl, n_replicas=1, thr=np.zeros(3, dtype=np.uint32), init_spins=chk)
    assert (res["trace"] == n_edges).all() and (res["final"] == chk).all()


@pytest.mark.parametrize("n", [7, 16, 33])
def test_complete_graph_all_plus_ends_balanced(oracle, n):
    u, v = W.complete_edges(n)
    csr = W.csr_from_edges(n, u, v, np.ones(u.size, dtype=np.int64), np.int8)
    order = np.arange(n, dtype=np.int32)               # n singleton colours
    res = oracle.anneal(n, *csr, order=order, n_replicas=4, seed=2, thr=np.zeros(3 * n, dtype=np.uint32))
    assert (res["trace"][-1] == (n // 2) * ((n + 1) // 2)).all()


def test_bipartite_positive_weights_max_cut_is_total_weight(oracle):
    # random bipartite graph, positive weights: the 2-colouring itself cuts everything
    n = 40
    u, v = W.erdos_renyi_edges(n, 0.3, 77)
    keep = (u % 2) != (v % 2)
    u, v = u[keep], v[keep]
    wt = np.abs(W.weights_from_hash(W.hash_pairs(77, u, v), "pm8"))
    csr = W.csr_from_edges(n, u, v, wt, np.int8)
    s = ((np.arange(n) % 2) * 2 - 1).astype(np.int8)
    _, cut = oracle.energy_cut(n, *csr, s[None, :])
    assert int(cut[0]) == int(wt.sum())


# ----------------------------------------------------------------------------
# flip step (Alg. 2; readings Q5, Q11) and schedules (Q6)
# ----------------------------------------------------------------------------
def test_flip_threshold_extremes(oracle):
    n = 200
    csr = small_graph(n, 0.05, 41, "pm4")
    colour, _ = W.greedy_colouring(n, csr[0], csr[1])
    order = oracle.order_from_colour(colour)
    init = W.random_spins(5, 1, n)
    never = oracle.anneal(n, *csr, order=order, thr=np.array([0], dtype=np.uint32), init_spins=init)
    always = oracle.anneal(n, *csr, mode=1, thr=np.array([0xFFFFFFFF], dtype=np.uint32), init_spins=init)
    jac = oracle.anneal(n, *csr, mode=1, thr=np.array([0], dtype=np.uint32), init_spins=init)
    # Jacobi: argmin from the start state is -sign(h) (tie -> -1); thr=2^32-1 flips all but w.p. 2^-32
    h = oracle.local_fields(n, *csr, init[0])
    argmin = np.where(h < 0, 1, -1)
    assert (jac["final"][0] == argmin).all()
    assert (always["final"][0] == -argmin).all()
    # GS with thr=0 is a pure descent step
    E0, _ = oracle.energy_cut(n, *csr, init)
    E1, _ = oracle.energy_cut(n, *csr, never["final"])
    assert E1[0] <= E0[0]


def test_flip_counter_words_and_domain(oracle):
    """Q11 / include/ising.h:18: the flip word of spin i, absolute sweep T, replica r is
    philox4x32_10(ctr=(i, T, r>>2, DOMAIN_FLIP=0), key=seed)[r&3].  Edgeless graph, Jacobi, tie rule MINUS: h = 0,
    the argmin is -1, so the spin after sweep T is +1 IFF that word < thr.  The expectation comes from the raw,
    KAT-pinned Philox function (not from the annealer), with sweep, replica group and spin all different and
    non-zero so that a permuted counter word or another domain constant fails."""
    n, R, first, off, M = 37, 9, 5, 3, 2
    seed = 0x1234_5678_9ABC_DEF1
    key = [seed & 0xFFFFFFFF, seed >> 32]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    col = np.zeros(0, dtype=np.int32)
    w = np.zeros(0, dtype=np.int8)
    thr = np.array([0x6000_0000, 0x9000_0000], dtype=np.uint32)
    for mode, order in ((1, None), (0, np.arange(n, dtype=np.int32))):
        for m in (1, 2):            # the state after sweep off and after sweep off + 1
            res = oracle.anneal(n, row_ptr, col, w, order=order, mode=mode, thr=thr[:m], n_replicas=R,
                                first_replica=first, seed=seed, sweep_offset=off)
            T = off + m - 1
            for r in range(R):
                rep = first + r
                for i in range(n):
                    word = int(oracle.philox4x32_10([i, T, rep >> 2, 0], key)[rep & 3])
                    assert (res["final"][r, i] == 1) == (word < int(thr[m - 1])), (mode, m, r, i)


@pytest.mark.parametrize("p", [0.5, 0.1, 0.003])
def test_flip_rate_statistics(oracle, p):
    # edgeless graph: h=0 -> argmin = -1 (MINUS); a spin ends +1 iff its Philox word < thr
    n = 400_000
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    col = np.zeros(0, dtype=np.int32)
    w = np.zeros(0, dtype=np.int8)
    thr = W.thresholds_from_probs(np.array([p]))
    res = oracle.anneal(n, row_ptr, col, w, mode=1, thr=thr, n_replicas=3, first_replica=5, seed=99)
    k = (res["final"] == 1).sum(axis=1)
    sigma = np.sqrt(n * p * (1 - p))
    assert (np.abs(k - n * p) < 5 * sigma).all()
    # the three replicas (ids 5,6,7: words 1,2,3 of one Philox call) are not copies of each other
    assert (res["final"][0] != res["final"][1]).any() and (res["final"][1] != res["final"][2]).any()


def test_init_spins_are_balanced_and_keyed_on_replica(oracle):
    n = 100_000
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    res = oracle.anneal(n, row_ptr, np.zeros(0, np.int32), np.zeros(0, np.int8), mode=1, tie_rule=1,
                        thr=np.zeros(1, np.uint32), n_replicas=4, seed=3)   # KEEP + h=0: state = init
    frac = (res["final"] == 1).mean(axis=1)
    assert (np.abs(frac - 0.5) < 5 * 0.5 / np.sqrt(n)).all()
    assert len({res["final"][r].tobytes() for r in range(4)}) == 4
    # the init bit is the low bit of the replica's word of philox(ctr=(i,0,r>>2,1), key=seed)
    for i in (0, 1, 77):
        out = oracle.philox4x32_10([i, 0, 0, 1], [3, 0])
        assert [1 if int(out[r]) & 1 else -1 for r in range(4)] == res["final"][:, i].tolist()


def test_schedule_endpoints_and_monotone():
    lin = W.linear_schedule(0.10, 0.0, 1000)
    assert int(lin[0]) == int(np.floor(0.10 * 2 ** 32)) and int(lin[-1]) == 0
    assert (np.diff(lin.astype(np.int64)) <= 0).all()
    ex = W.exponential_schedule(0.2, 1e-4, 500)
    assert int(ex[0]) == int(np.floor(0.2 * 2 ** 32))
    assert abs(int(ex[-1]) - int(np.floor(1e-4 * 2 ** 32))) <= 1
    assert (np.diff(ex.astype(np.int64)) <= 0).all()
    assert int(W.thresholds_from_probs(np.array([1.0]))[0]) == 0xFFFFFFFF


# ----------------------------------------------------------------------------
# order / replica / sweep semantics (readings Q8, Q10, Q11)
# ----------------------------------------------------------------------------
def _wl_small():
    wl = W.config2(n=300, p=0.03, sweeps=40, replicas=6)
    return wl


def test_order_inside_a_colour_class_does_not_matter(oracle):
    wl = _wl_small()
    base = oracle.anneal_workload(wl)
    order = oracle.order_from_colour(wl.colour)
    # reverse the order inside every class: a class is an independent set, so nothing changes
    rev = np.concatenate([order[wl.colour[order] == c][::-1] for c in range(wl.n_colours)]).astype(np.int32)
    assert (rev != order).any()
    other = oracle.anneal_workload(wl, order=rev)
    assert (base["trace"] == other["trace"]).all() and (base["final"] == other["final"]).all()
    # an order that breaks the classes generally does change the trajectory
    nat = oracle.anneal_workload(wl, order=np.arange(wl.n, dtype=np.int32))
    assert (nat["trace"] != base["trace"]).any()


def test_batch_split_invariance(oracle):
    wl = _wl_small()
    base = oracle.anneal_workload(wl)
    for r in range(wl.n_replicas):
        one = oracle.anneal_workload(wl, n_replicas=1, first_replica=r)
        assert (one["trace"][:, 0] == base["trace"][:, r]).all()
        assert (one["final"][0] == base["final"][r]).all()


def test_sweep_split_invariance(oracle):
    wl = _wl_small()
    base = oracle.anneal_workload(wl)
    k = 17
    a = oracle.anneal_workload(wl, thr=wl.thr[:k])
    b = oracle.anneal_workload(wl, thr=wl.thr[k:], sweep_offset=k, init_spins=a["final"])
    assert (np.concatenate([a["trace"], b["trace"]]) == base["trace"]).all()
    assert (b["final"] == base["final"]).all()


def test_best_tracking(oracle):
    wl = _wl_small()
    res = oracle.anneal_workload(wl)
    tr = res["trace"]
    assert (res["best_cut"] == tr.max(axis=0)).all()
    assert (res["best_sweep"] == tr.argmax(axis=0)).all()          # first argmax: earliest sweep wins
    csr = (wl.row_ptr, wl.col, wl.w)
    for r in range(wl.n_replicas):
        assert cut_by_definition(csr, res["best_spins"][r]) == int(res["best_cut"][r])
    off = oracle.anneal_workload(wl, sweep_offset=100)
    assert (off["best_sweep"] >= 100).all()


def test_multithreaded_wrapper_changes_nothing(oracle):
    wl = _wl_small()
    a = oracle.anneal_workload(wl)
    b = oracle.anneal_workload(wl, n_threads=4)
    assert all((a[k] == b[k]).all() for k in a)


# ----------------------------------------------------------------------------
# the generators produce what DESIGN.md's input recipe says
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("k,kw", [(1, {}), (2, {}), (3, dict(L=20, replicas=4, sweeps=5)),
                                  (4, dict(n=64, replicas=4, sweeps=5)),
                                  (5, dict(n=20000, replicas=4, sweeps=5))])
def test_generated_graphs_are_valid_inputs(k, kw):
    wl = W.build_config(k, **kw)
    n = wl.n
    src = np.repeat(np.arange(n), np.diff(wl.row_ptr))
    assert (src != wl.col).all()                                   # no self loops
    key = src.astype(np.int64) * n + wl.col
    assert (np.diff(key) > 0).all()                                # sorted, no duplicates
    rkey = wl.col.astype(np.int64) * n + src
    o = np.argsort(rkey, kind="stable")
    assert (rkey[o] == key).all() and (wl.w[o] == wl.w).all()      # symmetric with equal weights
    if wl.colour is not None:
        assert (wl.colour[src] != wl.colour[wl.col]).all()         # proper colouring
        assert wl.colour.min() == 0 and wl.colour.max() == wl.n_colours - 1
    if k == 4:
        assert wl.nnz == n * (n - 1) and set(np.unique(wl.w)) <= set(range(-8, 9)) - {0}
    if k == 5:
        assert set(np.unique(wl.w)) <= set(range(-4, 5)) - {0}


# ---------------------------------------------------------------------------------------------
# edge-list file loader: the layout of the paper's benchmark files (L190), synthetic content
# ---------------------------------------------------------------------------------------------
def test_edge_list_loader_builds_a_valid_workload(oracle, tmp_path):
    n = 60
    u, v = W.erdos_renyi_edges(n, 0.15, 91)
    wt = W.weights_from_hash(W.hash_pairs(91, u, v), "pm4")
    lines = ["%d %d" % (n, u.size + 3)]
    for a, b, c in zip(u, v, wt):
        lines.append("%d %d %d" % (b + 1, a + 1, c))          # 1-based, either orientation
    lines.append("%d %d %d" % (u[0] + 1, v[0] + 1, 2))        # duplicate pair: weights add up
    lines.append("7 7 5")                                      # self loop: dropped
    lines.append("%d %d %d" % (u[1] + 1, v[1] + 1, -int(wt[1])))   # cancels to zero: edge dropped
    path = tmp_path / "graph.txt"
    path.write_text("\n".join(lines) + "\n")
    wl = W.load_edge_list(str(path), replicas=3, sweeps=20, colouring="index")
    expect = wt.copy()
    expect[0] += 2
    keep = np.ones(u.size, dtype=bool)
    keep[1] = False
    ref = W.csr_from_edges(n, u[keep], v[keep], expect[keep], np.int8)
    np.testing.assert_array_equal(wl.row_ptr, ref[0])
    np.testing.assert_array_equal(wl.col, ref[1])
    np.testing.assert_array_equal(wl.w, ref[2])
    # proper colouring, usable by the oracle
    for i in range(n):
        nb = wl.col[wl.row_ptr[i]:wl.row_ptr[i + 1]]
        assert np.all(wl.colour[nb] != wl.colour[i])
    o = oracle.anneal_workload(wl, n_threads=1)
    assert o["trace"].shape == (20, 3) and np.all(o["best_cut"] == o["trace"].max(axis=0))


# ---------------------------------------------------------------------------------------------
# general Ising / QUBO front door (eq. (1)-(3) L39-53): external field by the gauge reduction
# ---------------------------------------------------------------------------------------------
def test_field_reduction_preserves_every_energy(oracle):
    from paper_1807_10750_b200 import frontdoor as F
    n = 9
    u, v = W.erdos_renyi_edges(n, 0.5, 7)
    w = W.weights_from_hash(W.hash_pairs(7, u, v), "pm4")
    f = (W.rand_u64(7, 3, n) % np.uint64(9)).astype(np.int64) - 4
    n2, u2, v2, w2 = F.ising_with_field(n, u, v, w, f)
    csr2 = W.csr_from_edges(n2, u2, v2, w2, np.int8)
    S2 = all_states(n2)
    E2, _ = oracle.energy_cut(n2, *csr2, S2)                 # pair energy of the augmented graph, every state
    dec = F.decode_field_solution(S2)
    Ef = np.array([F.field_energy(n, u, v, w, f, s) for s in dec])
    np.testing.assert_array_equal(E2, Ef)                    # E'(s, s_n) = E_field(s * s_n), state by state
    # and the minimum over the augmented graph is the minimum of the field problem
    Eall = np.array([F.field_energy(n, u, v, w, f, s) for s in all_states(n)])
    assert E2.min() == Eall.min()


def test_qubo_to_ising_matches_enumeration():
    from paper_1807_10750_b200 import frontdoor as F
    n = 8
    Q = (W.rand_u64(11, 5, n * n) % np.uint64(13)).astype(np.int64).reshape(n, n) - 6
    u, v, w, f, const = F.qubo_to_ising(Q)
    for code in range(1 << n):
        x = np.array([(code >> k) & 1 for k in range(n)], dtype=np.int64)
        s = 2 * x - 1
        assert 4 * int(x @ Q @ x) == const + F.field_energy(n, u, v, w, f, s)


def test_annealer_solves_a_small_field_problem(oracle):
    from paper_1807_10750_b200 import frontdoor as F
    n = 12
    u, v = W.erdos_renyi_edges(n, 0.4, 13)
    w = W.weights_from_hash(W.hash_pairs(13, u, v), "pm4")
    f = (W.rand_u64(13, 3, n) % np.uint64(7)).astype(np.int64) - 3
    wl = F.field_workload(n, u, v, w, f, replicas=8, sweeps=200, p0=0.2)
    o = oracle.anneal_workload(wl, n_threads=1)
    r = int(np.argmax(o["best_cut"]))
    s = F.decode_field_solution(o["best_spins"][r])
    Emin = min(F.field_energy(n, u, v, w, f, t) for t in all_states(n))
    assert F.field_energy(n, u, v, w, f, s) == Emin
    assert int(o["best_cut"][r]) == (wl.w_total - Emin) // 2


# ---------------------------------------------------------------------------------------------
# Algorithm 1's exact-N flip step: oracle mode 2
# ---------------------------------------------------------------------------------------------
def _one_sweep(oracle, n, csr, order, N, init, seed=3, sweep_offset=0):
    o = oracle.anneal(n, *csr, order=order, mode=2, n_replicas=init.shape[0], seed=seed,
                      thr=np.array([N], dtype=np.uint32), sweep_offset=sweep_offset, init_spins=init)
    return o["final"]


def test_exact_n_flips_exactly_n_distinct_spins(oracle):
    n = 90
    csr = small_graph(n, 0.1, 17)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "index")
    order = oracle.order_from_colour(colour)
    init = W.random_spins(5, 6, n)
    base = _one_sweep(oracle, n, csr, order, 0, init)                 # N = 0: the pure minimisation sweep
    for N in (1, 7, 45, 89, 90, 500):
        s = _one_sweep(oracle, n, csr, order, N, init)
        assert np.all((s != base).sum(axis=1) == min(N, n))           # exactly N distinct spins flipped (N >= n: all)
    # N = 0 is a descent sweep: identical to Algorithm 2 with a zero threshold
    o0 = oracle.anneal(n, *csr, order=order, mode=0, n_replicas=6, seed=3, thr=np.zeros(1, dtype=np.uint32), init_spins=init)
    np.testing.assert_array_equal(base, o0["final"])


def test_exact_n_subset_is_uniform_over_the_spins(oracle):
    """Empty graph: the minimisation sweep writes -1 everywhere (tie rule MINUS), so the +1 spins after the sweep
    are exactly the chosen subset; over many (replica, sweep) draws every spin is chosen N/n of the time."""
    n, N, R, M = 40, 6, 64, 60
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    col = np.zeros(0, dtype=np.int32)
    w = np.zeros(0, dtype=np.int8)
    order = np.arange(n, dtype=np.int32)
    counts = np.zeros(n, dtype=np.int64)
    pair_seen = set()
    for t in range(M):
        o = oracle.anneal(n, row_ptr, col, w, order=order, mode=2, n_replicas=R, seed=11,
                          thr=np.array([N], dtype=np.uint32), sweep_offset=t, n_threads=4)
        chosen = o["final"] == 1
        assert np.all(chosen.sum(axis=1) == N)
        counts += chosen.sum(axis=0)
        pair_seen.update(tuple(np.nonzero(c)[0]) for c in chosen)
    draws = R * M
    expect = draws * N / n
    sigma = np.sqrt(draws * (N / n) * (1 - N / n))
    assert np.all(np.abs(counts - expect) < 5 * sigma)
    assert len(pair_seen) > 0.99 * draws          # different replicas / sweeps draw different subsets


def test_exact_n_draw_counter_words_and_domain(oracle):
    """Reading Q5 (Algorithm 1, L92): draw k of sweep T, replica r uses philox4x32_10(ctr=(k, T, r>>2,
    DOMAIN_FLIPN=2), key=seed)[r&3] and x = floor(u (j+1) / 2^32), j = n - N + k (Floyd).  Empty graph, MINUS: the
    minimisation sweep writes -1 everywhere, so the +1 spins are exactly the subset -- recomputed here from the raw,
    KAT-pinned Philox function with non-zero sweep / replica group."""
    n, N, R, first, off = 23, 5, 6, 6, 4
    seed = 0xFEDC_BA98_7654_3211
    key = [seed & 0xFFFFFFFF, seed >> 32]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    o = oracle.anneal(n, row_ptr, np.zeros(0, np.int32), np.zeros(0, np.int8), order=np.arange(n, dtype=np.int32),
                      mode=2, n_replicas=R, first_replica=first, seed=seed, thr=np.array([N], dtype=np.uint32),
                      sweep_offset=off)
    for r in range(R):
        rep = first + r
        chosen = []
        for k in range(N):
            j = n - N + k
            u = int(oracle.philox4x32_10([k, off, rep >> 2, 2], key)[rep & 3])
            x = (u * (j + 1)) >> 32
            chosen.append(j if x in chosen else x)
        expect = -np.ones(n, dtype=np.int8)
        expect[chosen] = 1
        np.testing.assert_array_equal(o["final"][r], expect)


def test_exact_n_best_tracking_and_trace(oracle):
    n = 60
    csr = small_graph(n, 0.15, 23)
    colour, nc = W.greedy_colouring(n, csr[0], csr[1], "index")
    order = oracle.order_from_colour(colour)
    thr = np.array([8, 6, 4, 2, 1, 0, 0], dtype=np.uint32)
    o = oracle.anneal(n, *csr, order=order, mode=2, n_replicas=5, seed=2, thr=thr)
    E, cut = oracle.energy_cut(n, *csr, o["final"])
    np.testing.assert_array_equal(cut, o["trace"][-1])
    np.testing.assert_array_equal(o["best_cut"], o["trace"].max(axis=0))
    assert np.all(o["trace"][-1] >= o["trace"][-2])       # the last two sweeps are pure descent
