"""the Table-I-style accuracy report on user-supplied edge-list files.
Synthetic files only (the paper's benchmark files are not in this repository)."""
import numpy as np
import pytest

from paper_1807_10750_b200 import report as R
from paper_1807_10750_b200 import workloads as W


def write_graph(path, n, p, seed, wkind):
    u, v = W.erdos_renyi_edges(n, p, seed)
    wt = W.weights_from_hash(W.hash_pairs(seed, u, v), wkind)
    path.write_text("%d %d\n" % (n, u.size) + "".join("%d %d %d\n" % (a + 1, b + 1, c) for a, b, c in zip(u, v, wt)))
    return u.size


def oracle_runner(oracle):
    def run(wl, seed):
        o = oracle.anneal_workload(wl, seed=seed, n_threads=4)
        return int(o["best_cut"].max())
    return run


def test_report_rows_and_table_with_the_oracle_as_runner(tmp_path, oracle):
    e1 = write_graph(tmp_path / "a.txt", 60, 0.2, 5, "pm1")
    e2 = write_graph(tmp_path / "b.txt", 40, 0.3, 6, "pm4")
    (tmp_path / "bk").write_text("# best known\na.txt 200\nb 1000\n")
    bk = R.read_best_known(str(tmp_path / "bk"))
    assert bk == {"a.txt": 200, "b": 1000}
    rows = R.report_rows([str(tmp_path / "a.txt"), str(tmp_path / "b.txt")], bk, runs=3, sweeps=40, replicas=4, p0=0.1,
                         runner=oracle_runner(oracle))
    assert [r["graph"] for r in rows] == ["a.txt", "b.txt"] and [r["edges"] for r in rows] == [e1, e2]
    for r in rows:
        assert r["min"] <= r["mean"] <= r["max"] and r["runs"] == 3
    assert rows[0]["pct_of_best_known"] == pytest.approx(100.0 * rows[0]["mean"] / 200)
    assert rows[1]["best_known"] == 1000          # matched by the name without extension
    table = R.format_table(rows)
    assert "a.txt" in table and "% of bk" in table and len(table.splitlines()) == 4


@pytest.mark.gpu
def test_report_through_the_library_matches_the_oracle(tmp_path, oracle, capsys):
    write_graph(tmp_path / "g1.txt", 300, 0.03, 11, "pm1")
    write_graph(tmp_path / "g2.txt", 500, 0.02, 12, "pm4")
    files = [str(tmp_path / "g1.txt"), str(tmp_path / "g2.txt")]
    rows_gpu = R.report_rows(files, {}, runs=3, sweeps=60, replicas=8, p0=0.1)
    rows_cpu = R.report_rows(files, {}, runs=3, sweeps=60, replicas=8, p0=0.1, runner=oracle_runner(oracle))
    assert rows_gpu == rows_cpu
    assert R.main([str(tmp_path), "--runs", "2", "--sweeps", "30", "--replicas", "4"]) == 0
    assert "g2.txt" in capsys.readouterr().out
