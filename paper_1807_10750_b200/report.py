"""Accuracy report in the style of the paper's Table I for user-supplied edge-list files.

    python -m paper_1807_10750_b200.report DIR [--best-known FILE] [--runs 10] [--sweeps 1000] [--replicas 32]

Table I of the paper lists, per benchmark graph, the cut the annealer reaches as a percentage of the best-known cut,
"mean of 10 runs", 1000 sweeps each (L196).  This tool does the same through the library's public calls
(ising_load_csr / ising_anneal / ising_best_state) for every edge-list file in DIR (first line `n m`, then `i j w`,
1-based ids: the layout of the paper's benchmark set, L190).  The benchmark files themselves are
not part of this repository and are never fetched: the tool reports on whatever the user supplies.

A RUN = one Philox seed: `replicas` independent replicas annealed side by side, the run's result is the best cut over
its replicas (L239 "the best result could be picked from a number of GPU simulations").  Per file the table gives
n, #E, the mean / min / max of the runs' results, and -- when --best-known names a file of lines `<file name> <cut>` --
the mean as a percentage of the best-known cut.
"""
from __future__ import annotations

import argparse
import os
import sys
from typing import Callable, Dict, List, Optional

import numpy as np

from . import workloads as W


def read_best_known(path: Optional[str]) -> Dict[str, int]:
    out: Dict[str, int] = {}
    if not path:
        return out
    with open(path) as f:
        for line in f:
            parts = line.split()
            if len(parts) >= 2 and not line.lstrip().startswith("#"):
                out[parts[0]] = int(parts[1])
    return out


def gpu_runner(wl, seed: int) -> int:
    """Best cut over the replicas of one run (one seed) through the C ABI."""
    from . import binding as B
    p = B.load_workload(wl)
    try:
        B.anneal_workload(p, wl, seed=seed)
        _, cut, _, _ = B.ising_best_state(p, -1, want_spins=False)
        return int(cut)
    finally:
        p.free()


def report_rows(files: List[str], best_known: Dict[str, int], runs: int, sweeps: int, replicas: int, p0: float,
                runner: Callable = gpu_runner) -> List[dict]:
    rows = []
    for path in files:
        wl = W.load_edge_list(path, replicas=replicas, sweeps=sweeps, p0=p0, p_end=0.0)
        cuts = np.array([runner(wl, seed) for seed in range(runs)], dtype=np.int64)
        name = os.path.basename(path)
        bk = best_known.get(name, best_known.get(os.path.splitext(name)[0]))
        rows.append({"graph": name, "n": wl.n, "edges": wl.nnz // 2, "runs": runs, "mean": float(cuts.mean()),
                     "min": int(cuts.min()), "max": int(cuts.max()), "best_known": bk,
                     "pct_of_best_known": None if not bk else 100.0 * float(cuts.mean()) / bk})
    return rows


def format_table(rows: List[dict]) -> str:
    head = "%-24s %9s %10s %5s %12s %10s %10s %11s %8s" % ("graph", "#vertices", "#edges", "runs", "mean cut", "min", "max",
                                                          "best known", "% of bk")
    lines = [head, "-" * len(head)]
    for r in rows:
        lines.append("%-24s %9d %10d %5d %12.1f %10d %10d %11s %8s" % (
            r["graph"][:24], r["n"], r["edges"], r["runs"], r["mean"], r["min"], r["max"],
            "-" if r["best_known"] is None else str(r["best_known"]),
            "-" if r["pct_of_best_known"] is None else "%.2f" % r["pct_of_best_known"]))
    return "\n".join(lines)


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("dir", help="folder of edge-list files (first line 'n m', then 'i j w', 1-based ids)")
    ap.add_argument("--best-known", default=None, help="file of lines '<file name> <best-known cut>'")
    ap.add_argument("--runs", type=int, default=10, help="seeds per graph (Table I: mean of 10 runs)")
    ap.add_argument("--sweeps", type=int, default=1000, help="annealing sweeps per run (L196: 1000)")
    ap.add_argument("--replicas", type=int, default=32, help="replicas per run; the run's result is their best cut")
    ap.add_argument("--p0", type=float, default=0.10, help="flip probability of the first sweep (linear schedule to 0)")
    args = ap.parse_args(argv)
    files = sorted(os.path.join(args.dir, f) for f in os.listdir(args.dir)
                   if os.path.isfile(os.path.join(args.dir, f)) and not f.startswith(".")
                   and os.path.join(args.dir, f) != (args.best_known or ""))
    if not files:
        print("no files in %s" % args.dir, file=sys.stderr)
        return 1
    rows = report_rows(files, read_best_known(args.best_known), args.runs, args.sweeps, args.replicas, args.p0)
    print(format_table(rows))
    return 0


if __name__ == "__main__":
    sys.exit(main())
