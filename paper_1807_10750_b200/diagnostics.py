"""Where a sweep spends its time: SM-clock stamps of one sweep of an ising_anneal call (include/ising_debug.h).

    python -m paper_1807_10750_b200.diagnostics --workload cfg5 [--sweep 300] [--flags 0]

Changes no result.  Per engine (ising_problem_info(13)):
  persistent grid kernel      per virtual phase (colour classes, bulk pseudo-phase, chain): median / min / max over the CTAs
                              of the work (arrival at the barrier - departure from the previous one) and of the barrier
                              wait, and the phase's span; with a tail chain also the stamps inside the chain of CTA 0
  k_anneal_small              CTA 0: flips drawn, every colour-class segment, dE reduce, cut / best, capture
  k_dense_anneal              CTA 0: TMA issue done, MMA issue done, accumulators seen, epilogue done, barrier, bookkeeping
Stamps of different CTAs come from different SM clocks: only differences within a CTA are used.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np

from . import binding as B
from . import workloads as W


def stamps_of(wl, sweep: int, flags: int = 0):
    import torch
    p = B.load_workload(wl, flags=flags)
    buf = p.phase_timing(sweep)
    B.anneal_workload(p, wl, thr=wl.thr[:sweep + 3])
    torch.cuda.synchronize()
    return p, buf.cpu().numpy().astype(np.int64)


def report(wl, sweep: int, flags: int = 0, out=sys.stdout):
    p, b = stamps_of(wl, sweep, flags)
    eng = p.engine
    print("%s: engine %d, chain rows %d, virtual phases %d, chunks %d, sweep %d" % (
        wl.name, eng, p.info(14), p.info(15), p.info(16), sweep), file=out)
    if p.has_dense_engine and wl.mode == "jacobi":
        s = b.reshape(-1)[:8]
        names = ["start", "tma issued", "mma issued", "accumulators seen", "epilogue done", "cta at barrier", "barrier done",
                 "bookkeeping done"]
        print("  k_dense_anneal pass %d, CTA 0, cycles since pass start: %s" % (
            sweep, ", ".join("%s %d" % (n, v - s[0]) for n, v in zip(names, s))), file=out)
    elif eng == B.ENGINE_SMALL:
        s = b.reshape(-1)
        s = s[s != 0]
        d = np.diff(s)
        print("  k_anneal_small CTA 0, cycles: total %d; flips %d; segments %s; dE reduce %d; cut / best %d; capture %d" % (
            s[-1] - s[0], d[0], [int(x) for x in d[1:-3]], d[-3], d[-2], d[-1]), file=out)
    else:
        rows = p.info(15) + (1 if eng == B.ENGINE_GRID_TAIL_CHAIN else 0)
        total = 0
        if p.info(19) > 0:
            print("  chain overlap: virtual phase 0 = %d rows of colour class 0 without a chain neighbour, updated beside the "
                  "chain of the sweep before (row 0 below = that chain step's barrier)" % p.info(19), file=out)
        for ph in range(rows):
            arrive, leave = b[ph, :, 0], b[ph, :, 1]
            wait = leave - arrive
            if ph == 0:
                print("  phase 0: barrier wait med / min / max %d / %d / %d" % (np.median(wait), wait.min(), wait.max()), file=out)
                continue
            work = arrive - b[ph - 1, :, 1]
            span = int(np.median(leave - b[ph - 1, :, 1]))
            total += span
            print("  phase %2d: work med / min / max %6d / %6d / %6d   wait %5d / %5d / %5d   span %6d" % (
                ph, np.median(work), work.min(), work.max(), np.median(wait), wait.min(), wait.max(), span), file=out)
        print("  sum of spans (phases 1..): %d cycles" % total, file=out)
        if eng == B.ENGINE_GRID_TAIL_CHAIN:
            st = b[:, 0, 2:8].reshape(-1)
            st = st[st != 0]
            if st.size > 1:
                print("  chain of CTA 0 (start, then per chunk landed / per segment done): %s" % np.diff(st).tolist(), file=out)
    p.free()


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--sweep", type=int, default=8)
    ap.add_argument("--flags", type=int, default=0, help="ISING_LOAD_* engine-selection flags")
    a = ap.parse_args(argv)
    report(W.build_config(int(a.workload[3])), a.sweep, a.flags)
    return 0


if __name__ == "__main__":
    sys.exit(main())
