"""Writes tests/golden/oracle_tiny_trace.txt: the first moves of the Tiny config as computed by the CPU oracle
(calls only oracle/ and the input generator).  Regression pin of the oracle's arithmetic: a later change to
it must either reproduce these numbers or name, in its commit message, the passage that justifies the change.

    python tests/golden/make_oracle_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1609_07936_b200 import workloads as wl  # noqa: E402

SEED = 0x5A11


def compute():
    w = wl.make("tiny", simpson_intervals=100_000)
    o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, SEED)
    o.init_walkers(2)
    chi2_0 = o.chi2.copy()
    tr, _ = o.anneal(w.schedule[:2], trace_walkers=(0, 2))
    return w, chi2_0, tr, o


def main():
    w, chi2_0, tr, o = compute()
    with open(os.path.join(HERE, "oracle_tiny_trace.txt"), "w") as f:
        f.write("# oracle trace, Tiny config (BASELINE.json configs[0]), seed 0x5A11, walkers 0-1, sweeps 0-1, first 24 moves each\n")
        f.write("# written by tests/golden/make_oracle_golden.py (calls only oracle/); columns:\n")
        f.write("# walker sweep move p s flags rho delta_p delta_s dchi2 ln_u\n")
        f.write(f"# chi2_0 {float(chi2_0[0])!r} {float(chi2_0[1])!r}\n")
        for wk in range(2):
            for sw in range(2):
                for m in range(24):
                    t = tr[wk, sw, m]
                    f.write(f"{wk} {sw} {m} {t['p']} {t['s']} {t['flags']} {float(t['rho'])!r} {float(t['delta_p'])!r} "
                            f"{float(t['delta_s'])!r} {float(t['dchi2'])!r} {float(t['ln_u'])!r}\n")
        f.write(f"# final chi2 {float(o.chi2[0])!r} {float(o.chi2[1])!r}\n")


if __name__ == "__main__":
    main()
