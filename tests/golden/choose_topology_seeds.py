"""Chooses the topology seeds recorded in ami_inputs/configs.py::TOPOLOGY_SEEDS.

Calls only ``ami_inputs`` (integer diagram generator) and ``oracle/`` (construct); no CUDA
code.  Rule: the first seed whose table is constructible in the
default summation order (|alpha_p| = 1 throughout) and, for config 3, whose construction met a
double pole, so that the derivative path is measured.  Run from the repo root:

    python tests/golden/choose_topology_seeds.py
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))

import ami_inputs as A  # noqa: E402
import oracle  # noqa: E402


def scan(m, need_multipole, max_seed=200):
    for seed in range(max_seed):
        d = A.random_self_energy(m, seed)
        try:
            info = oracle.OracleTable.from_diagram(d).info()
        except oracle.OracleError as ex:
            print(f"  m={m} seed={seed}: rejected ({ex})")
            continue
        ok = (info["multipoles"] > 0 and info["deriv_terms"] > 0) or not need_multipole
        print(f"  m={m} seed={seed}: n_eps={d.n_eps} {info}{'  <- chosen' if ok else ''}")
        if ok:
            return seed
    raise SystemExit("no seed found")


if __name__ == "__main__":
    out = {"cfg3": scan(4, True), "cfg4": scan(6, False), "cfg5": scan(5, False), "stress8": scan(8, False)}
    print("TOPOLOGY_SEEDS =", out)
