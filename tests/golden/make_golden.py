"""Writes tests/golden/oracle_energies.json.  Calls ONLY oracle/ and workloads/ (never the CUDA path).

    python tests/golden/make_golden.py

Values: solvation energies [kJ/mol] of the D0 discretisation (oracle, dense O(N^2) matvec + numpy GMRES)
for the full-size configurations whose oracle solve takes minutes, so that the GPU tests can compare
against them without re-running the oracle.  Each entry records the parameters it was computed with.
"""
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))

import workloads as W          # noqa: E402
from oracle import Oracle      # noqa: E402


def main():
    out = {}
    cases = [
        ("kirkwood_l5", W.kirkwood_problem(5), dict(K=4, K_fine=19, thres=2.0, N_k=5), 1e-6),
        ("kirkwood_l4", W.kirkwood_problem(4), dict(K=4, K_fine=19, thres=2.0, N_k=5), 1e-8),
        ("born_l3", W.born_problem(3), dict(K=4, K_fine=19, thres=2.0, N_k=5), 1e-8),
    ]
    for name, prob, kw, tol in cases:
        t = time.time()
        o = Oracle(prob, **kw)
        x, it, rel = o.solve(tol=tol)
        out[name] = dict(E_solv_kJ_mol=o.solvation_energy(x), E_coul_kJ_mol=o.coulomb_energy(), iters=it,
                         rel_resid=rel, tol=tol, n_panels=o.npan, seconds=round(time.time() - t, 1), **kw)
        print(name, out[name], flush=True)
        with open(os.path.join(HERE, "oracle_energies.json"), "w") as f:
            json.dump(out, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
