"""Run the BASELINE.json configurations through the CUDA path and print one JSON line per (config, precision):
create / matvec / solve times, list statistics, stage times, energies.  The numbers of BASELINE.md section 5.

    python -m paper_1309_4018_b200.configs 0 1 2 3          # Born, Kirkwood, protein, multi-surface
    python -m paper_1309_4018_b200.configs 4 [spacing]      # binding energy: complex, receptor, ligand (P = 8)

Timing only (CUDA events over 10 warm matvecs); parity against the oracle is the job of tests/.
"""
import json
import sys
import time

import numpy as np


def run(name, prob, kw, tol, pg, torch):
    x = torch.tensor(np.random.default_rng(11).normal(size=2 * prob.n_panels), device="cuda")
    for pname, prec in (("fp64", pg.PRECISION_FP64), ("mixed", pg.PRECISION_MIXED)):
        t = time.perf_counter()
        h = pg.Handle.from_problem(prob, precision=prec, **kw)
        torch.cuda.synchronize()
        create_ms = 1e3 * (time.perf_counter() - t)
        y = h.matvec(x)
        for _ in range(3):
            h.matvec(x, y)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(10):
            h.matvec(x, y)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 10
        st = h.stats()
        h.profile(True)
        for _ in range(3):
            h.matvec(x, y)
        stages = {k: round(v[0] / 3, 4) for k, v in h.stage_times().items()}
        h.profile(False)
        t = time.perf_counter()
        xs, it, rr, rc = h.solve(tol=tol if pname == "fp64" else max(tol, 1e-5), max_iter=3000, raise_on_noconv=False)
        es, ec = h.energy(xs)
        torch.cuda.synchronize()
        solve_ms = 1e3 * (time.perf_counter() - t)
        print(json.dumps(dict(config=name, precision=pname, n_panels=prob.n_panels, n_surfaces=len(prob.surfaces),
                              n_charges=len(prob.charge_q), create_ms=create_ms, matvec_ms=ms,
                              direct_equiv=st["direct_equiv"], interactions_per_s=st["direct_equiv"] / (ms * 1e-3),
                              p2p_pairs=st["p2p_pairs"], m2p_evals=st["m2p_evals"], n_cells=st["n_cells"],
                              near_nnz=st["near_nnz"], device_MB=st["device_bytes"] / 1e6, stages_ms=stages,
                              kernels_per_matvec=st["kernels_per_matvec"], gmres_iters=it, rel_resid=rr, rc=rc,
                              solve_ms=solve_ms, E_solv_kJ_mol=es, E_coul_kJ_mol=ec)), flush=True)
        h.close()


def main():
    import torch
    import workloads as W
    import paper_1309_4018_b200 as pg
    which = [a for a in sys.argv[1:] if a in ("0", "1", "2", "3", "4")] or ["0", "1", "2", "3"]
    spacing = next((float(a) for a in sys.argv[1:] if "." in a), 0.55)
    if "0" in which:
        run("0 born_l3 direct", W.born_problem(3), dict(K=4, P=6, theta=0.0), 1e-8, pg, torch)
    if "1" in which:
        run("1 kirkwood_l5", W.kirkwood_problem(5), dict(K=4, P=6, theta=0.5), 1e-6, pg, torch)
    if "2" in which:
        run("2 protein_1000", W.protein_problem(1000, spacing=1.05), dict(K=4, P=6, theta=0.5), 1e-6, pg, torch)
    if "3" in which:
        run("3 multisurface_3000", W.multisurface_problem(3000, spacing=1.12), dict(K=4, P=6, theta=0.5), 1e-6, pg, torch)
    if "4" in which:
        for q in W.binding_problems(5000, 500, spacing=spacing):
            run("4 " + q.name, q, dict(K=4, P=8, theta=0.5), 1e-4, pg, torch)


if __name__ == "__main__":
    main()
