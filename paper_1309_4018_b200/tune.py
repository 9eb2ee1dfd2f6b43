"""Leaf-size sweep of the treecode matvec on a Kirkwood sphere (the tuning behind the NCRIT defaults).

    python -m paper_1309_4018_b200.tune [--level 5] [--P 6] [--theta 0.5]

Prints, per precision and NCRIT (panels per leaf), the matvec time (CUDA events, 20 matvecs, warm L2), the
direct-pair and M2P-evaluation counts and the per-stage times of `pygbe_profile`.  Timing only: accuracy is
checked by tests/ against the oracle.
"""
import argparse

import numpy as np


def main():
    import torch
    import workloads as W
    import paper_1309_4018_b200 as pg
    ap = argparse.ArgumentParser()
    ap.add_argument("--level", type=int, default=5)
    ap.add_argument("--P", type=int, default=6)
    ap.add_argument("--theta", type=float, default=0.5)
    ap.add_argument("--ncrit", type=int, nargs="*", default=[24, 32, 48, 64, 96, 128, 192, 256])
    a = ap.parse_args()
    prob = W.kirkwood_problem(a.level)
    x = torch.tensor(np.random.default_rng(1).normal(size=2 * prob.n_panels), device="cuda")
    for prec in (pg.PRECISION_MIXED, pg.PRECISION_FP64):
        for ncrit in a.ncrit:
            h = pg.Handle.from_problem(prob, K=4, P=a.P, theta=a.theta, precision=prec, ncrit=ncrit)
            y = h.matvec(x)
            for _ in range(3):
                h.matvec(x, y)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(20):
                h.matvec(x, y)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 20
            st = h.stats()
            h.profile(True)
            for _ in range(5):
                h.matvec(x, y)
            sg = h.stage_times()
            h.profile(False)
            print(f"prec {prec} ncrit {ncrit:4d}: {ms:.3f} ms p2p {st['p2p_pairs']:.3e} m2p {st['m2p_evals']:.3e} "
                  f"leaves {st['n_leaves']} | " + " ".join(f"{k}={v[0] / 5:.3f}" for k, v in sg.items()), flush=True)
            h.close()


if __name__ == "__main__":
    main()
