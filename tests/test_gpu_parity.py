"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances (BASELINE.json north_star; derivation in DESIGN.md "Tolerances"):
   direct mode (theta = 0), fp64           : rel-L2 <= 1e-11
   treecode P = 6, theta = 0.5             : rel-L2 <= 1e-4
   solvation energies                      : <= 0.1 % relative
"""
import json
import os

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-11
TOL_TREE = 1e-4
TOL_ENERGY = 1e-3
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_energies.json")


@pytest.fixture(scope="module")
def env(oracle_mod):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1309_4018_b200 as pg
    pg.lib()            # must load: there is no fallback
    return pg, torch, oracle_mod


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def gpu_matvec(pg, torch, prob, x, **kw):
    h = pg.Handle.from_problem(prob, **kw)
    y = h.matvec(torch.tensor(x, device="cuda")).cpu().numpy()
    return h, y


# ------------------------------------------------------------------------------------------- direct
@pytest.mark.parametrize("maker,level", [(W.born_problem, 0), (W.born_problem, 1), (W.born_problem, 2),
                                         (W.born_problem, 3), (W.stern_sphere_problem, 2),
                                         (W.cavity_sphere_problem, 2), (W.kirkwood_problem, 3)])
def test_direct_matvec_matches_oracle(env, maker, level):
    """theta = 0: same discretisation D0 as the oracle, different summation order only.  Levels 0-2 are
    ragged (20, 80, 320 panels: not a multiple of the 128-target group); level 3 spans 10 groups."""
    pg, torch, orc = env
    prob = maker(level)
    rng = np.random.default_rng(100 + level)
    o = orc.Oracle(prob)
    x = rng.normal(size=o.n)
    h, y = gpu_matvec(pg, torch, prob, x, K=4, theta=0.0)
    assert rel(y, o.matvec(x)) <= TOL_DIRECT
    assert rel(h.rhs().cpu().numpy(), o.rhs()) <= 1e-13
    st = h.stats()
    assert st["m2p_evals"] == 0 and st["p2p_pairs"] == st["direct_equiv"]
    h.close()


@pytest.mark.parametrize("K", [1, 3, 7])
def test_direct_other_gauss_rules(env, K):
    pg, torch, orc = env
    prob = W.born_problem(2)
    o = orc.Oracle(prob, K=K)
    x = np.random.default_rng(K).normal(size=o.n)
    h, y = gpu_matvec(pg, torch, prob, x, K=K, theta=0.0)
    assert rel(y, o.matvec(x)) <= TOL_DIRECT
    h.close()


@pytest.mark.parametrize("kw", [dict(K_fine=7, thres=1.25, N_k=5), dict(K_fine=19, thres=1.25, N_k=9),
                                dict(K_fine=19, thres=-1.0, N_k=5), dict(K_fine=19, thres=3.0, N_k=2)])
def test_direct_near_field_options(env, kw):
    """K_fine / thres / N_k (Tables 4, 6); thres < 0 switches the near-singular rule off."""
    pg, torch, orc = env
    prob = W.cavity_sphere_problem(1)
    okw = dict(kw)
    if okw["thres"] < 0:
        okw["thres"] = 0.0
    o = orc.Oracle(prob, K=4, **okw)
    x = np.random.default_rng(3).normal(size=o.n)
    h, y = gpu_matvec(pg, torch, prob, x, K=4, theta=0.0, **kw)
    assert rel(y, o.matvec(x)) <= TOL_DIRECT
    h.close()


def test_born_solve_and_energy(env):
    """BASELINE.json config 0 end to end: GMRES 1e-8, energy vs the oracle and vs the closed form."""
    pg, torch, orc = env
    from closed_forms import born
    prob = W.born_problem(3)
    o = orc.Oracle(prob)
    h = pg.Handle.from_problem(prob, K=4, theta=0.0)
    x, it, rr, rc = h.solve(tol=1e-8)
    assert rc == 0 and rr <= 1e-8
    xo, ito, _ = o.solve(tol=1e-8)
    assert abs(it - ito) <= 2
    es, ec = h.energy(x)
    eo = o.solvation_energy(xo)
    assert abs(es - eo) / abs(eo) < 1e-7
    assert ec == 0.0
    assert abs(es - born(1, 4, 4, 80, 0.125)) / 41.97 < 4e-3          # discretisation error, 0.33 %
    # true residual through the oracle's operator
    xn = x.cpu().numpy()
    assert np.linalg.norm(o.matvec(xn) - o.rhs()) / np.linalg.norm(o.rhs()) < 3e-8
    # host-buffer entry point gives the same answer
    xh, it2, rr2, es2, ec2 = h.solve_host(tol=1e-8)
    assert it2 == it and abs(es2 - es) < 1e-9 * abs(es) and rel(xh, xn) < 1e-9
    h.close()


def test_restarted_gmres_and_noconv(env):
    pg, torch, orc = env
    prob = W.cavity_sphere_problem(1)
    o = orc.Oracle(prob)
    xo, _, _ = o.solve(tol=1e-9)
    h = pg.Handle.from_problem(prob, K=4, theta=0.0)
    x, it, rr, rc = h.solve(tol=1e-9, restart=7, max_iter=2000)
    assert rc == 0 and rr <= 1e-9
    assert abs(h.energy(x)[0] - o.solvation_energy(xo)) / abs(o.solvation_energy(xo)) < 1e-6
    x2, it2, rr2, rc2 = h.solve(tol=1e-12, restart=5, max_iter=7, raise_on_noconv=False)
    assert rc2 == pg.PYGBE_ENOCONV and it2 == 7 and rr2 > 1e-12
    with pytest.raises(pg.PygbeError):
        h.solve(tol=1e-12, restart=5, max_iter=7)
    h.close()


# ----------------------------------------------------------------------------------------- treecode
@pytest.mark.parametrize("maker,level", [(W.kirkwood_problem, 4), (W.stern_sphere_problem, 3),
                                         (W.cavity_sphere_problem, 3)])
def test_treecode_matvec_matches_oracle(env, maker, level):
    """P = 6, theta = 0.5 (BASELINE.json configs 1-3) on meshes the oracle finishes in seconds that
    still span dozens of groups and leaves; multi-surface cases exercise several trees."""
    pg, torch, orc = env
    prob = maker(level)
    o = orc.Oracle(prob)
    x = np.random.default_rng(7 + level).normal(size=o.n)
    h, y = gpu_matvec(pg, torch, prob, x, K=4, P=6, theta=0.5)
    st = h.stats()
    assert st["m2p_evals"] > 0 and st["p2p_pairs"] < st["direct_equiv"]
    assert rel(y, o.matvec(x)) <= TOL_TREE
    h.close()


def test_treecode_error_decreases_with_order(env):
    pg, torch, orc = env
    prob = W.kirkwood_problem(3)
    o = orc.Oracle(prob)
    x = np.random.default_rng(11).normal(size=o.n)
    yo = o.matvec(x)
    errs = []
    for P in (1, 2, 4, 6, 8, 10, 12):
        h, y = gpu_matvec(pg, torch, prob, x, K=4, P=P, theta=0.6, ncrit=16)
        assert h.stats()["m2p_evals"] > 0
        errs.append(rel(y, yo))
        h.close()
    assert errs[3] <= TOL_TREE and errs[-1] < 1e-8
    assert all(b < a for a, b in zip(errs, errs[1:]))


@pytest.mark.parametrize("ncrit", [8, 40, 500])
def test_treecode_leaf_sizes(env, ncrit):
    pg, torch, orc = env
    prob = W.kirkwood_problem(3)
    o = orc.Oracle(prob)
    x = np.random.default_rng(12).normal(size=o.n)
    h, y = gpu_matvec(pg, torch, prob, x, K=4, P=6, theta=0.5, ncrit=ncrit)
    assert rel(y, o.matvec(x)) <= TOL_TREE
    h.close()


def test_kirkwood_full_size_sampled_rows(env):
    """BASELINE.json config 1 at full size (20480 panels, the configuration bench.py times): oracle rows
    computed one by one on a seeded sample; plus the Gauss identity as a size-independent property."""
    pg, torch, orc = env
    prob = W.kirkwood_problem(5)
    o = orc.Oracle(prob)
    rng = np.random.default_rng(2025)
    x = rng.normal(size=o.n)
    rows = np.sort(rng.choice(o.n, 600, replace=False))
    h, y = gpu_matvec(pg, torch, prob, x, K=4, P=6, theta=0.5)
    yo = o.matvec(x, rows)
    assert rel(y[rows], yo) <= TOL_TREE
    assert np.max(np.abs(y[rows] - yo)) <= 1e-3 * np.max(np.abs(yo))
    # Gauss identity through the treecode: phi = 1, dphi = 0 -> interior (Laplace) rows 1/2 - 1/2 = 0
    N = o.npan
    ones = torch.cat([torch.ones(N, dtype=torch.float64), torch.zeros(N, dtype=torch.float64)]).cuda()
    g = h.matvec(ones).cpu().numpy()
    assert np.max(np.abs(g[:N])) < 2e-4
    # solve + energy against the stored oracle value (tests/golden/make_golden.py) and Kirkwood's series
    xs, it, rr, rc = h.solve(tol=1e-6)
    es, ec = h.energy(xs)
    from closed_forms import kirkwood
    exact = kirkwood(W.spheres.KIRKWOOD_POS, W.spheres.KIRKWOOD_Q, 10.0, 4.0, 80.0, 0.125)
    assert abs(es - exact) / abs(exact) < 3e-3           # discretisation error of level 5 (~0.1 %)
    if os.path.exists(GOLDEN):
        gold = json.load(open(GOLDEN))
        if "kirkwood_l5" in gold:
            assert abs(es - gold["kirkwood_l5"]["E_solv_kJ_mol"]) / abs(es) < TOL_ENERGY
            assert abs(ec - gold["kirkwood_l5"]["E_coul_kJ_mol"]) / abs(ec) < 1e-12
    h.close()


def test_treecode_energy_vs_oracle(env):
    pg, torch, orc = env
    gold = json.load(open(GOLDEN)) if os.path.exists(GOLDEN) else {}
    prob = W.kirkwood_problem(4)
    h = pg.Handle.from_problem(prob, K=4, P=6, theta=0.5)
    x, it, rr, rc = h.solve(tol=1e-8)
    es, ec = h.energy(x)
    if "kirkwood_l4" in gold:
        eo = gold["kirkwood_l4"]["E_solv_kJ_mol"]
    else:
        o = orc.Oracle(prob)
        xo, _, _ = o.solve(tol=1e-8)
        eo = o.solvation_energy(xo)
    assert abs(es - eo) / abs(eo) < TOL_ENERGY
    h.close()


# ----------------------------------------------------------------------------------- edges and errors
def test_host_matvec_equals_device_matvec(env):
    pg, torch, orc = env
    prob = W.kirkwood_problem(3)
    h = pg.Handle.from_problem(prob, K=4, P=6, theta=0.5)
    x = np.random.default_rng(5).normal(size=h.n)
    yd = h.matvec(torch.tensor(x, device="cuda")).cpu().numpy()
    yh = h.matvec_host(x)
    assert rel(yh, yd) < 1e-13
    h.close()


def test_no_charges(env):
    pg, torch, orc = env
    v, t = W.icosphere(1, 3.0)
    h = pg.Handle([(v, t, 0, 1)], None, [4.0, 80.0], [0.0, 0.125], K=4, theta=0.0)
    assert float(h.rhs().abs().max()) == 0.0
    x, it, rr, rc = h.solve(tol=1e-8)
    assert it == 0 and float(x.abs().max()) == 0.0
    assert h.energy(x) == (0.0, 0.0)
    h.close()


def test_invalid_inputs(env):
    pg, torch, orc = env
    v, t = W.icosphere(1, 3.0)
    q = ([[0, 0, 0]], [1.0], [0])
    with pytest.raises(pg.PygbeError):                      # open mesh
        pg.Handle([(v, t[:-1], 0, 1)], q, [4.0, 80.0], [0.0, 0.125], check_mesh=True)
    with pytest.raises(pg.PygbeError):                      # flipped triangle
        t2 = t.copy(); t2[0] = t2[0][::-1]
        pg.Handle([(v, t2, 0, 1)], q, [4.0, 80.0], [0.0, 0.125], check_mesh=True)
    with pytest.raises(pg.PygbeError):                      # zero-area triangle
        t3 = t.copy(); t3[0] = [t3[0][0], t3[0][0], t3[0][1]]
        pg.Handle([(v, t3, 0, 1)], q, [4.0, 80.0], [0.0, 0.125])
    for bad in (dict(K=5), dict(P=0), dict(P=13), dict(theta=-0.1), dict(K_fine=11)):
        with pytest.raises(pg.PygbeError):
            pg.Handle([(v, t, 0, 1)], q, [4.0, 80.0], [0.0, 0.125], **bad)
    with pytest.raises(pg.PygbeError):                      # region out of range
        pg.Handle([(v, t, 0, 2)], q, [4.0, 80.0], [0.0, 0.125])
    with pytest.raises(pg.PygbeError):                      # charge region out of range
        pg.Handle([(v, t, 0, 1)], ([[0, 0, 0]], [1.0], [5]), [4.0, 80.0], [0.0, 0.125])
