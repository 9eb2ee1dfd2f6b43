"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, -m "not gpu").

Each test names the mistake it would catch.  Closed forms live in tests/closed_forms.py (scipy only).
"""
import math

import numpy as np
import pytest

import workloads as W
from closed_forms import C0, born, kirkwood, stern_sphere, cavity_sphere, layered_sphere


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


# ---------------------------------------------------------------------------------------------- tables
@pytest.mark.parametrize("K,deg", [(1, 1), (3, 2), (4, 3), (7, 5), (19, 9)])
def test_quadrature_moments(orc, K, deg):
    """sum_g w_g L1^a L2^b = 2 a! b!/(a+b+2)! for all a+b <= degree (weights sum to 1) -- catches any
    wrong node or weight in the rule tables (reading A5 / A7b)."""
    b, w = orc.quadrature(K)
    assert abs(w.sum() - 1) < 1e-14
    assert np.allclose(b.sum(axis=1), 1.0, atol=1e-15)
    for a in range(deg + 1):
        for c in range(deg + 1 - a):
            exact = 2.0 * math.factorial(a) * math.factorial(c) / math.factorial(a + c + 2)
            got = np.sum(w * b[:, 0] ** a * b[:, 1] ** c)
            assert abs(got - exact) < 2e-15, (K, a, c)
    # the rule is NOT exact one degree higher (guards against testing a vacuous condition)
    a, c = deg + 1, 0
    exact = 2.0 * math.factorial(a) * math.factorial(c) / math.factorial(a + c + 2)
    if K > 1:
        assert abs(np.sum(w * b[:, 0] ** a * b[:, 1] ** c) - exact) > 1e-8


def test_k19_positive_interior(orc):
    b, w = orc.quadrature(19)
    assert (w > 0).all() and (b > 0).all()


@pytest.mark.parametrize("N", [1, 2, 5, 9, 64])
def test_gauss_legendre(orc, N):
    x, w = orc.gauss_legendre(N)
    xr, wr = np.polynomial.legendre.leggauss(N)
    o = np.argsort(x)
    assert np.allclose(x[o], xr, atol=1e-14) and np.allclose(w[o], wr, atol=1e-14)


# ------------------------------------------------------------------------------------- self integral
def _asinh_closed_form(t):
    """int_T 1/r dA about the centroid: sum_sides h [asinh(s2/h) - asinh(s1/h)]."""
    t = np.asarray(t, float).reshape(3, 3)
    c = t.mean(axis=0)
    tot = 0.0
    for s in range(3):
        a, b = t[s], t[(s + 1) % 3]
        e = (b - a) / np.linalg.norm(b - a)
        sa, sb = np.dot(a - c, e), np.dot(b - c, e)
        h = np.linalg.norm((a - c) - sa * e)
        tot += h * (math.asinh(sb / h) - math.asinh(sa / h))
    return tot


def test_self_integral_equilateral(orc):
    """Unit equilateral triangle: int 1/r = 2.281037988902839 (closed form); N_k -> infinity."""
    t = [0, 0, 0, 1, 0, 0, 0.5, math.sqrt(3) / 2, 0]
    assert abs(_asinh_closed_form(t) - 2.281037988902839) < 1e-14
    v = orc.self_entry(t, 0.0, 64) * 4 * math.pi
    assert abs(v - 2.281037988902839) < 1e-13
    v5 = orc.self_entry(t, 0.0, 5) * 4 * math.pi
    assert abs(v5 - 2.281037988902839) / 2.28 < 3e-4      # N_k = 5 accuracy quoted in reading A6


def test_self_integral_general_triangle_and_yukawa_limit(orc):
    rng = np.random.default_rng(5)
    for _ in range(5):
        t = rng.normal(size=9)
        exact = _asinh_closed_form(t)
        assert abs(orc.self_entry(t, 0.0, 128) * 4 * math.pi - exact) < 1e-9 * exact
        # Yukawa: kappa -> 0 tends to Laplace, and is smaller for kappa > 0 with first-order slope -area
        v0 = orc.self_entry(t, 0.0, 64)
        v1 = orc.self_entry(t, 1e-6, 64)
        tt = t.reshape(3, 3)
        area = 0.5 * np.linalg.norm(np.cross(tt[1] - tt[0], tt[2] - tt[0]))
        # int (e^{-k r}/r) = int 1/r - k * area + O(k^2)
        assert abs((v0 - v1) * 4 * math.pi / 1e-6 - area) < 1e-3 * area


def test_self_integral_yukawa_bruteforce(orc):
    """Yukawa self integral against brute-force polar integration (scipy.dblquad-free: fine Gauss)."""
    t = np.array([0, 0, 0, 1.3, 0.1, 0, 0.4, 0.9, 0.2], float)
    kappa = 0.7
    tt = t.reshape(3, 3)
    c = tt.mean(axis=0)
    x, w = np.polynomial.legendre.leggauss(200)
    tot = 0.0
    # Duffy: split into 3 sub-triangles (c, a, b); map (u,v) in [0,1]^2 -> c + u((1-v)(a-c) + v(b-c))
    u = 0.5 * (x + 1); wu = 0.5 * w
    for s in range(3):
        a, b = tt[s] - c, tt[(s + 1) % 3] - c
        jac = np.linalg.norm(np.cross(a, b))
        for vi, wv in zip(u, wu):
            d = (1 - vi) * a + vi * b
            r = u * np.linalg.norm(d)
            tot += wv * np.sum(wu * np.exp(-kappa * r) / np.linalg.norm(d)) * jac
    got = orc.self_entry(t, kappa, 96) * 4 * math.pi
    assert abs(got - tot) < 1e-10 * tot


# ---------------------------------------------------------------------------------------- geometry/rhs
def test_geometry_and_rhs_closed_form(orc):
    """RHS of a centred charge is q/(4 pi eps1 |c_i|) on the interior rows and 0 on the exterior rows
    (eq. 9/11) -- catches a missing 1/(4 pi), 1/eps or a row-layout swap."""
    p = W.born_problem(2)
    o = orc.Oracle(p)
    c, n, A = o.geometry()
    v, t = p.surfaces[0].vertices, p.surfaces[0].triangles
    assert np.allclose(c, v[t].mean(axis=1))
    assert np.allclose(np.einsum("ij,ij->i", n, c / np.linalg.norm(c, axis=1)[:, None]), 1.0, atol=2e-2)
    assert abs(A.sum() - 4 * math.pi * 16) / (4 * math.pi * 16) < 0.03
    b = o.rhs()
    N = o.npan
    assert np.allclose(b[:N], 1.0 / (4 * math.pi * 4.0 * np.linalg.norm(c, axis=1)), rtol=1e-14)
    assert np.all(b[N:] == 0.0)


def test_coulomb_energy_two_charges(orc):
    p = W.born_problem(1)
    p.charge_xyz = np.array([[0.0, 0, 0], [0, 0, 2.0], [1.0, 0, 0]])
    p.charge_q = np.array([1.0, -0.5, 0.25]); p.charge_region = np.array([0, 0, 0], dtype=np.int32)
    o = orc.Oracle(p)
    pairs = (1.0 * -0.5) / 2.0 + (1.0 * 0.25) / 1.0 + (-0.5 * 0.25) / math.sqrt(5.0)
    assert abs(o.coulomb_energy() - C0 / (4 * math.pi * 4.0) * pairs) < 1e-10


# -------------------------------------------------------------------------------- eq. (10) structure
def test_eq10_block_structure(orc):
    """Dense operator on the 20-panel icosahedron equals [[I/2 + K_L, -V_L], [I/2 - K_Y, eps1/eps2 V_Y]]
    built entry by entry -- catches sign / block / eps-ratio mistakes (reading A1)."""
    p = W.born_problem(0)
    o = orc.Oracle(p)
    N = o.npan
    assert N == 20
    A = o.dense()
    VL = np.zeros((N, N)); KL = np.zeros((N, N)); VY = np.zeros((N, N)); KY = np.zeros((N, N))
    for i in range(N):
        for j in range(N):
            VL[i, j], KL[i, j] = o.entry(0, i, j)
            VY[i, j], KY[i, j] = o.entry(1, i, j)
    I = np.eye(N)
    ref = np.block([[0.5 * I + KL, -VL], [0.5 * I - KY, (4.0 / 80.0) * VY]])
    assert np.allclose(A, ref, rtol=0, atol=1e-15)
    assert np.all(np.diag(KL) == 0) and np.all(np.diag(VL) > 0)
    # Yukawa entries are smaller than Laplace ones and tend to them as kappa -> 0
    assert np.all(VY < VL)
    p0 = W.born_problem(0, kappa=1e-9)
    o0 = orc.Oracle(p0)
    assert abs(o0.entry(1, 3, 7)[0] - VL[3, 7]) < 1e-9 and abs(o0.entry(1, 3, 7)[1] - KL[3, 7]) < 1e-9


def test_lu_vs_gmres(orc):
    p = W.born_problem(1)
    o = orc.Oracle(p)
    A = o.dense(); b = o.rhs()
    x_lu = np.linalg.solve(A, b)
    x, it, rel = o.solve(tol=1e-12)
    assert rel <= 1e-12 and np.linalg.norm(A @ x - b) / np.linalg.norm(b) < 2e-12
    assert abs(o.solvation_energy(x) - o.solvation_energy(x_lu)) < 1e-8
    # sampled-row matvec agrees with the full one
    rows = np.array([0, 5, o.npan, 2 * o.npan - 1])
    assert np.array_equal(o.matvec(x, rows), o.matvec(x)[rows])


# ------------------------------------------------------------------------------------ Gauss identity
def test_gauss_identity(orc):
    """Laplace double layer of a unit density over a closed surface: -1/2 on the surface, -1 inside,
    0 outside (sign convention of reading A3: normal out of the enclosed region, derivative at the
    source) -- catches a flipped normal, d = y - x, or a wrong 1/(4 pi)."""
    p = W.born_problem(3, kappa=0.0)
    o = orc.Oracle(p, K=4, K_fine=19, thres=2.0)
    N = o.npan
    x = np.concatenate([np.ones(N), np.zeros(N)])
    y = o.matvec(x)                       # interior rows: 1/2 + sum_j K_L,ij
    rowsum = y[:N] - 0.5
    assert np.max(np.abs(rowsum + 0.5)) < 1e-4          # 4.3e-5 quoted in SURVEY 8(c) for thres 2
    o2 = orc.Oracle(p, K=4, K_fine=4, thres=0.0)        # no near-field treatment: much worse
    dev_plain = np.max(np.abs(o2.matvec(x)[:N] - 0.5 + 0.5))
    assert 1e-3 < dev_plain < 5e-3
    V, Kd = o.layer_potentials_at(0, [[0.3, -0.2, 0.5], [0, 0, 0], [9.0, 1.0, -2.0]])
    assert abs(Kd[0] + 1) < 2e-5 and abs(Kd[1] + 1) < 2e-5 and abs(Kd[2]) < 1e-6
    # single layer of unit density at the centre = area-weighted 1/(4 pi r) ~ R (to mesh accuracy)
    assert abs(V[1] - 4.0) < 0.03


# ------------------------------------------------------------------------------- paper's printed value
def _richardson(f_fine, f_coarse, r=4.0, p=1.0):
    return f_fine + (f_fine - f_coarse) / (r ** p - 1.0)          # eq. (16)


@pytest.fixture(scope="module")
def born_energies(orc):
    out = {}
    for kappa in (0.0, 0.125):
        for lvl in (1, 2, 3):
            o = orc.Oracle(W.born_problem(lvl, kappa=kappa))
            x, it, rel = o.solve(tol=1e-10)
            out[(kappa, lvl)] = o.solvation_energy(x)
    return out


def test_paper_sphere_value(born_energies):
    """analytic -41.2465 kJ/mol (R = 4 A, +1e, eps 4/80, kappa 0); the paper's Richardson
    value is -41.2467.  Fixes the unit constant (A17) and the whole assemble-solve-energy chain."""
    assert abs(born(1, 4, 4, 80, 0) - (-41.2465)) < 5e-5
    E = born_energies
    ext = _richardson(E[(0.0, 3)], E[(0.0, 2)])
    assert abs(ext - (-41.2465)) < 0.01                           # 2e-4 relative
    # observed order w.r.t. area ~ 1 (paper: 1.013), eq. (17)
    order = math.log((E[(0.0, 1)] - E[(0.0, 2)]) / (E[(0.0, 2)] - E[(0.0, 3)])) / math.log(4.0)
    assert 0.9 < order < 1.1


def test_born_with_salt(born_energies):
    """BASELINE.json config 0 closed form -41.970082 kJ/mol; level-3 D0 value is 0.33 % off
    (first-order discretisation error), Richardson from levels 2, 3 within 0.01 %."""
    E = born_energies
    exact = born(1, 4, 4, 80, 0.125)
    assert abs(exact - (-41.970082)) < 1e-6
    assert abs(E[(0.125, 3)] - exact) / abs(exact) < 4e-3
    assert abs(_richardson(E[(0.125, 3)], E[(0.125, 2)]) - exact) / abs(exact) < 1e-4
    # errors fall by ~4 per level
    e1, e2, e3 = (abs(E[(0.125, l)] - exact) for l in (1, 2, 3))
    assert 3.5 < e1 / e2 < 4.6 and 3.5 < e2 / e3 < 4.6


def test_kirkwood_series(orc):
    """Off-centre charges (BASELINE.json config 1 geometry at coarse levels) against the Kirkwood
    series: -7.5558587021 kJ/mol -- catches anything that a centred charge cannot see (double-layer
    term, normals, non-constant densities)."""
    exact = kirkwood(W.spheres.KIRKWOOD_POS, W.spheres.KIRKWOOD_Q, 10.0, 4.0, 80.0, 0.125)
    assert abs(exact - (-7.5558587021)) < 1e-9
    assert abs(kirkwood(W.spheres.KIRKWOOD_POS, W.spheres.KIRKWOOD_Q, 10.0, 4.0, 80.0, 0.0) - (-7.3820296213)) < 1e-9
    E = {}
    for lvl in (2, 3):
        o = orc.Oracle(W.kirkwood_problem(lvl))
        x, it, rel = o.solve(tol=1e-9)
        E[lvl] = o.solvation_energy(x)
    assert abs(E[3] - exact) / abs(exact) < 0.03
    assert abs(E[2] - exact) / abs(E[3] - exact) > 3.0
    assert abs(_richardson(E[3], E[2]) - exact) / abs(exact) < 3e-3


# --------------------------------------------------------------------------------- multi-surface rule
def test_stern_layer_analytic(orc):
    """Concentric Stern layer: -41.866708 kJ/mol.  Pins sigma/c for a surface seen from its outer
    region and the Laplace kernel in a region with eps2 (reading A4)."""
    exact = stern_sphere(1, 4, 6, 4, 80, 0.125)
    assert abs(exact - (-41.866708)) < 1e-6
    E = {}
    for lvl in (1, 2):
        o = orc.Oracle(W.stern_sphere_problem(lvl))
        x, it, rel = o.solve(tol=1e-10)
        E[lvl] = o.solvation_energy(x)
    assert abs(E[2] - exact) / abs(exact) < 0.02
    assert abs(_richardson(E[2], E[1]) - exact) / abs(exact) < 2e-3


def test_cavity_analytic(orc):
    """Concentric solvent-filled cavity, charge in the shell: -35.634859 kJ/mol.  Pins the inner
    boundary of the charged region (sigma = -1, c = eps_cav/eps1 = 20)."""
    exact = cavity_sphere(1, 2, 8, 5, 4, 80, 0.125, 80)
    assert abs(exact - (-35.634859)) < 1e-6
    E = {}
    for lvl in (1, 2):
        o = orc.Oracle(W.cavity_sphere_problem(lvl))
        x, it, rel = o.solve(tol=1e-10)
        E[lvl] = o.solvation_energy(x)
    assert abs(E[2] - exact) / abs(exact) < 0.04
    assert abs(_richardson(E[2], E[1]) - exact) / abs(exact) < 5e-3


def test_layered_closed_form_reduces_to_the_special_cases():
    """The general concentric-layer solution (any number of layers, Laplace or Yukawa each) against the four
    special cases derived separately above."""
    assert abs(layered_sphere(1, 0.0, [4], [4, 80], [0, 0.125], 0) - born(1, 4, 4, 80, 0.125)) < 1e-10
    assert abs(layered_sphere(1, 0.0, [4, 6], [4, 80, 80], [0, 0, 0.125], 0) - stern_sphere(1, 4, 6, 4, 80, 0.125)) < 1e-10
    assert abs(layered_sphere(1, 5.0, [2, 8], [80, 4, 80], [0, 0, 0.125], 1) - cavity_sphere(1, 2, 8, 5, 4, 80, 0.125, 80)) < 1e-9
    assert abs(layered_sphere(1, 3.0, [10], [4, 80], [0, 0.125], 0) - kirkwood([[0, 0, 3.0]], [1.0], 10, 4, 80, 0.125)) < 1e-9


def test_nested_ion_bearing_cavity_analytic(orc):
    """PAPER.md:131 "cavities ... large enough to contain ions ... an interior Stern layer": a cavity with salt
    (Yukawa, regular at the origin) inside its own Stern layer inside the protein shell inside an outer Stern
    layer inside the salt solvent; five regions, four surfaces, charge in the shell: -39.694277 kJ/mol.  Pins the
    per-region rule of reading A4 for a Yukawa region that is the *inside* of its only surface and for a Laplace
    region bounded on both sides by solvent-like media."""
    exact = layered_sphere(1, 5.0, [1.5, 2.5, 8, 10], [80, 80, 4, 80, 80], [0.5, 0, 0, 0, 0.125], 2)
    assert abs(exact - (-39.694277)) < 1e-6
    # the salt in the cavity matters: the same geometry with pure water inside differs by 6 %
    assert abs(layered_sphere(1, 5.0, [1.5, 2.5, 8, 10], [80, 80, 4, 80, 80], [0.0, 0, 0, 0, 0.125], 2) - exact) / abs(exact) > 0.05
    E = {}
    for lvl in (1, 2):
        o = orc.Oracle(W.nested_sphere_problem(lvl))
        x, it, rel = o.solve(tol=1e-10)
        E[lvl] = o.solvation_energy(x)
    assert abs(E[2] - exact) / abs(exact) < 0.02
    assert abs(_richardson(E[2], E[1]) - exact) / abs(exact) < 5e-3


def test_transparent_interfaces(orc):
    """A surface with identical media on both sides must not change the energy (up to discretisation):
    Stern surface with kappa_out = 0, cavity with eps_cav = eps1."""
    base = orc.Oracle(W.born_problem(2, kappa=0.0))
    xb, _, _ = base.solve(tol=1e-10)
    Eb = base.solvation_energy(xb)
    st = orc.Oracle(W.stern_sphere_problem(2, kappa=0.0))
    xs, _, _ = st.solve(tol=1e-10)
    assert abs(st.solvation_energy(xs) - Eb) / abs(Eb) < 1e-3
    ref = orc.Oracle(W.Problem([W.Surface(*W.icosphere(2, 8.0), 0, 1)], [4, 80], [0, 0.125],
                               [[0, 0, 5.0]], [1.0], [0]))
    xr, _, _ = ref.solve(tol=1e-10)
    Er = ref.solvation_energy(xr)
    cav = orc.Oracle(W.cavity_sphere_problem(2, eps_cav=4.0))
    xc, _, _ = cav.solve(tol=1e-10)
    assert abs(cav.solvation_energy(xc) - Er) / abs(Er) < 5e-3
    cav80 = orc.Oracle(W.cavity_sphere_problem(2))
    xc8, _, _ = cav80.solve(tol=1e-10)
    assert abs(cav80.solvation_energy(xc8) - Er) / abs(Er) > 0.03      # a real cavity does matter


# ------------------------------------------------------------- two small branches ("unpinned (mine)")
def test_rhs_of_a_charge_in_a_screened_region(orc):
    """orc_rhs with a charge sitting in a kappa != 0 region (eq. 9/11 with the Yukawa Green's function,
    PAPER.md:55-58, :98): rows of that region are q exp(-kappa r) / (4 pi eps r), rows of the other region 0.
    Every other test keeps its charges in kappa = 0 regions, so the exp(-kappa r) factor would go unnoticed."""
    p = W.born_problem(1)
    pos = np.array([[0.0, 0.0, 7.0], [5.0, -6.0, 1.0]])
    q = np.array([0.75, -1.25])
    p.charge_xyz, p.charge_q, p.charge_region = pos, q, np.array([1, 1], dtype=np.int32)
    o = orc.Oracle(p)
    c, _, _ = o.geometry()
    b = o.rhs()
    N = o.npan
    kappa, eps2 = 0.125, 80.0
    want = sum(qk * np.exp(-kappa * np.linalg.norm(c - rk, axis=1)) / (4 * math.pi * eps2 * np.linalg.norm(c - rk, axis=1))
               for qk, rk in zip(q, pos))
    assert np.all(b[:N] == 0.0)
    assert np.allclose(b[N:], want, rtol=1e-14, atol=0)
    # and it is not the Laplace value: the screening changes the rows by tens of per cent at these distances
    lap = sum(qk / (4 * math.pi * eps2 * np.linalg.norm(c - rk, axis=1)) for qk, rk in zip(q, pos))
    assert np.max(np.abs(b[N:] - lap) / np.abs(lap)) > 0.2


def test_near_singular_rule_switches_at_thres_squared_times_2A(orc):
    """Reading A7: the K_fine-point rule replaces the K-point rule iff |x_i - c_j|^2 < thres^2 * 2 A_j,
    strictly, with L_j = sqrt(2 A_j).  Constructed pair: source = right triangle with legs 1 (2A = 1 exactly),
    target = the same triangle lifted by 2 in z (centroid distance exactly 2, d^2 = 4 exactly).  The two candidate
    values come from the oracle itself with the rule forced on (thres huge) and off (thres 0)."""
    src = np.array([[0.0, 0, 0], [1.0, 0, 0], [0.0, 1, 0]])
    tgt = src + np.array([0.0, 0.0, 2.0])
    verts = np.concatenate([src, tgt])
    tris = np.array([[0, 1, 2], [3, 4, 5]], dtype=np.int32)
    p = W.Problem([W.Surface(verts, tris, 0, 1)], [4.0, 80.0], [0.0, 0.125], np.zeros((1, 3)), [1.0], [0])

    def entry(thres, region=1):
        return orc.Oracle(p, K=4, K_fine=19, thres=thres).entry(region, 1, 0)      # target panel 1, source panel 0

    fine, coarse = entry(1e9), entry(0.0)
    assert abs(fine[0] - coarse[0]) > 1e-6 * abs(fine[0])                        # the two rules differ measurably here
    assert entry(2.0) == coarse                      # d^2 = 4 = thres^2 * 2A: strict '<', the K-point rule stays
    assert entry(2.0 * (1 + 1e-15)) == fine          # one ulp above: K_fine
    assert entry(2.5) == fine                        # thres^2 * 2A = 6.25 > 4;  with L^2 = A it would be 3.125 < 4
    assert entry(1.99) == coarse
    assert entry(2.9, region=0) == orc.Oracle(p, thres=1e9).entry(0, 1, 0)       # same switch under the Laplace kernel
