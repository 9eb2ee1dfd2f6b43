"""CPU checks of the host logic behind the M2P (no GPU): the coefficient tables that the library builds at create
(csrc/tables.cuh, through pygbe_host_table) reproduce direct sums of exp(-kappa r)/r and 1/r when the series they encode is
evaluated in numpy the way the kernels do (csrc/m2p.cuh): regrouped form on harmonically reduced moments, and the Laplace
form (one polynomial in d / r^2).  DESIGN.md 7; eq. (13)-(14)."""
import math

import numpy as np
import pytest

import paper_1309_4018_b200 as pg


@pytest.fixture(scope="module")
def lib():
    from paper_1309_4018_b200.build import build
    build()
    return pg.lib()


def canonical(P):
    return [(kx, ky, n - kx - ky) for n in range(P + 1) for kx in range(n, -1, -1) for ky in range(n - kx, -1, -1)]


def moments(P, src, q):
    return np.array([np.sum(q * src[:, 0] ** k[0] * src[:, 1] ** k[1] * src[:, 2] ** k[2]) for k in canonical(P)])


def apply_table(tab, M):
    off, k, c, _ = tab
    return np.array([np.dot(c[off[p]:off[p + 1]], M[k[off[p]:off[p + 1]]]) for p in range(len(off) - 1)])


def radial(P, kappa, r):
    F = np.zeros(P + 1)
    E = math.exp(-kappa * r)
    F[0] = E / r
    if P >= 1:
        F[1] = -E * (kappa * r + 1) / r ** 3
    for m in range(1, P):
        F[m + 1] = -((2 * m + 1) * F[m] - kappa * kappa * F[m - 1]) / (r * r)
    return F


def eval_regrouped(P, kappa, W, d):
    """sum_m F^(m) Q_m with Q_m = sum_e W_{m,e} d^e, W in the kernel's stream order (ez <= 1)."""
    q = np.zeros(P + 1)
    p = 0
    for ex in range(P + 1):
        for ey in range(P + 1 - ex):
            for ez in range(min(1, P - ex - ey) + 1):
                mono = d[0] ** ex * d[1] ** ey * d[2] ** ez
                for J in range((P - ex - ey - ez) // 2 + 1):
                    q[ex + ey + ez + J] += W[p] * mono
                    p += 1
    assert p == len(W)
    return float(np.dot(radial(P, kappa, float(np.linalg.norm(d))), q))


def eval_laplace_form(P, Cf, d):
    """(1/r) sum_f C_f u^f, u = d / r^2, coefficients in Horner order (fx, fy, fz descending)."""
    r2 = float(d @ d)
    u = d / r2
    acc, p = 0.0, 0
    for fx in range(P, -1, -1):
        for fy in range(P - fx, -1, -1):
            for fz in range(P - fx - fy, -1, -1):
                acc += Cf[p] * u[0] ** fx * u[1] ** fy * u[2] ** fz
                p += 1
    assert p == len(Cf)
    return acc / math.sqrt(r2)


def cell(rng, a, nsrc=8):
    src = rng.uniform(-a / 2, a / 2, size=(nsrc, 3))
    q = rng.normal(size=nsrc)
    d = rng.normal(size=3)
    d *= (a / 0.5) * rng.uniform(1.1, 3.0) / np.linalg.norm(d)        # beyond the MAC distance for theta = 0.5
    return src, q, d


@pytest.mark.parametrize("kappa", [0.0, 0.125, 0.5])
def test_regrouped_table_on_reduced_moments(lib, kappa):
    assert len(pg.host_table(0, 6, kappa)[0]) - 1 == 84 and len(pg.host_table(0, 8, kappa)[0]) - 1 == 165
    prev = None
    for P in (2, 4, 6, 8, 12):
        rng = np.random.default_rng(5)                                # the same cells for every order
        tab = pg.host_table(0, P, kappa)
        errs = []
        for _ in range(10):
            a = rng.choice([2.0, 4.0, 8.0])
            src, q, d = cell(rng, a)
            exact = np.sum(q * np.exp(-kappa * np.linalg.norm(d - src, axis=1)) / np.linalg.norm(d - src, axis=1))
            got = eval_regrouped(P, kappa, apply_table(tab, moments(P, src, q)), d)
            errs.append(abs(got - exact) * np.linalg.norm(d) / np.sum(np.abs(q)))
        worst = max(errs)
        # truncation error of the Taylor series: ratio |y - y_c| / |x - y_c| <= (sqrt(3)/2) / 2.2 = 0.39, so the error falls
        # geometrically with the order (a wrong or missing coefficient of order n would leave an error ~ 0.39^n)
        assert worst < 3.0 * 0.40 ** (P + 1), (P, worst)
        prev = worst
    assert prev < 1e-7                                                # P = 12: the table itself is right to that level


def test_reduction_is_an_identity_of_the_series(lib):
    """The reduced table (kappa-dependent) and the plain regrouping give the same truncated series: compare against the
    unreduced sum  sum_{|k|<=P} a^k M^k  evaluated through symbolic-free recurrences of the radial form (all ez)."""
    rng = np.random.default_rng(6)
    P, kappa = 8, 0.125
    tab = pg.host_table(0, P, kappa)
    ks = canonical(P)
    ix = {k: i for i, k in enumerate(ks)}
    for _ in range(5):
        src, q, d = cell(rng, 4.0)
        M = moments(P, src, q)
        # unreduced regrouping, written out: W_{m,e} = (-1)^|e| / e! sum_{|j| = m - |e|} M^(e+2j) / (2^|j| j!)
        qm = np.zeros(P + 1)
        f = [math.factorial(i) for i in range(P + 1)]
        for ex in range(P + 1):
            for ey in range(P + 1 - ex):
                for ez in range(P + 1 - ex - ey):
                    n = ex + ey + ez
                    for J in range((P - n) // 2 + 1):
                        W = 0.0
                        for jx in range(J + 1):
                            for jy in range(J + 1 - jx):
                                jz = J - jx - jy
                                W += M[ix[(ex + 2 * jx, ey + 2 * jy, ez + 2 * jz)]] / (2 ** J * f[jx] * f[jy] * f[jz])
                        qm[n + J] += (-1) ** n / (f[ex] * f[ey] * f[ez]) * W * d[0] ** ex * d[1] ** ey * d[2] ** ez
        full = float(np.dot(radial(P, kappa, float(np.linalg.norm(d))), qm))
        red = eval_regrouped(P, kappa, apply_table(tab, M), d)
        assert abs(red - full) <= 1e-13 * np.sum(np.abs(q)) / np.linalg.norm(d)


def test_laplace_form_table(lib):
    prev = None
    for P in (2, 6, 8, 12):
        rng = np.random.default_rng(7)                                # the same cells for every order
        tab = pg.host_table(1, P)
        nc = (P + 1) * (P + 2) * (P + 3) // 6
        assert len(tab[0]) - 1 == nc and tab[3].max() == P
        errs = []
        for _ in range(10):
            a = rng.choice([2.0, 4.0, 8.0])
            src, q, d = cell(rng, a)
            exact = np.sum(q / np.linalg.norm(d - src, axis=1))
            got = eval_laplace_form(P, apply_table(tab, moments(P, src, q)), d)
            errs.append(abs(got - exact) * np.linalg.norm(d) / np.sum(np.abs(q)))
        worst = max(errs)
        assert worst < 3.0 * 0.40 ** (P + 1), (P, worst)
        prev = worst
    # same truncated series as the regrouped form at kappa = 0
    rng = np.random.default_rng(8)
    src, q, d = cell(rng, 4.0)
    M = moments(8, src, q)
    a = eval_laplace_form(8, apply_table(pg.host_table(1, 8), M), d)
    b = eval_regrouped(8, 0.0, apply_table(pg.host_table(0, 8, 0.0), M), d)
    assert abs(a - b) <= 1e-13 * np.sum(np.abs(q)) / np.linalg.norm(d)
