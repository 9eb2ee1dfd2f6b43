"""Richardson extrapolation and observed order of convergence (section 2.4).

    f_exact ~ f1 + (f1 - f2) / (r^p - 1)                      eq. (16), f1 fine, f2 coarse, r = h2 / h1
    p = log((f3 - f2) / (f2 - f1)) / log(r)                   eq. (17), three grids with constant ratio r

plus the mesh-refinement driver the paper runs on its sphere test (section 3.1): solvation
energy on a sequence of icosphere levels through the CUDA path.  Host arithmetic on three scalars only; every
solve runs in libpygbe.
"""
import math


def observed_order(f1, f2, f3, r):
    """eq. (17): f1 finest, f3 coarsest, constant refinement ratio r = h2/h1 = h3/h2."""
    return math.log((f3 - f2) / (f2 - f1)) / math.log(r)


def extrapolate(f1, f2, r, p):
    """eq. (16): f1 fine-grid, f2 coarse-grid value."""
    return f1 + (f1 - f2) / (r ** p - 1.0)


def sphere_refinement_study(levels=(3, 4, 5), radius=4.0, kappa=0.0, K=3, P=12, theta=0.5, tol=1e-6, **kw):
    """Solvation energy of the centred-charge sphere on the given icosphere levels (each level divides the
    mean panel area by 4), the observed order w.r.t. area and the extrapolated value.  Defaults are the
    paper's Table 3: eps 4/80, kappa = 0, K = 3, P = 12, GMRES tol 1e-6."""
    import workloads as W
    import paper_1309_4018_b200 as pg
    energies, areas = [], []
    for lvl in levels:
        prob = W.born_problem(lvl, radius=radius, kappa=kappa)
        h = pg.Handle.from_problem(prob, K=K, P=P, theta=theta, **kw)
        x, it, rr, rc = h.solve(tol=tol)
        energies.append(h.energy(x)[0])
        areas.append(4.0 * math.pi * radius * radius / prob.n_panels)
        h.close()
    out = {"levels": list(levels), "mean_panel_area": areas, "E_solv_kJ_mol": energies}
    if len(levels) >= 3:
        f3, f2, f1 = energies[-3], energies[-2], energies[-1]
        r = areas[-2] / areas[-1]
        p = observed_order(f1, f2, f3, r)
        out.update(order_wrt_area=p, extrapolated=extrapolate(f1, f2, r, p))
    return out


if __name__ == "__main__":
    import json
    print(json.dumps(sphere_refinement_study(), indent=1))
