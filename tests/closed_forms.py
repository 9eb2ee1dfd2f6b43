"""Closed-form solutions used to pin the oracle.  Derived from eq. (1) of the paper by
separation of variables; they share nothing with oracle/ or the CUDA path (scipy special functions
only).  C0 = qe^2 N_A 1e7 / eps0 [kJ A/(mol e^2)], the constant that reproduces PAPER.md:229."""
import numpy as np
from scipy.special import spherical_kn, eval_legendre

QE, NA, EPS0 = 1.60217646e-19, 6.0221415e23, 8.854187818e-12
C0 = QE * QE * NA * 1e7 / EPS0


def born(q, a, eps_in, eps_out, kappa):
    """Centred charge q in a sphere of radius a; solvent with inverse Debye length kappa."""
    return C0 * q * q / (8 * np.pi * a) * (1.0 / (eps_out * (1 + kappa * a)) - 1.0 / eps_in)


def kirkwood(pos, q, a, eps_in, eps_out, kappa, nmax=100):
    """Kirkwood series for point charges inside a sphere of radius a (origin-centred)."""
    pos = np.asarray(pos, float); q = np.asarray(q, float)
    r = np.linalg.norm(pos, axis=1)
    x = kappa * a
    tot = 0.0
    for n in range(nmax + 1):
        if kappa > 0:
            lam = x * spherical_kn(n, x, derivative=True) / spherical_kn(n, x)
        else:
            lam = -(n + 1.0)
        cn = (eps_in * (n + 1) + eps_out * lam) / (eps_in * n - eps_out * lam)
        for k in range(len(q)):
            for l in range(len(q)):
                if r[k] == 0 or r[l] == 0:
                    cosg = 1.0
                    rr = 0.0 if n > 0 else 1.0
                else:
                    cosg = np.dot(pos[k], pos[l]) / (r[k] * r[l])
                    rr = (r[k] * r[l]) ** n
                tot += q[k] * q[l] * cn * rr / a ** (2 * n + 1) * eval_legendre(n, np.clip(cosg, -1, 1))
    return 0.5 * C0 / (4 * np.pi * eps_in) * tot


def stern_sphere(q, R, a, eps_in, eps_out, kappa):
    """Centred charge; dielectric sphere R inside an ion-exclusion shell up to a; salt outside."""
    phi = q / (4 * np.pi) * (1 / (eps_out * R) - kappa / (eps_out * (1 + kappa * a)) - 1 / (eps_in * R))
    return 0.5 * C0 * q * phi


def cavity_sphere(q, r_c, R, r_k, eps_in, eps_out, kappa, eps_cav, nmax=60):
    """Charge on the axis at r_k inside a shell r_c < r < R (eps_in); cavity r < r_c (eps_cav, Laplace);
    solvent r > R (eps_out, kappa).  Per harmonic a 4x4 solve for scaled (F, B, G, A)."""
    Q = q / (4 * np.pi * eps_in)
    x = kappa * R
    phi = 0.0
    for n in range(nmax + 1):
        lam = x * spherical_kn(n, x, derivative=True) / spherical_kn(n, x) if kappa > 0 else -(n + 1.0)
        # unknowns: f = F r_c^n, b = B R^n, g = G r_c^-(n+1), A' = A k_n(x)
        t = (r_c / R) ** n            # B r_c^n = b t
        u = (r_c / R) ** (n + 1)      # G R^-(n+1) = g u
        ci = Q * r_c ** n / r_k ** (n + 1)    # Coulomb harmonic at r_c
        co = Q * r_k ** n / R ** (n + 1)      # Coulomb harmonic at R
        M = np.array([
            [1.0, -t, -1.0, 0.0],
            [eps_cav * n, -eps_in * n * t, eps_in * (n + 1), 0.0],
            [0.0, 1.0, u, -1.0],
            [0.0, eps_in * n, -eps_in * (n + 1) * u, -eps_out * lam],
        ])
        rhs = np.array([ci, eps_in * n * ci, -co, eps_in * (n + 1) * co])
        f, b, g, A = np.linalg.solve(M, rhs)
        phi += b * (r_k / R) ** n + g * (r_c / r_k) ** (n + 1)
    return 0.5 * C0 * q * phi
