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


def layered_sphere(q, r_k, radii, eps, kappa, charge_layer, nmax=60):
    """Charge q on the axis at radius r_k inside layer `charge_layer` (kappa = 0 there) of a concentric system:
    layer 0 is the ball r < radii[0], layer l lies between radii[l-1] and radii[l], the last layer is the
    exterior.  Layer l has (eps[l], kappa[l]).  Separation of variables of eq. (1): per Legendre order n the
    potential in layer l is A_l f_l(r) + B_l g_l(r) (+ the Coulomb harmonic in the charge's layer) with
    (f, g) = (r^n, r^-(n+1)) for kappa = 0 and (i_n(kappa r), k_n(kappa r)) otherwise; B_0 = 0, A_last = 0; phi and
    eps dphi/dr are continuous at every radius.  Returns the solvation energy 1/2 C0 q phi_reac(r_k)."""
    from scipy.special import spherical_in
    radii = [float(a) for a in radii]
    L = len(radii) + 1
    assert len(eps) == L and len(kappa) == L and kappa[charge_layer] == 0.0
    Q = q / (4 * np.pi * eps[charge_layer])

    def basis(l, n, r):
        """(f, f', g, g') of layer l at r, each pair scaled to O(1) at the layer's reference radius."""
        ref = radii[min(l, L - 2)]
        if kappa[l] == 0.0:
            f, df = (r / ref) ** n, n * (r / ref) ** n / r
            g, dg = (ref / r) ** (n + 1), -(n + 1) * (ref / r) ** (n + 1) / r
        else:
            k = kappa[l]
            fs, gs = spherical_in(n, k * ref), spherical_kn(n, k * ref)
            f, df = spherical_in(n, k * r) / fs, k * spherical_in(n, k * r, derivative=True) / fs
            g, dg = spherical_kn(n, k * r) / gs, k * spherical_kn(n, k * r, derivative=True) / gs
        return f, df, g, dg

    phi = 0.0
    for n in range((nmax if r_k > 0 else 0) + 1):
        # unknown index: A_l -> 2l, B_l -> 2l + 1
        M = np.zeros((2 * L, 2 * L)); rhs = np.zeros(2 * L)
        M[0, 1] = 1.0                      # B_0 = 0 (regular at the origin)
        M[1, 2 * (L - 1)] = 1.0            # A_last = 0 (decays at infinity)
        row = 2
        for i, a in enumerate(radii):      # interface between layers i and i + 1
            fi, dfi, gi, dgi = basis(i, n, a)
            fo, dfo, go, dgo = basis(i + 1, n, a)
            M[row, 2 * i], M[row, 2 * i + 1], M[row, 2 * i + 2], M[row, 2 * i + 3] = fi, gi, -fo, -go
            M[row + 1, 2 * i], M[row + 1, 2 * i + 1] = eps[i] * dfi, eps[i] * dgi
            M[row + 1, 2 * i + 2], M[row + 1, 2 * i + 3] = -eps[i + 1] * dfo, -eps[i + 1] * dgo
            if i == charge_layer:          # outer boundary of the charge's layer: Coulomb harmonic Q r_k^n / r^(n+1)
                c = Q * r_k ** n / a ** (n + 1) if r_k > 0 else (Q / a if n == 0 else 0.0)
                rhs[row] -= c
                rhs[row + 1] -= eps[i] * (-(n + 1) * c / a)
            if i + 1 == charge_layer:      # inner boundary: Q r^n / r_k^(n+1)
                c = Q * a ** n / r_k ** (n + 1)
                rhs[row] += c
                rhs[row + 1] += eps[i + 1] * (n * c / a)
            row += 2
        sol = np.linalg.solve(M, rhs)
        if r_k > 0:
            f, _, g, _ = basis(charge_layer, n, r_k)
            phi += sol[2 * charge_layer] * f + sol[2 * charge_layer + 1] * g
        else:
            phi += sol[2 * charge_layer]   # f = 1 at the origin for n = 0, g term absent (B_0 = 0)
    return 0.5 * C0 * q * phi
