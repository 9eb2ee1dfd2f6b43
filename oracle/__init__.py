"""CPU oracle of the PyGBe BEM operator -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes marshalling around oracle/pb_oracle.c (plain C, fp64, O(N^2)) plus a plain numpy GMRES
(oracle/gmres.py).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_1309_4018_b200 and shares no code with it;
inputs come from the `workloads` module (geometry only).

See pb_oracle.c's header for conventions, citations and the list of pins.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pb_oracle.c")
_LIB = os.path.join(_HERE, "libpb_oracle.so")
_lib = None


def build(force=False):
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_d = C.POINTER(C.c_double)
_i = C.POINTER(C.c_int)
_l = C.POINTER(C.c_long)
_PROB = [C.c_long, _d, _i, C.c_int, _i, _i, C.c_int, _d, _d, C.c_int, C.c_int, C.c_double, C.c_int]


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_quadrature.argtypes = [C.c_int, _d, _d]
        L.orc_gauss_legendre.argtypes = [C.c_int, _d, _d]
        L.orc_panel_geometry.argtypes = [C.c_long, _d, _d, _d, _d]
        L.orc_self_entry.argtypes = [_d, C.c_double, C.c_int, _d]
        L.orc_matvec.argtypes = _PROB + [_d, _l, C.c_long, _d]
        L.orc_entry.argtypes = _PROB + [C.c_int, C.c_long, C.c_long, _d, _d]
        L.orc_rhs.argtypes = _PROB + [C.c_long, _d, _d, _i, _d]
        L.orc_reaction_potential.argtypes = _PROB + [C.c_long, _d, _i, _d, _d]
        L.orc_solvation_energy.argtypes = [C.c_long, _d, _d, _d]
        L.orc_coulomb_energy.argtypes = [C.c_long, _d, _d, _i, C.c_int, _d, _d]
        L.orc_layer_potentials_at.argtypes = _PROB + [C.c_int, C.c_long, _d, _d, _d]
        L.orc_C0.restype = C.c_double
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what} failed with code {rc}")


def quadrature(K):
    b = np.zeros((K, 3)); w = np.zeros(K)
    _check(lib().orc_quadrature(K, _p(b, _d), _p(w, _d)), "quadrature")
    return b, w


def gauss_legendre(N):
    x = np.zeros(N); w = np.zeros(N)
    _check(lib().orc_gauss_legendre(N, _p(x, _d), _p(w, _d)), "gauss_legendre")
    return x, w


def self_entry(tri9, kappa, Nk=5):
    t = _f64(tri9).reshape(9)
    v = C.c_double()
    _check(lib().orc_self_entry(_p(t, _d), float(kappa), int(Nk), C.byref(v)), "self_entry")
    return v.value


def C0():
    return lib().orc_C0()


def num_threads():
    return lib().orc_num_threads()


class Oracle:
    """The D0 discretisation of one problem (workloads.Problem): matvec, rhs, solve, energies."""

    def __init__(self, problem, K=4, K_fine=19, thres=2.0, N_k=5):
        from workloads import concat_problem_arrays
        self.p = problem
        self.tri, self.surf, self.rin, self.rout = concat_problem_arrays(problem)
        self.eps, self.kappa = _f64(problem.eps), _f64(problem.kappa)
        self.K, self.K_fine, self.thres, self.N_k = int(K), int(K_fine), float(thres), int(N_k)
        self.npan = int(self.tri.shape[0])
        self.n = 2 * self.npan

    def _args(self):
        return [self.npan, _p(self.tri, _d), _p(self.surf, _i), len(self.rin), _p(self.rin, _i),
                _p(self.rout, _i), len(self.eps), _p(self.eps, _d), _p(self.kappa, _d), self.K,
                self.K_fine, self.thres, self.N_k]

    def geometry(self):
        c = np.zeros((self.npan, 3)); n = np.zeros((self.npan, 3)); A = np.zeros(self.npan)
        _check(lib().orc_panel_geometry(self.npan, _p(self.tri, _d), _p(c, _d), _p(n, _d), _p(A, _d)), "geom")
        return c, n, A

    def matvec(self, x, rows=None):
        x = _f64(x)
        assert x.shape == (self.n,)
        if rows is None:
            y = np.zeros(self.n)
            _check(lib().orc_matvec(*self._args(), _p(x, _d), None, 0, _p(y, _d)), "matvec")
        else:
            rows = np.ascontiguousarray(rows, dtype=np.int64)
            y = np.zeros(rows.shape[0])
            _check(lib().orc_matvec(*self._args(), _p(x, _d), _p(rows, _l), rows.shape[0], _p(y, _d)), "matvec")
        return y

    def entry(self, region, i, j):
        v = C.c_double(); k = C.c_double()
        _check(lib().orc_entry(*self._args(), int(region), int(i), int(j), C.byref(v), C.byref(k)), "entry")
        return v.value, k.value

    def rhs(self):
        b = np.zeros(self.n)
        q = self.p
        _check(lib().orc_rhs(*self._args(), len(q.charge_q), _p(q.charge_xyz, _d), _p(q.charge_q, _d),
                             _p(q.charge_region, _i), _p(b, _d)), "rhs")
        return b

    def dense(self):
        """Dense operator, column by column through the matrix-free matvec (tiny meshes only)."""
        A = np.zeros((self.n, self.n))
        e = np.zeros(self.n)
        for j in range(self.n):
            e[j] = 1.0
            A[:, j] = self.matvec(e)
            e[j] = 0.0
        return A

    def solve(self, tol=1e-8, restart=100, max_iter=1000):
        from .gmres import gmres
        b = self.rhs()
        x, iters, rel = gmres(self.matvec, b, tol=tol, restart=restart, max_iter=max_iter)
        return x, iters, rel

    def reaction_potential(self, x):
        x = _f64(x); q = self.p
        out = np.zeros(len(q.charge_q))
        _check(lib().orc_reaction_potential(*self._args(), len(q.charge_q), _p(q.charge_xyz, _d),
                                            _p(q.charge_region, _i), _p(x, _d), _p(out, _d)), "reaction")
        return out

    def solvation_energy(self, x):
        ph = self.reaction_potential(x)
        e = C.c_double()
        _check(lib().orc_solvation_energy(len(ph), _p(self.p.charge_q, _d), _p(ph, _d), C.byref(e)), "energy")
        return e.value

    def coulomb_energy(self):
        q = self.p
        e = C.c_double()
        _check(lib().orc_coulomb_energy(len(q.charge_q), _p(q.charge_xyz, _d), _p(q.charge_q, _d),
                                        _p(q.charge_region, _i), len(self.eps), _p(self.eps, _d),
                                        C.byref(e)), "coulomb")
        return e.value

    def layer_potentials_at(self, region, pts):
        pts = _f64(pts).reshape(-1, 3)
        V = np.zeros(len(pts)); Kd = np.zeros(len(pts))
        _check(lib().orc_layer_potentials_at(*self._args(), int(region), len(pts), _p(pts, _d),
                                             _p(V, _d), _p(Kd, _d)), "layer_potentials_at")
        return V, Kd
