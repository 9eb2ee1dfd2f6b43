"""Plain restarted GMRES in numpy -- part of the oracle (TEST INFRASTRUCTURE).

PAPER.md:169 ("PyGBe uses a Krylov method ... one evaluation of the treecode per iteration"); tolerances
in Tables 1, 3.  Reading A16: x0 = 0, no preconditioner, stop when the
true-residual estimate ||b - A x|| / ||b|| <= tol, restart 100.  Textbook Arnoldi with modified
Gram-Schmidt and Givens rotations (Saad & Schultz).  Parity unpinned for the iterate path: only the
final residual and the energies derived from x are checked.
"""
import numpy as np


def gmres(matvec, b, tol=1e-8, restart=100, max_iter=1000):
    n = b.shape[0]
    x = np.zeros(n)
    bnorm = np.linalg.norm(b)
    if bnorm == 0.0:
        return x, 0, 0.0
    iters = 0
    rel = 1.0
    while iters < max_iter:
        r = b - matvec(x) if iters > 0 else b.copy()
        beta = np.linalg.norm(r)
        rel = beta / bnorm
        if rel <= tol:
            break
        m = min(restart, max_iter - iters)
        V = np.zeros((m + 1, n))
        H = np.zeros((m + 1, m))
        cs = np.zeros(m); sn = np.zeros(m)
        g = np.zeros(m + 1); g[0] = beta
        V[0] = r / beta
        k = 0
        for j in range(m):
            w = matvec(V[j])
            for i in range(j + 1):
                H[i, j] = np.dot(V[i], w)
                w -= H[i, j] * V[i]
            H[j + 1, j] = np.linalg.norm(w)
            if H[j + 1, j] > 0:
                V[j + 1] = w / H[j + 1, j]
            for i in range(j):
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -sn[i] * H[i, j] + cs[i] * H[i + 1, j]
                H[i, j] = t
            d = np.hypot(H[j, j], H[j + 1, j])
            cs[j], sn[j] = H[j, j] / d, H[j + 1, j] / d
            H[j, j] = d; H[j + 1, j] = 0.0
            g[j + 1] = -sn[j] * g[j]
            g[j] = cs[j] * g[j]
            iters += 1
            k = j + 1
            rel = abs(g[j + 1]) / bnorm
            if rel <= tol:
                break
        yk = np.linalg.solve(np.triu(H[:k, :k]), g[:k])
        x = x + V[:k].T @ yk
        if rel <= tol:
            break
    return x, iters, rel
