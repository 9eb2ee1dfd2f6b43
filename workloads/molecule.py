"""Protein-like synthetic molecules (BASELINE.json configs 2-4): geometry generation ONLY.

Stand-ins for the MSMS / pdb2pqr inputs of the paper (Tables 1-6; 1HEL, 3BTK are not available).
Recipe:
  atoms    confined self-avoiding random walk, 1.5 A steps; radii U(1.2, 2.0); charges U(-0.6, 0.6) shifted
           so that the total is the nearest integer
  surface  isosurface rho = 1 of rho(x) = sum_i exp(-B(|x - c_i|^2 / R_i^2 - 1)), R_i = r_i + probe,
           B = 2.3, extracted by marching tetrahedra on a regular grid (Kuhn split of each cube into six
           tetrahedra, which is face-compatible between neighbouring cubes, so the mesh is watertight),
           edge crossings clamped to [0.1, 0.9] of the edge (no zero-area triangles), outermost connected
           component kept, triangles oriented from rho > 1 (inside) to rho < 1 (outside).
No kernel, quadrature or operator arithmetic of the method lives here.
"""
import itertools

import numpy as np

from .problem import Problem, Surface
from .spheres import icosphere


def saw_molecule(n_atoms, seed, step=1.5, exclusions=(), excl_radius=5.0, n_candidates=8):
    """Confined self-avoiding walk.  Returns (centres [n,3], radii [n], charges [n], R_conf).
    exclusions: points the walk keeps `excl_radius` away from (room for solvent-filled cavities)."""
    rng = np.random.default_rng(seed)
    r_conf = (n_atoms * 20.0 * 3.0 / (4.0 * np.pi)) ** (1.0 / 3.0)
    excl = np.asarray(exclusions, dtype=np.float64).reshape(-1, 3)
    pos = np.zeros((n_atoms, 3))
    # start away from the exclusion spheres
    for _ in range(1000):
        p0 = rng.normal(size=3)
        p0 *= rng.uniform(0, 0.5 * r_conf) / np.linalg.norm(p0)
        if excl.shape[0] == 0 or np.min(np.linalg.norm(excl - p0, axis=1)) > excl_radius:
            break
    pos[0] = p0
    i, rejects = 1, 0
    while i < n_atoms:
        # a plain confined walk hugs the wall and leaves the middle of the sphere almost empty (a porous body
        # whose holes open to the outside); so several candidate steps are drawn and the admissible one with
        # the fewest atoms within 4.5 A is taken, which fills the sphere evenly like a folded chain
        d = rng.normal(size=(n_candidates, 3))
        cand = pos[i - 1] + step * d / np.linalg.norm(d, axis=1, keepdims=True)
        d2 = np.sum((cand[:, None, :] - pos[None, :i, :]) ** 2, axis=2)        # [cand, placed atoms]
        ok = np.linalg.norm(cand, axis=1) <= r_conf
        if i > 1:
            ok &= np.min(d2[:, :i - 1], axis=1) >= step * step
        if excl.shape[0]:
            ok &= np.min(np.linalg.norm(cand[:, None, :] - excl[None, :, :], axis=2), axis=1) > excl_radius
        if ok.any():
            crowd = np.sum(d2 < 4.5 * 4.5, axis=1).astype(float)
            crowd[~ok] = np.inf
            pos[i] = cand[int(np.argmin(crowd))]
            i += 1
            rejects = 0
        else:
            rejects += n_candidates
            if rejects >= 100:
                i = max(1, i - 10)
                rejects = 0
    radii = rng.uniform(1.2, 2.0, size=n_atoms)
    q = rng.uniform(-0.6, 0.6, size=n_atoms)
    q += (np.rint(q.sum()) - q.sum()) / n_atoms
    return pos, radii, q, r_conf


def _density_grid(centres, R, spacing, B, pad):
    lo = centres.min(axis=0) - R.max() - pad
    hi = centres.max(axis=0) + R.max() + pad
    n = np.ceil((hi - lo) / spacing).astype(int) + 1
    rho = np.zeros(n, dtype=np.float64)
    ax = [lo[a] + spacing * np.arange(n[a]) for a in range(3)]
    for c, Ri in zip(centres, R):
        cut = Ri * np.sqrt(1.0 + 14.0 / B)            # contribution < e^-14 beyond
        i0 = np.maximum(np.floor((c - cut - lo) / spacing).astype(int), 0)
        i1 = np.minimum(np.ceil((c + cut - lo) / spacing).astype(int) + 1, n)
        gx = (ax[0][i0[0]:i1[0]] - c[0]) ** 2
        gy = (ax[1][i0[1]:i1[1]] - c[1]) ** 2
        gz = (ax[2][i0[2]:i1[2]] - c[2]) ** 2
        d2 = gx[:, None, None] + gy[None, :, None] + gz[None, None, :]
        rho[i0[0]:i1[0], i0[1]:i1[1], i0[2]:i1[2]] += np.exp(-B * (d2 / (Ri * Ri) - 1.0))
    return rho, lo, n


# Kuhn split: for every permutation (a, b, c) of the axes the tetrahedron 0, e_a, e_a+e_b, e_a+e_b+e_c
_KUHN = []
for perm in itertools.permutations(range(3)):
    v = [np.zeros(3, dtype=int)]
    for a in perm:
        w = v[-1].copy(); w[a] += 1
        v.append(w)
    _KUHN.append(np.array(v))
_KUHN = np.array(_KUHN)          # [6 tets][4 corners][3]


def marching_tetrahedra(f, lo, spacing):
    """Isosurface f = 0 of a grid function (f > 0 inside).  Returns (vertices [nv,3], triangles [nt,3])
    oriented with the normal pointing from f > 0 to f < 0."""
    n = np.array(f.shape)
    f = np.where(f == 0.0, -1e-300, f)
    inside = f > 0
    # cubes with a sign change
    s = inside[:-1, :-1, :-1].astype(np.int8)
    tot = np.zeros_like(s)
    for dx, dy, dz in itertools.product((0, 1), repeat=3):
        tot += inside[dx:n[0] - 1 + dx, dy:n[1] - 1 + dy, dz:n[2] - 1 + dz]
    cubes = np.argwhere((tot > 0) & (tot < 8))
    stride = np.array([n[1] * n[2], n[2], 1], dtype=np.int64)
    ff = f.ravel()
    tri_a, tri_b = [], []          # endpoints (grid vertex ids) of the edges carrying the triangle corners
    orient_in, orient_out = [], []
    for tet in _KUHN:
        ids = ((cubes[:, None, :] + tet[None, :, :]) * stride[None, None, :]).sum(axis=2)   # [nc,4]
        val = ff[ids]
        ins = val > 0
        cnt = ins.sum(axis=1)
        for k in (1, 2, 3):
            sel = np.nonzero(cnt == k)[0]
            if sel.size == 0:
                continue
            I, V = ids[sel], ins[sel]
            # sort corners: inside ones first (stable), so the case analysis is uniform
            order = np.argsort(~V, axis=1, kind="stable")
            I = np.take_along_axis(I, order, axis=1)
            if k == 1:      # corner 0 inside: triangle on edges (0,1), (0,2), (0,3)
                a = np.stack([I[:, 0], I[:, 0], I[:, 0]], axis=1); b = np.stack([I[:, 1], I[:, 2], I[:, 3]], axis=1)
                tri_a.append(a); tri_b.append(b); orient_in.append(I[:, 0]); orient_out.append(I[:, 1])
            elif k == 3:    # corner 3 outside: triangle on edges (0,3), (1,3), (2,3)
                a = np.stack([I[:, 0], I[:, 1], I[:, 2]], axis=1); b = np.stack([I[:, 3], I[:, 3], I[:, 3]], axis=1)
                tri_a.append(a); tri_b.append(b); orient_in.append(I[:, 0]); orient_out.append(I[:, 3])
            else:           # corners 0, 1 inside; 2, 3 outside: quad (0,2), (0,3), (1,3), (1,2) -> two triangles
                a1 = np.stack([I[:, 0], I[:, 0], I[:, 1]], axis=1); b1 = np.stack([I[:, 2], I[:, 3], I[:, 3]], axis=1)
                a2 = np.stack([I[:, 0], I[:, 1], I[:, 1]], axis=1); b2 = np.stack([I[:, 2], I[:, 3], I[:, 2]], axis=1)
                tri_a += [a1, a2]; tri_b += [b1, b2]
                orient_in += [I[:, 0], I[:, 0]]; orient_out += [I[:, 2], I[:, 2]]
    A = np.concatenate(tri_a); Bv = np.concatenate(tri_b)
    oin = np.concatenate(orient_in); oout = np.concatenate(orient_out)
    # one vertex per grid edge (welded by construction)
    lo_id = np.minimum(A, Bv).ravel(); hi_id = np.maximum(A, Bv).ravel()
    key = lo_id * (int(n.prod()) + 1) + hi_id
    uniq, first, inv = np.unique(key, return_index=True, return_inverse=True)
    ea, eb = lo_id[first], hi_id[first]

    def coords(ids):
        return np.stack([ids // stride[0], (ids % stride[0]) // stride[1], ids % stride[1]], axis=1) * spacing + lo

    fa, fb = ff[ea], ff[eb]
    t = np.clip(fa / (fa - fb), 0.1, 0.9)
    verts = coords(ea) + t[:, None] * (coords(eb) - coords(ea))
    tris = inv.reshape(-1, 3)
    # orientation: normal must point from the inside corner to the outside corner of the tetrahedron
    nrm = np.cross(verts[tris[:, 1]] - verts[tris[:, 0]], verts[tris[:, 2]] - verts[tris[:, 0]])
    flip = np.einsum("ij,ij->i", nrm, coords(oout) - coords(oin)) < 0
    tris[flip] = tris[flip][:, [0, 2, 1]]
    return verts, tris.astype(np.int64)


def _outer_component(verts, tris):
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    nv = verts.shape[0]
    e = np.concatenate([tris[:, [0, 1]], tris[:, [1, 2]]], axis=0)
    g = coo_matrix((np.ones(len(e)), (e[:, 0], e[:, 1])), shape=(nv, nv))
    ncomp, lab = connected_components(g, directed=False)
    if ncomp > 1:
        ext = [np.ptp(verts[lab == c], axis=0).sum() if np.any(lab == c) else 0 for c in range(ncomp)]
        keep = int(np.argmax(ext))
        tris = tris[lab[tris[:, 0]] == keep]
    used = np.unique(tris)
    remap = -np.ones(nv, dtype=np.int64); remap[used] = np.arange(used.size)
    return verts[used], remap[tris]


def validate_closed_mesh(verts, tris):
    """True iff every directed edge occurs exactly once and its reverse exactly once (closed, manifold,
    consistently oriented) and no triangle is degenerate."""
    t = np.asarray(tris, dtype=np.int64)
    e = np.concatenate([t[:, [0, 1]], t[:, [1, 2]], t[:, [2, 0]]], axis=0)
    nv = int(t.max()) + 1
    k = e[:, 0] * nv + e[:, 1]
    kr = e[:, 1] * nv + e[:, 0]
    if np.unique(k).size != k.size:
        return False
    if not np.array_equal(np.sort(k), np.sort(kr)):
        return False
    v = np.asarray(verts)
    area = 0.5 * np.linalg.norm(np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]]), axis=1)
    return bool(np.all(area > 0))


def density_surface(centres, radii, spacing, probe=1.4, B=2.3, max_tries=4):
    """Closed outward-oriented triangulation of {rho = 1}.  If the grid happens to produce a non-manifold
    edge (isosurface through a grid vertex), the grid is shifted by a fraction of the spacing and redone."""
    R = np.asarray(radii) + probe
    pad = 2 * spacing
    for attempt in range(max_tries + 4):
        rho, lo, n = _density_grid(np.asarray(centres) + 0.37 * spacing * attempt, R, spacing, B, pad=pad)
        # where many atoms overlap the tails add up and the isosurface lies outside every R_i: the grid must
        # contain it with a margin, otherwise the mesh would be cut open at the box
        edge_max = max(rho[:2].max(), rho[-2:].max(), rho[:, :2].max(), rho[:, -2:].max(), rho[:, :, :2].max(),
                       rho[:, :, -2:].max())
        if edge_max >= 1.0:
            pad += 0.5 * R.max()
            continue
        v, t = marching_tetrahedra(rho - 1.0, lo, spacing)
        v = v - 0.37 * spacing * attempt
        v, t = _outer_component(v, t)
        if validate_closed_mesh(v, t):
            return np.ascontiguousarray(v), np.ascontiguousarray(t.astype(np.int32))
    raise RuntimeError("density_surface: could not produce a closed manifold mesh")


def protein_problem(n_atoms=1000, spacing=0.75, seed=13094020, eps_in=4.0, eps_out=80.0, kappa=0.125):
    """BASELINE.json config 2: single dielectric interface around a synthetic protein.  `spacing` sets the
    triangle count (the config's '~40 k triangles' governs the work)."""
    pos, rad, q, _ = saw_molecule(n_atoms, seed)
    v, t = density_surface(pos, rad, spacing)
    return Problem([Surface(v, t, 0, 1)], [eps_in, eps_out], [0.0, kappa], pos, q, np.zeros(n_atoms, dtype=np.int32),
                   name=f"protein_{n_atoms}", meta=dict(n_atoms=n_atoms, spacing=spacing))


def _cavity_centres(rng, n_atoms, n_cav, sep=12.0, wall=8.0):
    r_conf = (n_atoms * 20.0 * 3.0 / (4.0 * np.pi)) ** (1.0 / 3.0)
    pts = []
    for it in range(200000):
        if it % 500 == 499:
            pts = []                                   # stuck: start over
        p = rng.normal(size=3)
        p *= rng.uniform(0, max(r_conf - wall, 1.0)) / np.linalg.norm(p)
        if all(np.linalg.norm(p - c) >= sep for c in pts):
            pts.append(p)
        if len(pts) == n_cav:
            return np.array(pts)
    raise RuntimeError("no room for the cavities")


def multisurface_problem(n_atoms=3000, spacing=0.8, seed=13094021, n_cavities=2, cavity_level=2, stern=2.0,
                         eps_in=4.0, eps_out=80.0, kappa=0.125, cav_sep=12.0, cav_wall=8.0):
    """BASELINE.json config 3: SES + solvent-filled spherical cavities (R = 3 A, eps_out, kappa = 0, normals
    pointing into the protein) + Stern surface (density inflated by a further `stern` A; kappa = 0 inside it).
    Regions: 0 protein, 1 Stern layer, 2 solvent, 3 cavities."""
    rng = np.random.default_rng(seed)
    for attempt in range(50):
        cav = _cavity_centres(rng, n_atoms, n_cavities, cav_sep, cav_wall) if n_cavities else np.zeros((0, 3))
        pos, rad, q, _ = saw_molecule(n_atoms, seed + 1000 + attempt, exclusions=cav, excl_radius=5.0)
        v, t = density_surface(pos, rad, spacing)
        # every cavity must sit strictly inside the dielectric interface; otherwise redraw
        if all(np.min(np.linalg.norm(v - c, axis=1)) >= 3.0 + 1.0 for c in cav):
            break
    else:
        raise RuntimeError("could not place the cavities inside the dielectric interface")
    surfaces = [Surface(v, t, 0, 1)]
    for c in cav:
        vc, tc = icosphere(cavity_level, 3.0, center=c)
        surfaces.append(Surface(vc, tc, 3, 0))
    vs, ts = density_surface(pos, rad, spacing, probe=1.4 + stern)
    surfaces.append(Surface(vs, ts, 1, 2))
    return Problem(surfaces, [eps_in, eps_out, eps_out, eps_out], [0.0, 0.0, kappa, 0.0], pos, q,
                   np.zeros(n_atoms, dtype=np.int32), name=f"multisurface_{n_atoms}",
                   meta=dict(n_atoms=n_atoms, spacing=spacing, cavities=cav.tolist()))


def binding_problems(n_receptor=5000, n_ligand=500, spacing=0.8, seed=13094022, separation=3.0, stern=2.0,
                     eps_in=4.0, eps_out=80.0, kappa=0.125, only=("complex", "receptor", "ligand")):
    """BASELINE.json config 4: (complex, receptor, ligand), each with a Stern layer (eq. 7).
    The ligand is moved along a seeded direction until the two dielectric interfaces are `separation` apart;
    the complex has both bodies as one surface (same region pair) and ONE Stern surface from the union
    density (the two 2 A shells overlap at 3 A separation).  Regions: 0 protein, 1 Stern layer, 2 solvent.
    `only` selects which of the three problems are built (the others are returned as None): each needs its own
    Stern surface, the most expensive piece of the generation."""
    rng = np.random.default_rng(seed)
    pr, rr, qr, rc_r = saw_molecule(n_receptor, seed + 1)
    pl, rl, ql, rc_l = saw_molecule(n_ligand, seed + 2)
    vr, tr = density_surface(pr, rr, spacing)
    vl, tl = density_surface(pl, rl, spacing)
    d = rng.normal(size=3); d /= np.linalg.norm(d)
    from scipy.spatial import cKDTree
    tree = cKDTree(vr)
    lo, hi = 0.0, rc_r + rc_l + 20.0
    for _ in range(40):                      # bisection on the offset along d
        mid = 0.5 * (lo + hi)
        # "is any ligand vertex closer than `separation` to the receptor surface": the bounded query prunes
        # almost every node of the tree (the unbounded nearest-neighbour query took 2.5 s per step at full size)
        near = np.isfinite(tree.query(vl + mid * d, distance_upper_bound=separation, workers=-1)[0]).any()
        inside = np.min(np.linalg.norm((pl + mid * d)[:, None, :] - pr[None, ::10, :], axis=2)) < 3.0
        if near or inside:
            lo = mid
        else:
            hi = mid
    off = hi * d
    pl2, vl2 = pl + off, vl + off
    eps = [eps_in, eps_out, eps_out]
    kap = [0.0, 0.0, kappa]

    def make(bodies, atoms, radii, charges, name):
        if name not in only:
            return None
        surf = [Surface(v, t, 0, 1) for v, t in bodies]
        vs, ts = density_surface(atoms, radii, spacing, probe=1.4 + stern)
        surf.append(Surface(vs, ts, 1, 2))
        return Problem(surf, eps, kap, atoms, charges, np.zeros(len(charges), dtype=np.int32), name=name,
                       meta=dict(spacing=spacing))

    cplx = make([(vr, tr), (vl2, tl)], np.concatenate([pr, pl2]), np.concatenate([rr, rl]),
                np.concatenate([qr, ql]), "complex")
    rec = make([(vr, tr)], pr, rr, qr, "receptor")
    lig = make([(vl2, tl)], pl2, rl, ql, "ligand")
    return cplx, rec, lig
