"""Sphere workloads: icosphere meshes and the Born / Kirkwood / concentric test problems.

Recipe A20: 12-vertex icosahedron (0,+-1,+-phi) cyclic permutations, normalised; 4-way
midpoint split with midpoints projected to the sphere at every level; outward CCW orientation.
Level 3 = 1280, level 5 = 20480 triangles (BASELINE.json configs 0 and 1; the paper's sphere test is
PAPER.md:217, section 3.1).
"""
import numpy as np
from .problem import Problem, Surface


def icosphere(level: int, radius: float = 1.0, center=(0.0, 0.0, 0.0), inward: bool = False):
    """Return (vertices [nv,3] f64, triangles [nt,3] i32) of a subdivided icosahedron.
    inward=True flips the winding (normals point to the sphere centre)."""
    g = (1.0 + np.sqrt(5.0)) / 2.0
    v = []
    for s1 in (1.0, -1.0):
        for s2 in (1.0, -1.0):
            v.append((0.0, s1 * 1.0, s2 * g))
            v.append((s1 * 1.0, s2 * g, 0.0))
            v.append((s2 * g, 0.0, s1 * 1.0))
    v = np.array(v, dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    # faces = all vertex triples that are mutually nearest neighbours (edge length 2/|v|)
    d = np.linalg.norm(v[:, None, :] - v[None, :, :], axis=2)
    edge = d[d > 1e-12].min()
    adj = np.abs(d - edge) < 1e-9
    faces = []
    for a in range(12):
        for b in range(a + 1, 12):
            if not adj[a, b]:
                continue
            for c in range(b + 1, 12):
                if adj[a, c] and adj[b, c]:
                    faces.append((a, b, c))
    f = np.array(faces, dtype=np.int64)
    assert f.shape[0] == 20
    # orient outward
    nrm = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
    cen = v[f].mean(axis=1)
    flip = np.einsum("ij,ij->i", nrm, cen) < 0
    f[flip] = f[flip][:, [0, 2, 1]]
    for _ in range(level):
        nv = v.shape[0]
        e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
        es = np.sort(e, axis=1)
        key = es[:, 0] * nv + es[:, 1]
        uniq, inv = np.unique(key, return_inverse=True)
        a, b = uniq // nv, uniq % nv
        mid = v[a] + v[b]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        v = np.concatenate([v, mid], axis=0)
        nt = f.shape[0]
        m01 = nv + inv[0:nt]
        m12 = nv + inv[nt:2 * nt]
        m20 = nv + inv[2 * nt:3 * nt]
        f = np.concatenate([
            np.stack([f[:, 0], m01, m20], axis=1),
            np.stack([f[:, 1], m12, m01], axis=1),
            np.stack([f[:, 2], m20, m12], axis=1),
            np.stack([m01, m12, m20], axis=1),
        ], axis=0)
    if inward:
        f = f[:, [0, 2, 1]]
    verts = v * radius + np.asarray(center, dtype=np.float64)[None, :]
    return np.ascontiguousarray(verts), np.ascontiguousarray(f.astype(np.int32))


def born_problem(level=3, radius=4.0, eps_in=4.0, eps_out=80.0, kappa=0.125, q=1.0):
    """BASELINE.json config 0: centred charge in a sphere (salt added per config)."""
    v, t = icosphere(level, radius)
    return Problem([Surface(v, t, 0, 1)], [eps_in, eps_out], [0.0, kappa],
                   [[0.0, 0.0, 0.0]], [q], [0], name=f"born_l{level}",
                   meta=dict(radius=radius, level=level))


# positions drawn with numpy.random.default_rng(13094019): rng.uniform(-7,7,3) rejected until |p|<=7
KIRKWOOD_POS = np.array([
    [-2.276048729836991, -2.47004431717631, -1.359221450319754],
    [-4.286126885504283, -3.10957091901824, -0.573994653139292],
    [1.590316718189031, -0.102582285057529, -3.101315615703335],
])
KIRKWOOD_Q = np.array([1.0, -1.0, 0.5])


def kirkwood_problem(level=5, radius=10.0, eps_in=4.0, eps_out=80.0, kappa=0.125):
    """BASELINE.json config 1: three off-centre charges in a 10 A sphere."""
    v, t = icosphere(level, radius)
    return Problem([Surface(v, t, 0, 1)], [eps_in, eps_out], [0.0, kappa],
                   KIRKWOOD_POS.copy(), KIRKWOOD_Q.copy(), [0, 0, 0], name=f"kirkwood_l{level}",
                   meta=dict(radius=radius, level=level))


def stern_sphere_problem(level=2, r_in=4.0, r_stern=6.0, eps_in=4.0, eps_out=80.0, kappa=0.125, q=1.0):
    """Concentric dielectric sphere + Stern sphere: regions 0 protein, 1 Stern layer (eps_out, 0),
    2 solvent (eps_out, kappa).  Pins the multi-surface rule."""
    v0, t0 = icosphere(level, r_in)
    v1, t1 = icosphere(level, r_stern)
    return Problem([Surface(v0, t0, 0, 1), Surface(v1, t1, 1, 2)],
                   [eps_in, eps_out, eps_out], [0.0, 0.0, kappa],
                   [[0.0, 0.0, 0.0]], [q], [0], name=f"stern_l{level}",
                   meta=dict(r_in=r_in, r_stern=r_stern, level=level))


def cavity_sphere_problem(level=2, r_cav=2.0, r_out=8.0, r_charge=5.0, eps_in=4.0, eps_out=80.0,
                          kappa=0.125, q=1.0, eps_cav=None):
    """Solvent-filled concentric cavity inside a protein shell; charge on the z axis in the shell.
    Regions: 0 protein shell, 1 solvent (eps_out, kappa), 2 cavity (eps_cav, 0).  The cavity surface
    has region_in = cavity, region_out = protein, i.e. its normal points into the protein."""
    if eps_cav is None:
        eps_cav = eps_out
    vo, to = icosphere(level, r_out)
    vc, tc = icosphere(level, r_cav)
    return Problem([Surface(vo, to, 0, 1), Surface(vc, tc, 2, 0)],
                   [eps_in, eps_out, eps_cav], [0.0, kappa, 0.0],
                   [[0.0, 0.0, r_charge]], [q], [0], name=f"cavity_l{level}",
                   meta=dict(r_cav=r_cav, r_out=r_out, r_charge=r_charge, level=level))


def nested_sphere_problem(level=2, radii=(1.5, 2.5, 8.0, 10.0), r_charge=5.0, eps_in=4.0, eps_out=80.0,
                          kappa_cav=0.5, kappa=0.125, q=1.0):
    """An ion-bearing cavity with its own Stern layer inside a protein shell with an outer Stern layer
    ("cavities ... large enough to contain ions ... an interior Stern layer"), all concentric:
        r < radii[0]            region 4: cavity solvent with salt (eps_out, kappa_cav)
        radii[0] < r < radii[1] region 3: cavity Stern layer (eps_out, 0)
        radii[1] < r < radii[2] region 0: protein (eps_in, 0), charge on the z axis at r_charge
        radii[2] < r < radii[3] region 1: outer Stern layer (eps_out, 0)
        r > radii[3]            region 2: solvent with salt (eps_out, kappa)
    Four surfaces, every normal pointing away from the centre (region_in = the inner side)."""
    a0, a1, a2, a3 = radii
    s0 = Surface(*icosphere(level, a0), 4, 3)
    s1 = Surface(*icosphere(level, a1), 3, 0)
    s2 = Surface(*icosphere(level, a2), 0, 1)
    s3 = Surface(*icosphere(level, a3), 1, 2)
    return Problem([s0, s1, s2, s3], [eps_in, eps_out, eps_out, eps_out, eps_out], [0.0, 0.0, kappa, 0.0, kappa_cav],
                   [[0.0, 0.0, r_charge]], [q], [0], name=f"nested_l{level}",
                   meta=dict(radii=tuple(radii), r_charge=r_charge, level=level))
