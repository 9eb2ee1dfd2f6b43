"""Readers for real-molecule input (the paper's inputs: atomic charges
and radii from pdb2pqr, triangulated solvent-excluded surfaces from MSMS).  No such files are in this
container; the readers are exercised by tests/test_io.py on files written from the synthetic workloads.

    charges = read_pqr("1abc.pqr")                      # dict(xyz [n,3] A, q [n] e, radius [n] A)
    verts, tris = read_msms("1abc")                     # 1abc.vert + 1abc.face
    prob = problem_from_files("1abc.pqr", "1abc", stern="1abc_stern", cavities=["1abc_cav0"])
    h = Handle.from_problem(prob, K=4, P=6, theta=0.5)

Formats.  PQR: whitespace-separated records ATOM / HETATM whose last five fields are x y z charge radius (the
columns before them vary between writers and are ignored).  MSMS .vert: lines "x y z nx ny nz ..." (only the
first three fields are used); .face: lines "i j k ..." with 1-based vertex indices.  Comment lines ('#') and the
four-field count line MSMS puts after them are skipped; files stripped to bare "x y z" / "i j k" rows work too.
Orientation: the library wants triangles counter-clockwise seen from region_out, i.e. normals pointing from
region_in to region_out (include/pygbe.h); `orient="auto"` flips every triangle of a closed
surface whose signed volume is negative, `orient="keep"` trusts the file, `orient="flip"` swaps.
"""
import numpy as np

from workloads.problem import Problem, Surface


def read_pqr(path):
    xyz, q, rad = [], [], []
    with open(path) as f:
        for line in f:
            rec = line[:6].strip().upper()
            if rec not in ("ATOM", "HETATM"):
                continue
            parts = line.split()
            if len(parts) < 6:
                raise ValueError(f"{path}: short ATOM record: {line!r}")
            try:
                x, y, z, c, r = (float(v) for v in parts[-5:])
            except ValueError as e:
                raise ValueError(f"{path}: cannot parse the last five fields of {line!r}") from e
            xyz.append((x, y, z)); q.append(c); rad.append(r)
    if not xyz:
        raise ValueError(f"{path}: no ATOM / HETATM records")
    return dict(xyz=np.asarray(xyz, float), q=np.asarray(q, float), radius=np.asarray(rad, float))


def _records(path):
    """Whitespace-split data lines of an MSMS file: '#' comments dropped, and the count line MSMS writes after them
    ("n n_spheres density probe_radius": four fields, unlike the records that follow) dropped as well."""
    rows = []
    with open(path) as f:
        for line in f:
            s = line.strip()
            if s and not s.startswith("#"):
                rows.append(s.split())
    if len(rows) >= 2 and len(rows[0]) == 4 and len(rows[1]) != 4:
        rows = rows[1:]
    if not rows:
        raise ValueError(f"{path}: no records")
    return rows


def read_msms(stem, orient="auto"):
    """Read `stem`.vert and `stem`.face; returns (vertices [n,3] float64, triangles [m,3] int32, 0-based)."""
    try:
        verts = np.asarray([[float(v) for v in r[:3]] for r in _records(stem + ".vert")], float)
        tris = np.asarray([[int(v) for v in r[:3]] for r in _records(stem + ".face")], np.int64) - 1
    except (ValueError, IndexError) as e:
        raise ValueError(f"{stem}.vert / .face: malformed record ({e})") from e
    if tris.min() < 0 or tris.max() >= len(verts):
        raise ValueError(f"{stem}.face: vertex indices outside 1..{len(verts)}")
    tris = orient_triangles(verts, tris.astype(np.int32), orient)
    return np.ascontiguousarray(verts), np.ascontiguousarray(tris)


def signed_volume(verts, tris):
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    return float(np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0)


def orient_triangles(verts, tris, orient="auto"):
    if orient == "keep":
        return tris
    if orient == "flip" or (orient == "auto" and signed_volume(verts, tris) < 0):
        return np.ascontiguousarray(tris[:, [0, 2, 1]])
    if orient not in ("auto", "flip"):
        raise ValueError(f"orient = {orient!r}")
    return tris


def write_pqr(path, xyz, q, radius):
    with open(path, "w") as f:
        for i, (p, c, r) in enumerate(zip(xyz, q, radius)):
            f.write("ATOM  %5d  C   MOL A%4d    %8.3f%8.3f%8.3f %8.4f %7.4f\n" % (i + 1, 1 + i // 10, p[0], p[1], p[2], c, r))


def write_msms(stem, verts, tris, header=True):
    """Write a surface the way MSMS does (3 header lines, unit normals, 1-based faces)."""
    verts = np.asarray(verts, float); tris = np.asarray(tris)
    n = np.zeros_like(verts)
    fn = np.cross(verts[tris[:, 1]] - verts[tris[:, 0]], verts[tris[:, 2]] - verts[tris[:, 0]])
    for k in range(3):
        np.add.at(n, tris[:, k], fn)
    n /= np.maximum(np.linalg.norm(n, axis=1, keepdims=True), 1e-300)
    with open(stem + ".vert", "w") as f:
        if header:
            f.write("# MSMS solvent excluded surface vertices for %s\n#vertex #sphere density probe_r\n" % stem)
            f.write("%7d %7d  %.2f  %.2f\n" % (len(verts), 0, 1.0, 1.4))
        for p, m in zip(verts, n):
            f.write("%9.3f %9.3f %9.3f %9.3f %9.3f %9.3f %7d %7d %2d\n" % (p[0], p[1], p[2], m[0], m[1], m[2], 0, 1, 2))
    with open(stem + ".face", "w") as f:
        if header:
            f.write("# MSMS solvent excluded surface faces for %s\n#faces  #sphere density probe_r\n" % stem)
            f.write("%7d %7d  %.2f  %.2f\n" % (len(tris), 0, 1.0, 1.4))
        for t in tris:
            f.write("%6d %6d %6d %2d %6d\n" % (t[0] + 1, t[1] + 1, t[2] + 1, 1, 1))


def problem_from_files(pqr, mesh, stern=None, cavities=(), eps_in=4.0, eps_out=80.0, kappa=0.125, orient="auto", name=""):
    """Molecule = dielectric body (region 0: eps_in, charges of `pqr`) bounded by the surface `mesh`, optional
    solvent-filled cavities inside it (one region, eps_out, no salt: PAPER.md:131), optional Stern surface `stern`
    around it (ion-exclusion layer, eps_out, no salt: PAPER.md:127), solvent outside (eps_out, kappa)."""
    ch = read_pqr(pqr)
    v, t = read_msms(mesh, orient)
    surfaces, eps, kap = [], [eps_in], [0.0]
    if stern is not None:
        eps += [eps_out, eps_out]; kap += [0.0, kappa]         # 1 Stern layer, 2 solvent
        surfaces.append(Surface(v, t, 0, 1))
        vs, ts = read_msms(stern, orient)
        surfaces.append(Surface(vs, ts, 1, 2))
    else:
        eps += [eps_out]; kap += [kappa]                       # 1 solvent
        surfaces.append(Surface(v, t, 0, 1))
    if cavities:
        rc = len(eps)
        eps.append(eps_out); kap.append(0.0)
        for c in cavities:
            vc, tc = read_msms(c, orient)                      # oriented outward from the cavity = into the protein
            surfaces.append(Surface(vc, tc, rc, 0))
    return Problem(surfaces, eps, kap, ch["xyz"], ch["q"], np.zeros(len(ch["q"]), np.int32), name=name or str(mesh),
                   meta=dict(radius=ch["radius"]))
