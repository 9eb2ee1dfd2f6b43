"""CPU tests of the input generators (geometry only) and of the oracle on the molecule-like inputs."""
import numpy as np
import pytest

import workloads as W


def _signed_volume(v, t):
    n = np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]])
    return float(np.einsum("ij,ij->i", v[t[:, 0]], n).sum() / 6.0), n


@pytest.mark.parametrize("level,ntri", [(0, 20), (1, 80), (3, 1280)])
def test_icosphere(level, ntri):
    v, t = W.icosphere(level, 2.5, center=(1.0, -2.0, 0.5))
    assert t.shape == (ntri, 3) and W.validate_closed_mesh(v, t)
    assert np.allclose(np.linalg.norm(v - np.array([1.0, -2.0, 0.5]), axis=1), 2.5)
    vol, n = _signed_volume(v - np.array([1.0, -2.0, 0.5]), t)
    assert vol > 0 and np.abs(n.sum(axis=0)).max() < 1e-12       # outward, closed: sum A n = 0
    vi, ti = W.icosphere(level, 2.5, inward=True)
    assert _signed_volume(vi, ti)[0] < 0


def test_saw_molecule_recipe():
    pos, rad, q, rc = W.saw_molecule(300, 7)
    assert pos.shape == (300, 3) and np.all(np.linalg.norm(pos, axis=1) <= rc + 1e-12)
    assert np.allclose(np.linalg.norm(np.diff(pos, axis=0), axis=1), 1.5)
    d = np.linalg.norm(pos[:, None] - pos[None], axis=2)
    iu = np.triu_indices(300, 2)                                   # non-adjacent pairs
    assert d[iu].min() >= 1.5 - 1e-12
    assert rad.min() >= 1.2 and rad.max() <= 2.0
    assert abs(q.sum() - round(q.sum())) < 1e-12
    pos2, _, _, _ = W.saw_molecule(300, 7)
    assert np.array_equal(pos, pos2)                               # seeded


def test_density_surface_is_closed_and_oriented():
    pos, rad, q, rc = W.saw_molecule(150, 3)
    v, t = W.density_surface(pos, rad, 1.0)
    assert W.validate_closed_mesh(v, t)
    vol, n = _signed_volume(v, t)
    assert vol > 150 * 20.0                                        # encloses the atoms, outward oriented
    assert np.abs(n.sum(axis=0)).max() < 1e-9
    # every atom centre is inside: winding number via the solid angle identity (sum of A n.(c - x)/|c - x|^3)
    c = v[t].mean(axis=1); area_n = 0.5 * n
    for x in pos[::30]:
        d = c - x
        w = np.sum(np.einsum("ij,ij->i", area_n, d) / np.linalg.norm(d, axis=1) ** 3) / (4 * np.pi)
        assert abs(w - 1.0) < 0.05
    # a sphere is reproduced: one atom -> radius where exp(-B(r^2/R^2 - 1)) = 1, i.e. r = R
    v1, t1 = W.density_surface(np.zeros((1, 3)), np.array([1.6]), 0.25)
    assert abs(np.linalg.norm(v1, axis=1).mean() - 3.0) < 0.02


def test_problem_builders_regions():
    p = W.multisurface_problem(n_atoms=300, spacing=1.4, cavity_level=1, cav_sep=8.0, cav_wall=6.5)
    assert [(s.region_in, s.region_out) for s in p.surfaces] == [(0, 1), (3, 0), (3, 0), (1, 2)]
    assert list(p.kappa) == [0.0, 0.0, 0.125, 0.0] and list(p.eps) == [4.0, 80.0, 80.0, 80.0]
    for s in p.surfaces:
        assert W.validate_closed_mesh(s.vertices, s.triangles)
    ses, stern = p.surfaces[0], p.surfaces[-1]
    assert _signed_volume(stern.vertices, stern.triangles)[0] > _signed_volume(ses.vertices, ses.triangles)[0]
    for cav in p.surfaces[1:3]:                                    # cavity normals point into the protein
        c = cav.vertices.mean(axis=0)
        assert _signed_volume(cav.vertices - c, cav.triangles)[0] > 0
        assert np.min(np.linalg.norm(p.charge_xyz - c, axis=1)) > 3.0
    cplx, rec, lig = W.binding_problems(n_receptor=200, n_ligand=50, spacing=1.4)
    assert len(cplx.surfaces) == 3 and len(rec.surfaces) == 2 and len(lig.surfaces) == 2
    assert len(cplx.charge_q) == len(rec.charge_q) + len(lig.charge_q)
    # rigid geometry: the complex's bodies are the receptor's and the ligand's
    assert np.array_equal(cplx.surfaces[0].vertices, rec.surfaces[0].vertices)
    assert np.array_equal(cplx.surfaces[1].vertices, lig.surfaces[0].vertices)
    from scipy.spatial import cKDTree
    gap = cKDTree(cplx.surfaces[0].vertices).query(cplx.surfaces[1].vertices)[0].min()
    assert 2.9 < gap < 3.6


def test_oracle_on_a_molecule_gauss_identity(oracle_mod):
    """Gauss identity on a marching-tetrahedra surface (slivers included): phi = 1 gives interior rows
    1/2 + sum_j K_L,ij ~ 0; checks orientation and near-field treatment on irregular panels."""
    p = W.protein_problem(60, spacing=1.5, seed=5)
    o = oracle_mod.Oracle(p)
    N = o.npan
    x = np.concatenate([np.ones(N), np.zeros(N)])
    y = o.matvec(x)
    # slivers next to a target defeat the centroid-distance near-field rule locally (max), not globally (median)
    assert np.median(np.abs(y[:N])) < 2e-3 and np.max(np.abs(y[:N])) < 0.3


def test_cache_is_shared_between_processes(tmp_path, monkeypatch):
    """workloads.cached: two processes asking for the same problem at once build it once (lock file); the stored
    .npz reproduces the problem exactly."""
    import subprocess
    import sys
    import textwrap
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, time
        sys.path.insert(0, {root!r})
        os.environ["PYGBE_WORKLOAD_CACHE"] = {str(tmp_path / "cache")!r}
        import workloads as W
        def build():
            open(os.path.join({str(tmp_path)!r}, "built_%d" % os.getpid()), "w").close()
            time.sleep(1.0)
            return W.protein_problem(40, spacing=1.6, seed=3)
        p = W.cached("t_protein_40", build)
        print(p.n_panels, float(p.surfaces[0].vertices.sum()))
    """))
    procs = [subprocess.Popen([sys.executable, str(script)], stdout=subprocess.PIPE, text=True) for _ in range(3)]
    outs = [p.communicate(timeout=300)[0].strip() for p in procs]
    assert all(p.returncode == 0 for p in procs) and len(set(outs)) == 1
    assert len([f for f in os.listdir(tmp_path) if f.startswith("built_")]) == 1
    assert not [f for f in os.listdir(tmp_path / "cache") if f.endswith(".lock")]
    monkeypatch.setenv("PYGBE_WORKLOAD_CACHE", str(tmp_path / "cache"))
    p = W.cached("t_protein_40", lambda: (_ for _ in ()).throw(AssertionError("must come from the cache")))
    q = W.protein_problem(40, spacing=1.6, seed=3)
    assert np.array_equal(p.surfaces[0].vertices, q.surfaces[0].vertices) and np.array_equal(p.charge_q, q.charge_q)
    assert np.array_equal(p.surfaces[0].triangles, q.surfaces[0].triangles) and list(p.eps) == list(q.eps)
