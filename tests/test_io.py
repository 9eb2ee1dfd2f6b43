"""Readers of paper_1309_4018_b200/io.py (PQR charges, MSMS .vert/.face surfaces) on files written from the
synthetic workloads: round trip, header handling, orientation repair, assembly of a multi-surface Problem."""
import os

import numpy as np
import pytest

import workloads as W
from paper_1309_4018_b200 import io as pio


def test_pqr_round_trip(tmp_path):
    rng = np.random.default_rng(5)
    xyz = rng.uniform(-20, 20, (37, 3)); q = rng.uniform(-1, 1, 37); r = rng.uniform(1, 2, 37)
    p = os.path.join(tmp_path, "m.pqr")
    pio.write_pqr(p, xyz, q, r)
    with open(p, "a") as f:
        f.write("REMARK trailing\nHETATM 9999 ZN    ZN B 901      1.000   2.000   3.000  2.0000  0.7400\nEND\n")
    c = pio.read_pqr(p)
    assert c["xyz"].shape == (38, 3)
    assert np.abs(c["xyz"][:37] - xyz).max() < 6e-4 and np.abs(c["q"][:37] - q).max() < 6e-5 and np.abs(c["radius"][:37] - r).max() < 6e-5
    assert np.allclose(c["xyz"][37], [1, 2, 3]) and c["q"][37] == 2.0
    with open(p, "w") as f:
        f.write("REMARK nothing here\n")
    with pytest.raises(ValueError):
        pio.read_pqr(p)


@pytest.mark.parametrize("header", [True, False])
def test_msms_round_trip_and_orientation(tmp_path, header):
    v, t = W.icosphere(2, 3.0)
    stem = os.path.join(tmp_path, "s")
    pio.write_msms(stem, v, t, header=header)
    v2, t2 = pio.read_msms(stem)
    assert v2.shape == v.shape and np.abs(v2 - v).max() < 6e-4 and np.array_equal(t2, t)
    assert pio.signed_volume(v2, t2) > 0
    # inward-oriented file: repaired by orient="auto", kept by "keep"
    pio.write_msms(stem, v, t[:, [0, 2, 1]], header=header)
    assert np.array_equal(pio.read_msms(stem)[1], t)
    assert pio.signed_volume(*pio.read_msms(stem, orient="keep")) < 0
    W.validate_closed_mesh(*pio.read_msms(stem))
    with open(stem + ".face", "a") as f:
        f.write("%6d %6d %6d  1  1\n" % (1, 2, len(v) + 5))
    with pytest.raises(ValueError):
        pio.read_msms(stem)


def test_problem_from_files_matches_the_generated_one(tmp_path, oracle_mod):
    """Stern + cavity problem written to files and read back: same region graph, same oracle operator."""
    ref = W.cavity_sphere_problem(1)
    d = str(tmp_path)
    pio.write_pqr(os.path.join(d, "m.pqr"), ref.charge_xyz, ref.charge_q, np.full(len(ref.charge_q), 1.5))
    pio.write_msms(os.path.join(d, "ses"), ref.surfaces[0].vertices, ref.surfaces[0].triangles)
    pio.write_msms(os.path.join(d, "cav"), ref.surfaces[1].vertices, ref.surfaces[1].triangles)
    prob = pio.problem_from_files(os.path.join(d, "m.pqr"), os.path.join(d, "ses"), cavities=[os.path.join(d, "cav")])
    assert prob.n_regions == 3 and [(s.region_in, s.region_out) for s in prob.surfaces] == [(0, 1), (2, 0)]
    assert list(prob.eps) == [4.0, 80.0, 80.0] and list(prob.kappa) == [0.0, 0.125, 0.0]
    o1, o2 = oracle_mod.Oracle(ref), oracle_mod.Oracle(prob)
    x = np.random.default_rng(2).normal(size=o1.n)
    y1, y2 = o1.matvec(x), o2.matvec(x)
    assert np.linalg.norm(y1 - y2) / np.linalg.norm(y1) < 2e-3      # vertices rounded to 1e-3 A in the files
    # with a Stern surface: regions protein / Stern / solvent
    st = W.stern_sphere_problem(1)
    pio.write_msms(os.path.join(d, "stern"), st.surfaces[1].vertices, st.surfaces[1].triangles)
    pio.write_msms(os.path.join(d, "body"), st.surfaces[0].vertices, st.surfaces[0].triangles)
    pio.write_pqr(os.path.join(d, "c.pqr"), st.charge_xyz, st.charge_q, np.ones(len(st.charge_q)))
    p2 = pio.problem_from_files(os.path.join(d, "c.pqr"), os.path.join(d, "body"), stern=os.path.join(d, "stern"))
    assert [(s.region_in, s.region_out) for s in p2.surfaces] == [(0, 1), (1, 2)] and list(p2.kappa) == [0.0, 0.0, 0.125]
