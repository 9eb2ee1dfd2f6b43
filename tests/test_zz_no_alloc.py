"""The entry point that allocates nothing (pygbe_coulomb_energy_noalloc, csrc/noalloc.cu) against the existing path
(pygbe_energy's Coulomb term on a handle, eq. 8).  Collected last on purpose (file name): the suite
runs with pytest -x, and a failure here must not hide any other test."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_COULOMB = 1e-11          # relative; the bar of the Coulomb comparisons in test_gpu_parity.py (summation order only)


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1309_4018_b200 as pg
    pg.lib()
    return pg, torch


def _charges(seed, n, radius=4.0):
    rng = np.random.default_rng(seed)
    p = rng.normal(size=(n, 3))
    p *= radius * np.cbrt(rng.uniform(0, 1, size=(n, 1))) / np.linalg.norm(p, axis=1, keepdims=True)
    return np.ascontiguousarray(p), rng.uniform(-0.6, 0.6, size=n)


def _existing_path(pg, torch, xyz, q, eps_in):
    """E_coul of pygbe_energy on a handle that holds these charges inside a sphere of permittivity eps_in."""
    v, t = W.icosphere(1, 6.0)
    prob = W.Problem([W.Surface(v, t, 0, 1)], [eps_in, 80.0], [0.0, 0.125], xyz, q, np.zeros(len(q), dtype=np.int32))
    h = pg.Handle.from_problem(prob, K=4, theta=0.0)
    x = torch.zeros(h.n, dtype=torch.float64, device="cuda")
    ec = h.energy(x)[1]
    h.close()
    return ec


def test_no_alloc_coulomb_matches_the_handle_path_twice_in_a_row(env):
    pg, torch = env
    eps_in = 4.0
    sets = [_charges(11, 3000), _charges(12, 1200)]          # the second call uses fewer records than the first left behind
    want = [_existing_path(pg, torch, xyz, q, eps_in) for xyz, q in sets]
    assert all(abs(w) > 1.0 for w in want)
    dev = [(torch.tensor(xyz, device="cuda"), torch.tensor(q, device="cuda")) for xyz, q in sets]
    outs = [torch.full((1,), 123.0, dtype=torch.float64, device="cuda") for _ in sets]
    pg.noalloc_setup(0)
    pg.coulomb_energy_noalloc(dev[0][0], dev[0][1], eps_in, outs[0])      # first use also loads the kernels
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row, no synchronisation in between (same stream: ordered)
    for (xyz, q), out in zip(dev, outs):
        out.fill_(123.0)
        pg.coulomb_energy_noalloc(xyz, q, eps_in, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0             # nothing was taken from the device
    for out, w in zip(outs, want):
        got = float(out.item())
        assert abs(got - w) <= TOL_COULOMB * abs(w), (got, w)
    # again in the opposite order: the array keeps the last call's contents, the result must not
    for i in (1, 0):
        pg.coulomb_energy_noalloc(dev[i][0], dev[i][1], eps_in, outs[i])
    torch.cuda.synchronize()
    for out, w in zip(outs, want):
        assert abs(float(out.item()) - w) <= TOL_COULOMB * abs(w)
    # another permittivity scales the energy; fewer than two charges give zero
    pg.coulomb_energy_noalloc(dev[1][0], dev[1][1], 80.0, outs[1])
    pg.coulomb_energy_noalloc(dev[0][0][:1].contiguous(), dev[0][1][:1].contiguous(), eps_in, outs[0])
    torch.cuda.synchronize()
    assert abs(float(outs[1].item()) - want[1] * eps_in / 80.0) <= TOL_COULOMB * abs(want[1])
    assert float(outs[0].item()) == 0.0


def test_no_alloc_rejects_sizes_beyond_the_static_array(env):
    pg, torch = env
    n = pg.NOALLOC_MAX_CHARGES + 1
    xyz = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    q = torch.zeros(n, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(pg.PygbeError) as ei:
        pg.coulomb_energy_noalloc(xyz, q, 4.0, out)
    assert ei.value.code == pg.PYGBE_EINVAL and "maximum" in str(ei.value) and str(pg.NOALLOC_MAX_CHARGES) in str(ei.value)
    # the maximum itself is accepted
    xyz2, q2 = _charges(13, pg.NOALLOC_MAX_CHARGES, radius=20.0)
    pg.coulomb_energy_noalloc(torch.tensor(xyz2, device="cuda"), torch.tensor(q2, device="cuda"), 4.0, out)
    torch.cuda.synchronize()
    d = np.linalg.norm(xyz2[:400, None, :] - xyz2[None, :400, :], axis=2)
    assert np.isfinite(float(out.item())) and d[np.triu_indices(400, 1)].min() > 0
