"""On-disk cache of generated problems ("one generator writes .npz files that both read").

The large molecule meshes take 20-130 s to generate; tests and bench.py ask for them through `cached`, which
stores the finished Problem as an .npz in a temporary directory (never in the repository) keyed by the builder's
name, its arguments and a hash of the generator sources, so a stale file is never picked up after the recipe
changes.  Geometry only, like the rest of this package.
"""
import hashlib
import os
import tempfile

import numpy as np

from .problem import Problem, Surface

_HERE = os.path.dirname(os.path.abspath(__file__))


def _source_hash():
    h = hashlib.sha1()
    for f in ("molecule.py", "spheres.py", "problem.py"):
        with open(os.path.join(_HERE, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def cache_dir():
    d = os.environ.get("PYGBE_WORKLOAD_CACHE") or os.path.join(tempfile.gettempdir(), "pygbe_workloads")
    os.makedirs(d, exist_ok=True)
    return d


def save_problem(path, p):
    arrs = dict(eps=p.eps, kappa=p.kappa, charge_xyz=p.charge_xyz, charge_q=p.charge_q, charge_region=p.charge_region,
                n_surfaces=np.array(len(p.surfaces)), name=np.array(p.name),
                regions=np.array([[s.region_in, s.region_out] for s in p.surfaces], dtype=np.int32))
    for i, s in enumerate(p.surfaces):
        arrs[f"v{i}"] = s.vertices
        arrs[f"t{i}"] = s.triangles
    tmp = path + ".tmp%d.npz" % os.getpid()
    np.savez(tmp, **arrs)
    os.replace(tmp, path)


def load_problem(path):
    z = np.load(path)
    reg = z["regions"]
    surfaces = [Surface(z[f"v{i}"], z[f"t{i}"], int(reg[i, 0]), int(reg[i, 1])) for i in range(int(z["n_surfaces"]))]
    return Problem(surfaces, z["eps"], z["kappa"], z["charge_xyz"], z["charge_q"], z["charge_region"], name=str(z["name"]))


def cached(tag, build, wait_seconds=900.0):
    """Problem `tag` (a string naming builder and arguments) from the cache, else build() and store it.  When several
    processes ask at once (one rank per GPU under torchrun), one of them builds -- it holds an exclusive lock file --
    and the others wait for the .npz to appear (or, if the builder dies, for the lock to go stale) instead of all
    generating the same mesh side by side."""
    import time
    path = os.path.join(cache_dir(), "%s_%s.npz" % (tag, _source_hash()))
    lock = path + ".lock"

    def try_load():
        if os.path.exists(path):
            try:
                return load_problem(path)
            except Exception:
                try:
                    os.remove(path)
                except OSError:
                    pass
        return None

    p = try_load()
    if p is not None:
        return p
    have_lock = False
    t0 = time.time()
    while True:
        try:
            os.close(os.open(lock, os.O_CREAT | os.O_EXCL | os.O_WRONLY))
            have_lock = True
            break
        except FileExistsError:
            time.sleep(0.5)
            p = try_load()
            if p is not None:
                return p
            try:
                stale = time.time() - os.path.getmtime(lock) > wait_seconds
            except OSError:
                stale = False                                   # lock just went away: try to take it
            if stale or time.time() - t0 > wait_seconds:
                break                                           # builder died or is too slow: build here, without the lock
        except OSError:
            break                                               # cache directory not writable: just build
    try:
        p = try_load() or build()
        try:
            if not os.path.exists(path):
                save_problem(path, p)
        except OSError:
            pass
        return p
    finally:
        if have_lock:
            try:
                os.remove(lock)
            except OSError:
                pass
