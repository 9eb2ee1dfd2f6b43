"""Plain containers for a multi-surface Poisson-Boltzmann BEM input (no arithmetic of the method).

A problem = closed triangulated surfaces + point charges + a region table (Fig. 4).
Surface normals follow the triangle winding: counter-clockwise seen from region_out, so the normal
points region_in -> region_out (reading A3 in DESIGN.md).
"""
from dataclasses import dataclass, field
import numpy as np


@dataclass
class Surface:
    vertices: np.ndarray      # [nv,3] float64, Angstrom
    triangles: np.ndarray     # [nt,3] int32, 0-based
    region_in: int
    region_out: int

    def __post_init__(self):
        self.vertices = np.ascontiguousarray(self.vertices, dtype=np.float64)
        self.triangles = np.ascontiguousarray(self.triangles, dtype=np.int32)

    @property
    def n_panels(self):
        return int(self.triangles.shape[0])


@dataclass
class Problem:
    surfaces: list                      # list[Surface]
    eps: np.ndarray                     # [n_regions]
    kappa: np.ndarray                   # [n_regions], 1/Angstrom
    charge_xyz: np.ndarray              # [nq,3]
    charge_q: np.ndarray                # [nq] units of e
    charge_region: np.ndarray           # [nq] int32
    name: str = ""
    meta: dict = field(default_factory=dict)

    def __post_init__(self):
        self.eps = np.ascontiguousarray(self.eps, dtype=np.float64)
        self.kappa = np.ascontiguousarray(self.kappa, dtype=np.float64)
        self.charge_xyz = np.ascontiguousarray(self.charge_xyz, dtype=np.float64).reshape(-1, 3)
        self.charge_q = np.ascontiguousarray(self.charge_q, dtype=np.float64).reshape(-1)
        self.charge_region = np.ascontiguousarray(self.charge_region, dtype=np.int32).reshape(-1)

    @property
    def n_panels(self):
        return sum(s.n_panels for s in self.surfaces)

    @property
    def n_unknowns(self):
        return 2 * self.n_panels

    @property
    def n_regions(self):
        return int(self.eps.shape[0])


def concat_problem_arrays(p: Problem):
    """Flatten the surfaces to per-panel arrays: corner coordinates [N,9], surface id [N],
    plus per-surface region_in / region_out.  Pure indexing, no geometry is computed."""
    tri, surf = [], []
    for s, S in enumerate(p.surfaces):
        tri.append(S.vertices[S.triangles].reshape(-1, 9))
        surf.append(np.full(S.n_panels, s, dtype=np.int32))
    tri = np.ascontiguousarray(np.concatenate(tri, axis=0))
    surf = np.ascontiguousarray(np.concatenate(surf))
    rin = np.array([S.region_in for S in p.surfaces], dtype=np.int32)
    rout = np.array([S.region_out for S in p.surfaces], dtype=np.int32)
    return tri, surf, rin, rout
