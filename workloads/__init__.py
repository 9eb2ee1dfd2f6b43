"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds geometry and input generation ONLY (meshes, charges, region tables).
None of the method's arithmetic (kernels, quadrature, operators, energies) lives here.
Recipes are stated in DESIGN.md "Input recipe"; they follow SURVEY.md section 8(d) and stand in for
the MSMS / pdb2pqr molecules of PAPER.md:195, Tables 1-6, which are not available.
"""
from .spheres import (icosphere, born_problem, kirkwood_problem, stern_sphere_problem, cavity_sphere_problem,
                      nested_sphere_problem)
from .problem import Problem, Surface, concat_problem_arrays
from .molecule import (saw_molecule, density_surface, marching_tetrahedra, validate_closed_mesh,
                       protein_problem, multisurface_problem, binding_problems)
from .cache import cached, save_problem, load_problem

SEED0 = 13094018

__all__ = [
    "icosphere", "born_problem", "kirkwood_problem", "stern_sphere_problem", "cavity_sphere_problem",
    "nested_sphere_problem",
    "Problem", "Surface", "concat_problem_arrays", "saw_molecule", "density_surface", "marching_tetrahedra",
    "validate_closed_mesh", "protein_problem", "multisurface_problem", "binding_problems", "SEED0",
    "cached", "save_problem", "load_problem",
]
