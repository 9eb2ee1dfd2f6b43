"""CPU-side checks of the boundary: the shared library loads and exports every symbol that
include/pygbe.h declares; struct layouts of the binding match the header's field lists."""
import ctypes as C
import os
import re

import pytest

import paper_1309_4018_b200 as pg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pygbe.h")


@pytest.fixture(scope="module")
def built_lib():
    from paper_1309_4018_b200.build import build
    build()
    return pg.lib()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pygbe_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for must in ("pygbe_create", "pygbe_matvec", "pygbe_solve", "pygbe_energy", "pygbe_rhs", "pygbe_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(built_lib):
    for name in _declared_functions():
        assert hasattr(built_lib, name), f"{name} declared in pygbe.h but not exported"


def test_version_and_error_string(built_lib):
    assert b"sm_100a" in built_lib.pygbe_version()
    assert built_lib.pygbe_last_error() is not None


def test_struct_fields_match_header():
    src = open(HEADER).read()
    for struct, cls in (("pygbe_surface", pg.pygbe_surface), ("pygbe_charges", pg.pygbe_charges),
                        ("pygbe_options", pg.pygbe_options), ("pygbe_stats_t", pg.pygbe_stats_t)):
        end = re.search(r"\}\s*" + struct + r"\s*;", src).start()
        body = src[src.rfind("typedef struct {", 0, end) + len("typedef struct {"):end]
        body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
        names = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            decl = re.sub(r"^(const\s+)?[A-Za-z_0-9]+\s*", "", decl, count=1)     # drop the type
            for part in decl.split(","):
                names.append(re.sub(r"[\*\s]|\[.*\]", "", part))
        assert names == [n for n, _ in cls._fields_], struct


def test_invalid_arguments_are_rejected_without_a_gpu(built_lib):
    """Argument validation happens before any CUDA call, so it can be exercised on the CPU box."""
    h = C.c_void_p(123)
    rc = built_lib.pygbe_create(None, 0, None, None, None, 0, 4, 6, 0.5, None, C.byref(h))
    assert rc == pg.PYGBE_EINVAL and h.value is None
    assert b"missing" in built_lib.pygbe_last_error()
    assert built_lib.pygbe_num_unknowns(None) < 0
    assert built_lib.pygbe_matvec(None, None, None) == pg.PYGBE_EINVAL
    assert built_lib.pygbe_solve(None, 1e-6, 10, 10, None, None, None) == pg.PYGBE_EINVAL


def test_no_cpu_fallback():
    """The product never imports the oracle and raises without a device."""
    import torch
    pkg = os.path.join(ROOT, "paper_1309_4018_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "pb_oracle" not in text, f
    if not torch.cuda.is_available():
        import workloads as W
        with pytest.raises(RuntimeError):
            pg.Handle.from_problem(W.born_problem(1))


def _create_args(surfs, n_regions, eps=None, kappa=None):
    import numpy as np
    import workloads as W
    keep = []
    arr = (pg.pygbe_surface * len(surfs))()
    for i, (level, radius, rin, rout) in enumerate(surfs):
        v, t = W.icosphere(level, radius)
        v = np.ascontiguousarray(v, dtype=np.float64); t = np.ascontiguousarray(t, dtype=np.int32)
        keep += [v, t]
        arr[i] = pg.pygbe_surface(v.ctypes.data_as(C.POINTER(C.c_double)), v.shape[0],
                                  t.ctypes.data_as(C.POINTER(C.c_int32)), t.shape[0], rin, rout)
    eps = np.array(eps if eps is not None else [4.0] + [80.0] * (n_regions - 1), dtype=np.float64)
    kappa = np.array(kappa if kappa is not None else [0.0] * n_regions, dtype=np.float64)
    keep += [eps, kappa]
    dp = C.POINTER(C.c_double)
    return keep, (arr, len(surfs), None, eps.ctypes.data_as(dp), kappa.ctypes.data_as(dp), n_regions, 4, 6, 0.5)


def test_region_graph_must_be_a_tree(built_lib):
    """SURVEY 8(b) EINVAL list: 'region graph not a tree'.  Checked on the host before any CUDA call."""
    h = C.c_void_p(1)
    # three nested spheres whose region ids close a cycle: 0-1, 1-2, 2-0
    keep, args = _create_args([(1, 2.0, 0, 1), (1, 4.0, 1, 2), (1, 6.0, 2, 0)], 3)
    assert built_lib.pygbe_create(*args, None, C.byref(h)) == pg.PYGBE_EINVAL and h.value is None
    assert b"not a tree" in built_lib.pygbe_last_error()
    # two components that no surface joins: 0-1 and 2-3
    keep, args = _create_args([(1, 2.0, 0, 1), (1, 4.0, 2, 3)], 4)
    assert built_lib.pygbe_create(*args, None, C.byref(h)) == pg.PYGBE_EINVAL
    assert b"not a tree" in built_lib.pygbe_last_error()
    # the same pair in opposite directions
    keep, args = _create_args([(1, 2.0, 0, 1), (1, 4.0, 1, 0)], 2)
    assert built_lib.pygbe_create(*args, None, C.byref(h)) == pg.PYGBE_EINVAL
    # the size query validates its arguments the same way
    n = C.c_size_t(7)
    keep, args = _create_args([(1, 2.0, 0, 1), (1, 4.0, 1, 2), (1, 6.0, 2, 0)], 3)
    assert built_lib.pygbe_workspace_size(*args, None, 100, C.byref(n)) == pg.PYGBE_EINVAL and n.value == 0
    assert built_lib.pygbe_workspace_size(*args, None, 100, None) == pg.PYGBE_EINVAL


def test_options_reject_bad_workspace_and_group_mac(built_lib):
    h = C.c_void_p(1)
    keep, args = _create_args([(1, 2.0, 0, 1)], 2)
    opt = pg.pygbe_options(group_mac=2)
    assert built_lib.pygbe_create(*args, C.byref(opt), C.byref(h)) == pg.PYGBE_EINVAL
    opt = pg.pygbe_options(workspace=C.c_void_p(0x1001), workspace_bytes=1 << 20)     # not 256-byte aligned
    assert built_lib.pygbe_create(*args, C.byref(opt), C.byref(h)) == pg.PYGBE_EINVAL
    assert b"aligned" in built_lib.pygbe_last_error()
    opt = pg.pygbe_options(workspace_bytes=1 << 20)                                   # size without a block
    assert built_lib.pygbe_create(*args, C.byref(opt), C.byref(h)) == pg.PYGBE_EINVAL


def test_no_environment_knobs_in_the_product_build():
    """Tuning knobs are compiled out unless -DPYGBE_TUNING: the only getenv of the library sits behind that flag."""
    csrc = os.path.join(ROOT, "paper_1309_4018_b200", "csrc")
    hits = []
    for f in sorted(os.listdir(csrc)):
        for i, line in enumerate(open(os.path.join(csrc, f)), 1):
            if re.search(r"\bgetenv\s*\(", line) and not line.strip().startswith("//"):
                hits.append((f, i))
    assert hits == [("common.cuh", hits[0][1])] and len(hits) == 1


def test_no_library_kernels_in_the_product():
    """North star: hand-written kernels, a GMRES "built on its own reduction kernels": no CUB / Thrust / cuBLAS include
    anywhere in the library's sources (the Morton sort and the block reductions are csrc/blockops.cuh)."""
    csrc = os.path.join(ROOT, "paper_1309_4018_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        text = open(os.path.join(csrc, f)).read()
        for lib in ("cub/", "thrust/", "cublas", "cusparse", "cusolver"):
            assert not re.search(r"#include\s*[<\"]" + lib, text), (f, lib)
