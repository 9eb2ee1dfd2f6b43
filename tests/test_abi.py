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
