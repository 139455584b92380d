"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every function that
include/phx.h declares; the Python binding lists the same names; host-side argument validation works
without touching a device."""
import ctypes as C
import os
import re

import numpy as np

from paper_2410_09146_b200 import phx, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "phx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(phx_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_five_north_star_calls():
    names = declared_functions()
    for need in ("phx_init_mesh", "phx_prim_to_cons", "phx_cons_to_prim", "phx_rk_stage", "phx_cfl_dt"):
        assert need in names


def test_library_exports_every_declared_symbol():
    L = C.CDLL(phx.LIB_PATH)
    for name in declared_functions():
        assert hasattr(L, name), name
    assert sorted(phx.EXPORTS) == declared_functions()


def test_params_struct_matches_header_field_order():
    src = open(os.path.join(ROOT, "include", "phx.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} phx_params;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(int|double)\s+", "", decl)
        for f in decl.split(","):
            fields.append(re.sub(r"\[.*", "", f.strip()))
    assert fields == [n for n, _ in phx.Params._fields_]


def test_null_and_invalid_arguments_are_rejected_before_any_launch():
    L = phx.lib()
    out = C.c_void_p()
    assert L.phx_init_mesh(None, None, C.byref(out)) == phx.EINVAL
    p = wl.default_params(nx=8, ny=8, nz=8, ng=1)
    assert L.phx_init_mesh(C.byref(phx.make_params(p)), None, C.byref(out)) == phx.EINVAL
    assert b"ng" in L.phx_last_error()
    p = wl.default_params(nx=8, ny=8, nz=8, recon=7)
    assert L.phx_init_mesh(C.byref(phx.make_params(p)), None, C.byref(out)) == phx.EUNSUPPORTED
    assert L.phx_field_elems(None) == 0
    assert L.phx_free_mesh(None) == phx.OK


def test_workload_layout_helpers_round_trip():
    p = wl.default_params(nbx=2, nby=3, nbz=1, nx=4, ny=4, nz=1, ng=2)
    rng = np.random.default_rng(0)
    q = rng.standard_normal((8, 1, 12, 8))
    b = wl.finish(p, q)
    assert b.shape == wl.alloc_shape(p) == (6, 8, 1, 8, 8)
    assert np.array_equal(wl.from_blocks(p, b), q)
