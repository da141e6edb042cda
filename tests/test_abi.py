"""CPU-side checks of the C-ABI boundary: libpic.so builds for sm_100a, loads, and exports every
function include/pic.h declares; argument validation that needs no GPU returns the documented
status codes.  No compute call is made here."""
import ctypes as C
import os
import re

import paper_2603_24508_b200 as pic
from paper_2603_24508_b200 import build as pic_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pic_[a-z_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = pic_build.build()
    assert os.path.exists(path)
    L = C.CDLL(path)
    names = declared_functions()
    assert len(names) >= 19
    for name in names:
        assert hasattr(L, name), f"{name} declared in include/pic.h but not exported by libpic.so"
    assert sorted(pic.EXPORTS) == names, "Python binding and header disagree on the entry points"


def test_binding_exposes_the_same_names():
    for name in declared_functions():
        assert hasattr(pic, name), f"binding lacks {name}"


def test_strerror_and_workspace_size():
    assert pic.pic_strerror(pic.PIC_OK) == "ok"
    assert "argument" in pic.pic_strerror(pic.PIC_EINVAL)
    assert pic.pic_strerror(-99) == "unknown status"
    cap = 1_000_000
    b = pic.pic_workspace_bytes(1000, cap)
    assert 16 * cap <= b <= 18 * cap
    assert pic.pic_workspace_bytes(1000, 0) < 8192


def test_argument_validation_without_gpu():
    L = pic.lib()
    h = C.c_void_p()
    assert L.pic_create(None, None, 1, C.byref(h)) == pic.PIC_EINVAL
    g = pic.pic_grid_desc()
    d = (pic.pic_species_desc * 1)()
    g.nc, g.dx, g.dt = 0, 1.0, 0.1
    assert L.pic_create(C.byref(g), d, 1, C.byref(h)) == pic.PIC_EINVAL  # nc < 1 / no E
    E = (C.c_double * 3)(0.0, float("nan"), 0.0)
    g.nc = 2
    g.E_nodes = C.cast(E, C.POINTER(C.c_double))
    assert L.pic_create(C.byref(g), d, 1, C.byref(h)) == pic.PIC_EINVAL  # non-finite E
    assert h.value is None
    assert L.pic_push(None, 1) == pic.PIC_EINVAL
    assert L.pic_arrange(None) == pic.PIC_EINVAL
    assert L.pic_wall_flux(None, None) == pic.PIC_EINVAL
    assert L.pic_sync(None) == pic.PIC_EINVAL
    assert L.pic_run_host(None, None, 0, 0) == pic.PIC_EINVAL
    assert L.pic_push_all(None, 1) == pic.PIC_EINVAL
    assert L.pic_cycle(None, 1, None, 0, None, None) == pic.PIC_EINVAL
    assert L.pic_solve_field(None, None, 0, None) == pic.PIC_EINVAL
    assert L.pic_deposit(None, 1.0, None, 0) == pic.PIC_EINVAL
    L.pic_destroy(None)
