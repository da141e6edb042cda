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


def test_ctypes_mirrors_have_the_layout_of_the_header(tmp_path):
    """The four public structs are declared twice: in include/pic.h and, by hand, as ctypes classes in the binding.
    A strict C11 client compiled against the header prints sizeof and every offsetof; they must equal the mirrors'."""
    import subprocess
    mirrors = {"pic_grid_desc": pic.pic_grid_desc, "pic_species_desc": pic.pic_species_desc,
               "pic_wall_flux_t": pic.pic_wall_flux_t, "pic_host_species": pic.pic_host_species}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "pic.h"', 'int main(void) {']
    for name, cls in mirrors.items():
        lines.append(f'    printf("{name} size %zu\\n", sizeof({name}));')
        for field, _ in cls._fields_:
            lines.append(f'    printf("{name} {field} %zu\\n", offsetof({name}, {field}));')
    lines += ['    return 0;', '}']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines) + "\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c11", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                    "-o", str(exe), str(src)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split("\n")
    seen = 0
    for line in filter(None, out):
        name, field, value = line.split()
        cls = mirrors[name]
        want = C.sizeof(cls) if field == "size" else getattr(cls, field).offset
        assert int(value) == want, f"{name}.{field}: header {value}, ctypes mirror {want}"
        seen += 1
    assert seen == sum(len(c._fields_) + 1 for c in mirrors.values())
    # every member of the header's structs is mirrored (a member added to the header only would shift nothing above)
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "pic.h")).read(), flags=re.S)
    for name, cls in mirrors.items():
        body = re.search(r"typedef struct \{([^}]*)\} " + name + ";", hdr).group(1)
        members = re.findall(r"\*?\b([A-Za-z_]\w*)\s*(?:\[\d+\])?\s*[,;]", body)
        assert sorted(members) == sorted(f for f, _ in cls._fields_), f"{name}: header members {members}"
