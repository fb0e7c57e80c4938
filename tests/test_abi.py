"""CPU checks of the C-ABI: the library builds, loads without a GPU and exports every symbol that
include/hamr.h declares; the binding's struct matches the oracle's (same parameter block)."""
import ctypes as C
import os
import re

from paper_1912_10192_b200 import build, hamr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "hamr.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(hamr_[a-z_0-9]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    build.build_lib()
    L = C.CDLL(hamr.LIB_PATH)
    names = _declared()
    assert "hamr_step" in names and "hamr_grid_create" in names and len(names) >= 20
    for s in names:
        assert hasattr(L, s), s
    assert sorted(hamr.SYMBOLS) == names


def test_binding_params_layout_matches_header_order():
    txt = open(os.path.join(ROOT, "include", "hamr.h")).read()
    body = txt[txt.index("typedef struct {"):txt.index("} hamr_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        for part in decl.split(",")[0:]:
            name = re.sub(r"\[.*?\]", "", part.strip().split()[-1])
            fields.append(name)
    assert fields == [f[0] for f in hamr.Params._fields_]


def test_bad_arguments_are_rejected_without_a_gpu():
    L = hamr.lib()
    assert L.hamr_grid_create(None, None) == hamr.EINVAL
    n = C.c_size_t(0)
    from paper_1912_10192_b200 import inputs as I
    par = hamr.pack_params(I.torus_params())
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK and n.value > 0
    par.n[0] = 0
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.EINVAL
    assert L.hamr_step(None, 1, None, None) == hamr.EINVAL
