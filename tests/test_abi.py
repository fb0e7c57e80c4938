"""CPU checks of the C-ABI: the library builds, loads without a GPU and exports every symbol that
include/hamr.h declares; the binding's struct matches the oracle's (same parameter block)."""
import ctypes as C
import os
import re

from paper_1912_10192_b200 import build, hamr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(header="hamr.h"):
    txt = open(os.path.join(ROOT, "include", header)).read()
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
    dbg = _declared("hamr_debug.h")
    assert "hamr_debug_geometry" in dbg and "hamr_bench_fp64" in dbg
    for s in dbg:
        assert hasattr(L, s), s
    assert sorted(hamr.DEBUG_SYMBOLS) == dbg
    assert not set(dbg) & set(names)


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
    # the spherical map needs x2 = (0, pi) with polar boundaries: a wedge or an outflow x2 is refused, as is a map
    # that does not go with the metric
    for change in (dict(xmin=(1.2, 0.1, 0.0)), dict(xmax=(50.0, 3.0, 2.0 * 3.141592653589793)),
                   dict(bc_lo=(I.BC_OUTFLOW, I.BC_OUTFLOW, I.BC_PERIODIC)), dict(map=1)):
        par = hamr.pack_params(dict(I.torus_params(), **change))
        assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.EINVAL, change
    par = hamr.pack_params(dict(I.torus_params(), map=2))
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK
    # NEXT-2 (entropy backup, drift-frame floors): flags 0 / 1, gamma_ad < 2; four more arrays
    base = n.value
    par = hamr.pack_params(dict(I.torus_params(), entropy_backup=1, drift_floors=1))
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK and n.value > base
    par = hamr.pack_params(dict(I.torus_params(), entropy_backup=1, drift_floors=1, nb=(8, 8, 8)))   # blocks on one time level: fine
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK
    par = hamr.pack_params(dict(I.torus_params(), entropy_backup=1, deref_theta_deg=(15.0,), deref_factor=(2,)))   # derefined rows: fine
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK
    par = hamr.pack_params(dict(I.torus_params(), entropy_backup=1, drift_floors=1, nb=(8, 8, 8), lat_max_level=1))   # LAT: fine
    assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.OK
    for change in (dict(entropy_backup=2),
                   dict(drift_floors=-1), dict(entropy_backup=1, gamma_ad=2.0)):
        par = hamr.pack_params(dict(I.torus_params(), **change))
        assert L.hamr_workspace_bytes(C.byref(par), C.byref(n)) == hamr.EINVAL, change
    assert L.hamr_step(None, 1, None, None) == hamr.EINVAL
