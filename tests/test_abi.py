"""Host-side checks of the C-ABI library (no GPU): it loads, exports every symbol include/petar.h
declares, and its host-only entry points behave."""
import ctypes as C
import os
import re

import pytest

import paper_2006_16560_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2006_16560_b200 import build
    build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "petar.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(petar_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    names = _declared()
    assert {"petar_tree_build", "petar_long_range_force", "petar_neighbor_list"} <= set(names)
    L = C.CDLL(P.library_path())
    for n in names:
        assert hasattr(L, n), n
    assert set(P.binding.EXPORTS) == set(names)


def test_workspace_query_and_param_validation():
    p = P.PetarParams.make(theta=0.3, multipole=2)
    b1, b2 = P.petar_workspace_bytes(1 << 16, p), P.petar_workspace_bytes(1 << 20, p)
    assert 0 < b1 < b2 < 64e9
    assert P.petar_workspace_bytes(-1, p) == 0
    for bad in (dict(multipole=3), dict(rho=1.5), dict(n_leaf=0), dict(n_group=4, n_leaf=8), dict(theta=-1.0)):
        kw = dict(theta=0.3, multipole=2); kw.update(bad)
        assert P.petar_workspace_bytes(1000, P.PetarParams.make(**kw)) == 0
    # a larger arena request is honoured
    p2 = P.PetarParams.make(theta=0.3, multipole=2, list_entries_per_particle=4096.0)
    assert P.petar_workspace_bytes(1 << 20, p2) > b2


def test_error_strings_and_null_handles():
    assert P.petar_strerror(0) == "ok"
    assert "workspace" in P.petar_strerror(-2)
    L = P.lib()
    assert L.petar_tree_destroy(None) == 0
    assert L.petar_long_range_force(None, None, None, None, None, None, None) == -4      # PETAR_ENOTBUILT
    assert L.petar_neighbor_list(None, None, None, 0, None, None) == -4
    h = C.c_void_p()
    p = P.PetarParams.make(theta=0.3, multipole=5)
    assert L.petar_tree_build(None, None, None, None, None, None, 10, C.byref(p), None, 0, None, C.byref(h)) == -1
    p = P.PetarParams.make(theta=0.3, multipole=2)
    assert L.petar_tree_build(None, None, None, None, None, None, 10, C.byref(p), None, 0, None, C.byref(h)) == -1  # NULL arrays
    assert L.petar_tree_build(None, None, None, None, None, None, 10, C.byref(p), None, 0, None, None) == -1


def test_noalloc_entry_point_host_checks():
    """petar_short_range_force_noalloc refuses a size beyond its built-in array, and bad arguments, before it touches the
    GPU (so this runs without one); the error text names the limit."""
    L = P.lib()
    nul = [None] * 10
    out = [None] * 7
    big = P.SHORT_RANGE_NOALLOC_MAX_N + 1
    call = lambda n, rho: L.petar_short_range_force_noalloc(*nul, C.c_int64(n), C.c_double(1.0), C.c_double(rho), *out, None)
    assert call(big, 0.1) == -6                      # PETAR_ECAPACITY
    assert call(-1, 0.1) == -1 and call(10, 1.5) == -1 and call(10, 0.1) == -1      # N < 0, bad ratio, NULL arrays
    assert call(0, 0.1) == 0                          # nothing to do
    assert "PETAR_SHORT_RANGE_NOALLOC_MAX_N" in P.petar_strerror(-6)
    hdr = open(os.path.join(ROOT, "include", "petar.h")).read()
    assert f"#define PETAR_SHORT_RANGE_NOALLOC_MAX_N {P.SHORT_RANGE_NOALLOC_MAX_N}" in hdr


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or anything under _work/)."""
    pkg = os.path.join(ROOT, "paper_2006_16560_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f), errors="ignore").read()
                assert "import oracle" not in txt and "from oracle" not in txt and "_work/" not in txt, f
                assert "petar_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2006_16560_b200" not in txt and "from paper_2006_16560_b200" not in txt
            assert "#include \"../" not in txt and "petar.h" not in txt
