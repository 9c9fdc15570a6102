"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/gray.h declares
(-m "not gpu": no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1303_5057_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "gray.h")).read()
    return sorted(set(re.findall(r"GRAY_API\s+[\w\s\*]+?\b(gray_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for need in ("gray_init_rays", "gray_integrate", "gray_classify", "gray_shadow_edge"):
        assert need in names
    assert len(names) >= 10


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in _declared():
        assert hasattr(L, name), name


def test_no_compute_free_calls(libpath):
    L = ctypes.CDLL(libpath)
    L.gray_version.restype = ctypes.c_char_p
    L.gray_workspace_bytes.restype = ctypes.c_size_t
    L.gray_workspace_bytes.argtypes = [ctypes.c_uint64]
    assert b"sm_100a" in L.gray_version()
    assert L.gray_workspace_bytes(1 << 30) >= 256


def test_argument_errors_are_reported_before_any_launch(libpath):
    import paper_1303_5057_b200.gray as g
    L = g.lib()
    st = g._State()
    st.prec = 7
    assert L.gray_init_rays(ctypes.byref(st), 0.5, 1000.0, 60.0, 10.0, 8, 8, 0, None) == -1   # GRAY_ERR_ARG
    assert b"prec" in L.gray_last_error()
    st.prec = g.GRAY_F32
    st.n = 0
    assert L.gray_init_rays(ctypes.byref(st), 1.5, 1000.0, 60.0, 10.0, 8, 8, 0, None) == -2   # GRAY_ERR_DOMAIN
    assert L.gray_init_rays(ctypes.byref(st), 0.5, 1000.0, 60.0, 500.0, 8, 8, 0, None) == -2  # pixel outside 1.01 r_obs
    assert L.gray_init_rays(ctypes.byref(st), 0.5, 1000.0, 60.0, 10.0, 8, 8, 0, None) == 0    # empty batch: no launch
    st.n = 4
    assert L.gray_init_rays(ctypes.byref(st), 0.5, 1000.0, 60.0, 10.0, 8, 8, 0, None) == -1   # NULL device pointers
    sp = g.StepParams().c
    st.n = 0
    assert L.gray_integrate(ctypes.byref(st), 0, 10, ctypes.byref(sp), None, 0, None) == -3    # GRAY_ERR_WORKSPACE
    # option combinations that have no kernel are refused by name, not approximated
    for kw, code in ((dict(frozen=True, xi_epsilon=1e-3), -5), (dict(frozen=True, stop_at_equator=True), -5),
                     (dict(system=g.SYS_REDUCED, xi_epsilon=1e-3), -5), (dict(system=g.SYS_REDUCED, frozen=True), -5),
                     (dict(system=g.SYS_REDUCED, stop_at_equator=True), -5), (dict(xi_epsilon=-1.0), -2),
                     (dict(system=7), -1), (dict(photons_per_thread=3), -1), (dict(rule=9), -1), (dict(schedule=5), -1)):
        sp = g.StepParams(**kw).c
        assert L.gray_integrate(ctypes.byref(st), 0, 10, ctypes.byref(sp), None, 0, None) == code, kw
    st.prec = g.GRAY_F64
    sp = g.StepParams(photons_per_thread=2).c
    assert L.gray_integrate(ctypes.byref(st), 0, 10, ctypes.byref(sp), None, 0, None) == -5   # packed FP32 needs GRAY_F32
    st.prec = g.GRAY_F32
    assert L.gray_init_rays_polar(ctypes.byref(st), 0.5, 1000.0, 60.0, 7.5, 1.5, 10, 5, 0, None) == -2      # R_lo >= R_hi
    assert L.gray_init_rays_polar(ctypes.byref(st), 0.5, 1000.0, 60.0, 1.5, 7.5, 10, 1, 0, None) == -2      # n_theta < 2
    v = ctypes.c_double()
    assert L.gray_packed_peak(7, 16, ctypes.byref(v), None) == -1 and L.gray_fma_peak(2, 16, ctypes.byref(v), None) == -1


def test_product_does_not_import_the_oracle():
    # the oracle is test infrastructure: nothing in the package or at the ABI may import, include or link it
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|from\s+\.+oracle|#\s*include\s*[\"<][^\n]*oracle)", re.M)
    for top in ("paper_1303_5057_b200", "include"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, top)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    assert not pat.search(open(os.path.join(dirpath, f)).read()), (dirpath, f)
    out = os.popen("ldd " + os.path.join(ROOT, "paper_1303_5057_b200", "libgray.so")).read()
    assert "oracle" not in out


def test_shard_range_partitions():
    from paper_1303_5057_b200.workloads import shard_range
    for n in (0, 1, 7, 4096, 2 ** 30 + 3):
        for ws in (1, 2, 3, 8):
            parts = [shard_range(n, r, ws) for r in range(ws)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(ws - 1))
            assert max(h - l for l, h in parts) - min(h - l for l, h in parts) <= 1
