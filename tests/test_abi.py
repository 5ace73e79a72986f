"""CPU-side checks of the boundary: libsugauge.so builds (nvcc cross-compiles sm_100a without a GPU),
loads, and exports every function include/su_gauge.h declares - and nothing else. No compute calls."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "su_gauge.h")
TEST_HEADER = os.path.join(ROOT, "include", "su_gauge_test.h")      # micro-benchmarks and test hooks: not product interface
TEST_ONLY = ["su_debug_kp_math", "su_fused_dep_debug", "su_fused_schedule_debug", "su_measure_fma_peak", "su_measure_l2_peak"]


def _names(path):
    text = open(path).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(su_[a-z0-9_]+)\s*\(", text)))


def _declared():
    return sorted(_names(HEADER) + _names(TEST_HEADER))


def test_product_header_holds_no_benchmark_or_debug_entry_point():
    assert _names(TEST_HEADER) == TEST_ONLY
    assert not set(_names(HEADER)) & set(TEST_ONLY)
    assert not [n for n in _names(HEADER) if "debug" in n or "measure" in n]


@pytest.fixture(scope="module")
def libpath():
    from paper_1112_4533_b200 import build
    return build.build()


def test_header_declares_the_north_star_calls():
    names = _declared()
    for required in ("su_lattice_create", "su_init_cold", "su_init_hot", "su_sweep", "su_plaquette",
                     "su_polyakov", "su_reunitarize", "su_export_links"):
        assert required in names


def test_library_exports_exactly_the_declared_symbols(libpath):
    out = subprocess.run(["nm", "-D", "--defined-only", libpath], capture_output=True, text=True, check=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("su_"))
    assert exported == _declared()
    lib = ctypes.CDLL(libpath)
    for name in _declared():
        assert getattr(lib, name) is not None


def test_binding_covers_the_header(libpath):
    import paper_1112_4533_b200 as su
    assert sorted(su.ABI_SYMBOLS) == _declared()
    su.lib()


def test_pure_host_entry_points(libpath):
    """su_lattice_bytes and argument validation run without a GPU."""
    import paper_1112_4533_b200 as su
    V = 48 ** 4
    assert su.lattice_bytes(3, (48,) * 4, "fp64") == 4 * V * 18 * 8            # ~3 GB (BASELINE.json configs[2])
    assert su.lattice_bytes(3, (48,) * 4, "fp32", recon12=True) == 4 * V * 12 * 4
    assert su.lattice_bytes(2, (8,) * 4, "fp64") == 4 * 8 ** 4 * 4 * 8
    assert su.lattice_bytes(4, (24,) * 4, "fp32") == 4 * 24 ** 4 * 32 * 4
    assert su.lattice_bytes(3, (4, 4, 4, 5), "fp64") == 0                      # odd extent
    assert su.lattice_bytes(4, (4, 4, 4, 4), "fp64", recon12=True) == 0        # RECON12 is SU(3) only
    L = su.lib()
    assert L.su_sweep(None, 6.0, 1, 4) == su.SU_EINVAL
    assert L.su_lattice_destroy(None) == su.SU_EINVAL
    assert L.su_last_error(None) == b"null lattice handle"
    assert L.su_lattice_create(3, 4, 4, 4, 4, 1, None) == su.SU_EINVAL
    h = ctypes.c_void_p()
    assert L.su_lattice_create(3, 4, 4, 4, 3, 1, ctypes.byref(h)) == su.SU_EINVAL
    assert L.su_lattice_create(1, 4, 4, 4, 4, 1, ctypes.byref(h)) == su.SU_EINVAL
    assert L.su_lattice_create(su.SU_MAX_NC + 1, 4, 4, 4, 4, 1, ctypes.byref(h)) == su.SU_EUNSUPPORTED


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1112_4533_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower().replace("no cpu fallback", ""), f
