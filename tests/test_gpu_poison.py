"""NaN-poison pass over every kernel family (pytest -m gpu): the link buffer is filled with 0xFF
bytes (NaN in fp32 and fp64) before every initialisation and import, so a read of a never-written element (pad sites of
the tiled planes, stale halos) would surface as a non-finite observable or link - the repository's stand-in for
compute-sanitizer's initcheck, which is closed on this GPU pool (profiles/r02e_sanitizers.md). Run against a library
built with device-side asserts on every checkerboard index the kernels form it is also the stand-in for memcheck:

    SUG_BUILD_VARIANT=check SUG_NVCC_EXTRA=-DSUG_CHECK=1 python -m paper_1112_4533_b200.build
    SU_GAUGE_LIB=paper_1112_4533_b200/libsugauge_check.so python -m pytest tests/test_gpu_poison.py -m gpu

Covers the register kernels (SU(2) quaternion, SU(3) 18- and 12-real, SU(4)), the row-per-lane generic kernels (SU(6)),
the runtime-Nc warp-per-link kernels (Nc = 9), fused multi-sub-step launches, two t-slabs with the fused halo push, both
reductions, reunitarisation, hot start and import / export, once each on a ragged lattice. Results are checked by
tests/test_gpu_parity.py and friends; this file only asks that nothing uninitialised is ever read.
(Until round 2 this was the stand-alone script tests/sanitizer_case.py.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DIMS = (4, 6, 4, 6)
BETA = {2: 2.3, 3: 6.0, 4: 11.0, 6: 25.0, 9: 57.0}


@pytest.fixture(scope="module")
def su():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1112_4533_b200 as su
    return su


CASES = [dict(Nc=2, precision="fp64"), dict(Nc=3, precision="fp64"), dict(Nc=3, precision="fp32", recon12=True),
         dict(Nc=3, precision="fp64", fuse=4, reunit_on_store=True), dict(Nc=3, precision="fp32", fuse=8),
         dict(Nc=4, precision="fp64"), dict(Nc=3, precision="fp64", kernel="generic"), dict(Nc=6, precision="fp64"),
         dict(Nc=6, precision="fp32"), dict(Nc=9, precision="fp64")]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "-".join(f"{k}{v}" for k, v in c.items()))
def test_poisoned_buffer_never_shows(su, case):
    Nc, precision = case["Nc"], case["precision"]
    L = su.Lattice(Nc, DIMS, precision, case.get("recon12", False), case.get("kernel", "auto"))
    L.buffer.fill_(0xFF)                                     # all-ones = NaN in fp32 and fp64
    if case.get("fuse", 1) > 1:
        L.set_option("fuse", case["fuse"])
    if case.get("reunit_on_store"):
        L.set_option("reunit_on_store", 1)
    L.init_hot(3)
    L.sweep(BETA[Nc], 1, 1)
    L.substep(BETA[Nc], 0, 0, 1, 2, want_attempts=True)
    L.reunitarize()
    p, q = L.plaquette(), L.polyakov()
    links = L.export_links()
    assert np.isfinite(p) and np.isfinite(abs(q)) and np.isfinite(links).all()
    L.buffer.fill_(0xFF)
    L.import_links(links)
    assert np.isfinite(L.plaquette()) and np.array_equal(L.export_links(), links)
    L.init_cold(1)
    assert L.plaquette() == 1.0
    L.close()


@pytest.mark.parametrize("Nc,beta", [(3, 6.0), (6, 25.0)])
def test_poisoned_slabs_never_show(su, Nc, beta):
    from paper_1112_4533_b200.slab import SlabGroup
    S = SlabGroup(Nc, (8, 4, 4, 4), 2, "fp64")
    for sl in S.slabs:
        sl.buffer.fill_(0xFF)
    S.init_hot(2)
    S.sweep(beta, 1, 1)
    S.reunitarize()
    assert np.isfinite(S.plaquette()) and np.isfinite(S.export_links()).all()
    S.close()
