"""One small pass of every kernel family, written for compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_case.py

compute-sanitizer is CLOSED on this GPU pool (profiles/r02_sanitizers.md quotes the refusal), so the same script is
run against a build with device-side asserts on every checkerboard index the kernels form

    SUG_BUILD_VARIANT=check SUG_NVCC_EXTRA=-DSUG_CHECK=1 python -m paper_1112_4533_b200.build
    SU_GAUGE_LIB=paper_1112_4533_b200/libsugauge_check.so python tests/sanitizer_case.py

(our own bounds check) and with the link buffer POISONED with NaN bit patterns before every initialisation, so a read
of a never-written element (pad sites of the tiled planes, stale halos) would surface as a non-finite observable
(our own initcheck). Covers the register kernels (SU(2) quaternion, SU(3) 18- and
12-real, SU(4)), the row-per-lane generic kernels (SU(6): operands staged in shared memory with warp-level barriers,
shadow lanes), the runtime-Nc warp-per-link kernels (Nc = 9), a fused multi-sub-step launch (ticket table, completion
counters), two t-slabs with the fused halo push, both reductions, reunitarisation, hot start and import / export.
Not a test of results (tests/test_gpu_*.py are); it only has to touch every code path once on a ragged lattice."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_1112_4533_b200 as su                           # noqa: E402
from paper_1112_4533_b200.slab import SlabGroup              # noqa: E402

DIMS = (4, 6, 4, 6)
BETA = {2: 2.3, 3: 6.0, 4: 11.0, 6: 25.0, 9: 57.0}


def one(Nc, precision, recon12=False, kernel="auto", fuse=1, reunit_on_store=False):
    L = su.Lattice(Nc, DIMS, precision, recon12, kernel)
    L.buffer.fill_(0xFF)                                     # all-ones = NaN in fp32 and fp64
    if fuse > 1:
        L.set_option("fuse", fuse)
    if reunit_on_store:
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
    print(f"SU({Nc}) {precision}{' r12' if recon12 else ''} {kernel} fuse={fuse}: plaquette {p:.6f} |polyakov| {abs(q):.4f}", flush=True)


def main():
    one(2, "fp64")
    one(3, "fp64")
    one(3, "fp32", recon12=True)
    one(3, "fp64", fuse=4, reunit_on_store=True)
    one(3, "fp32", fuse=8)
    one(4, "fp64")
    one(3, "fp64", kernel="generic")
    one(6, "fp64")
    one(6, "fp32")
    one(9, "fp64")
    S = SlabGroup(3, (8, 4, 4, 4), 2, "fp64")
    for sl in S.slabs:
        sl.buffer.fill_(0xFF)
    S.init_hot(2)
    S.sweep(6.0, 1, 1)
    S.reunitarize()
    assert np.isfinite(S.plaquette()) and np.isfinite(S.export_links()).all()
    print(f"2 slabs SU(3): plaquette {S.plaquette():.6f}", flush=True)
    S.close()
    S = SlabGroup(6, (8, 4, 4, 4), 2, "fp64")
    S.init_hot(2)
    S.sweep(25.0, 1, 1)
    print(f"2 slabs SU(6): plaquette {S.plaquette():.6f}", flush=True)
    S.close()
    print("sanitizer case done")


if __name__ == "__main__":
    main()
