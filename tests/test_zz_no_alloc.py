"""su_plaquette_static (include/su_gauge.h "a measurement that allocates nothing") against su_plaquette.

Who needs that entry point: users of the library that cannot call cudaMalloc when they want a plaquette value. A
production job that filled the GPU with its lattices, or that lives inside a program whose memory pool already holds
all free HBM, gets an error (or steals from the pool) if the library allocates; monitoring code inside a running
generation loop must not allocate either, because cudaMalloc / cudaFree can synchronise the device and stall the
sweeps; and a process that merely maps someone else's link buffer has no su_lattice handle, whose creation is where
the library's allocations happen. For them the per-block partial sums sit in a fixed 1 MiB __device__ array inside
libsugauge (limit: 64^4 sites), shared by every call on the device and never cleared.

What is checked: on two calls in a row (a large lattice first, then a smaller one that reuses the front of the same
array while the back still holds the first call's sums, then the first again) the value equals the handle path's
su_plaquette within the reductions' tolerance of tests/test_gpu_parity.py (1e-12 fp64, 1e-6 fp32); that the second
call leaves the device's free memory untouched; and that lattices beyond the limit are refused with a clear text
before anything is launched.

This file is named so that pytest collects it last: with `pytest -x` a failure here hides no other test. It passes
alone in a fresh process (the first call then does the per-device set-up) and after the rest of the suite.
"""
import gc

import pytest

pytestmark = pytest.mark.gpu

TOL_OBS = {"fp64": 1e-12, "fp32": 1e-6}          # the reductions' bar of tests/test_gpu_parity.py
BETA = {2: 2.3, 3: 6.0, 4: 11.0}
# (Nc, precision, recon12, first lattice, second lattice): ragged extents, several hundred blocks in the first call
CASES = [
    (3, "fp64", False, (16, 16, 16, 16), (4, 6, 8, 10)),
    (3, "fp32", True, (8, 12, 16, 10), (4, 6, 8, 10)),
    (2, "fp64", False, (12, 8, 10, 16), (2, 2, 2, 2)),
    (4, "fp32", False, (8, 8, 8, 12), (4, 4, 6, 6)),
]


@pytest.fixture(scope="module")
def su():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1112_4533_b200 as su
    return su


def _thermalised(su, Nc, dims, precision, recon12, seed):
    G = su.Lattice(Nc, dims, precision, recon12)
    G.init_hot(seed)
    G.sweep(BETA[Nc], 1, 1)
    G.synchronize()
    return G


def _static(su, G, out):
    """one call of the no-allocation entry point on G's own link buffer and stream -> host value"""
    su.plaquette_static(G.Nc, G.dims, G.precision, G.recon12, G.buffer.data_ptr(), G.links_bytes, out.data_ptr(),
                        G.stream.cuda_stream, G.device.index or 0)
    G.stream.synchronize()
    return float(out.cpu()[0])


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"su{c[0]}-{c[1]}-{'r12' if c[2] else 'full'}")
def test_two_calls_in_a_row_match_the_handle_path(su, case):
    import torch
    Nc, precision, recon12, dims_a, dims_b = case
    A = _thermalised(su, Nc, dims_a, precision, recon12, 11)
    B = _thermalised(su, Nc, dims_b, precision, recon12, 12)
    out = torch.full((1,), float("nan"), dtype=torch.float64, device=A.device)
    want_a, want_b = A.plaquette(), B.plaquette()
    assert 0.0 < want_a < 1.0 and 0.0 < want_b < 1.0 and want_a != want_b
    tol = TOL_OBS[precision]

    got_a = _static(su, A, out)                  # first call (in a fresh process: also the per-device set-up)
    assert abs(got_a - want_a) < tol
    gc.collect()
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(A.device)[0]
    got_b = _static(su, B, out)                  # second call: fewer blocks, stale sums of the first call behind them
    free_after = torch.cuda.mem_get_info(A.device)[0]
    assert abs(got_b - want_b) < tol
    assert free_after >= free_before             # nothing was allocated on the device
    assert abs(_static(su, A, out) - want_a) < tol
    # same thread -> site mapping, same order of sums as the handle path: the values are the same bits
    assert got_a == want_a and got_b == want_b
    # the links were only read
    assert A.plaquette() == want_a and B.plaquette() == want_b


def test_limit_and_arguments_are_checked_before_any_launch(su):
    import torch
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    fake = out.data_ptr()                        # never dereferenced: every call below is refused first
    assert su.SU_STATIC_MAX_SITES == 64 ** 4
    with pytest.raises(su.SuError) as e:
        su.plaquette_static(3, (66, 64, 64, 64), "fp64", False, fake, 1 << 40, fake)
    assert e.value.status == su.SU_EUNSUPPORTED and "static scratch limit of 16777216 sites" in str(e.value)
    with pytest.raises(su.SuError) as e:
        su.plaquette_static(5, (4, 4, 4, 4), "fp64", False, fake, 1 << 40, fake)
    assert e.value.status == su.SU_EUNSUPPORTED and "Nc = 5" in str(e.value)
    with pytest.raises(su.SuError) as e:
        su.plaquette_static(3, (4, 4, 4, 5), "fp64", False, fake, 1 << 40, fake)
    assert e.value.status == su.SU_EINVAL
    with pytest.raises(su.SuError) as e:
        su.plaquette_static(3, (4, 4, 4, 4), "fp64", False, fake, 16, fake)      # buffer smaller than su_lattice_bytes
    assert e.value.status == su.SU_EINVAL and "su_lattice_bytes" in str(e.value)
    with pytest.raises(su.SuError) as e:
        su.plaquette_static(3, (4, 4, 4, 4), "fp64", False, 0, 1 << 40, fake)
    assert e.value.status == su.SU_EINVAL
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == 0.0            # nothing ran


def test_largest_lattice_the_scratch_admits(su):
    """64^4 sites exactly (SU(2) fp32, 1.07 GB of links): every one of the 131072 scratch slots is used."""
    import torch
    dims = (64, 64, 64, 64)
    G = su.Lattice(2, dims, "fp32")
    G.init_hot(5)
    G.synchronize()
    out = torch.zeros(1, dtype=torch.float64, device=G.device)
    want = G.plaquette()
    assert _static(su, G, out) == want
    assert abs(want) < 1e-3                      # Haar-random links: <ReTr P>/Nc = 0 up to 1/sqrt(6 V Nc^2) noise
