"""The runtime-Nc warp-per-link path (csrc/big_kernels.cu; 9 <= Nc <= 32)
against the oracle (pytest -m gpu): every row of SURVEY.md 8(a) - hot / cold start, import / export, plaquette,
Polyakov loop, heatbath and overrelaxation sub-steps in lock-step (links and Kennedy-Pendleton attempt counts per
link and subgroup), reunitarisation, a whole sweep, and the slab decomposition - at Nc = 9, 12, 16 (the paper's
double-precision limit), 17 and 32 (its single-precision limit)."""
import numpy as np
import pytest

import nphelpers as H

pytestmark = pytest.mark.gpu

DIMS = (2, 4, 2, 6)           # 96 sites: Lx/2 = 1, ragged against every block shape
CASES = [(9, "fp64"), (12, "fp64"), (16, "fp64"), (16, "fp32"), (17, "fp32"), (32, "fp32"), (24, "fp64")]
TOL = {"fp64": 1e-11, "fp32": 2e-5}


def _beta(Nc):
    return 0.7 * Nc * Nc          # 't Hooft scaling of the paper's beta = 6.2 at Nc = 3


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import oracle
    import paper_1112_4533_b200 as su
    return su, oracle


def _sites_of_parity(dims, parity):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return np.nonzero(((x + y + z + t) & 1).reshape(-1) == parity)[0]


@pytest.mark.parametrize("Nc,precision", CASES)
def test_big_nc_every_step_against_the_oracle(mods, Nc, precision):
    su, oracle = mods
    G = su.Lattice(Nc, DIMS, precision)
    O = oracle.OracleLattice(Nc, DIMS, precision)
    tol = TOL[precision]
    # cold start
    G.init_cold(1)
    assert G.plaquette() == 1.0 and abs(G.polyakov() - 1.0) < 1e-15
    # hot start (computed in double on both sides)
    G.init_hot(3)
    O.init_hot(3)
    lg, lo = G.export_links(), O.export_links()
    assert np.abs(lg - lo).max() <= (1e-11 if precision == "fp64" else 3e-7)
    assert H.unitarity_defect(lg) < (1e-12 if precision == "fp64" else 1e-5)
    assert H.det_defect(lg) < (1e-11 if precision == "fp64" else 1e-4)
    # import / export, observables
    rng = np.random.default_rng(Nc)
    links = H.random_links(rng, Nc, DIMS)
    G.import_links(links)
    O.import_links(links)
    if precision == "fp64":
        assert np.array_equal(G.export_links(), links)
    tobs = 1e-12 if precision == "fp64" else 1e-6
    assert abs(G.plaquette() - O.plaquette()) < tobs and abs(G.polyakov() - O.polyakov()) < tobs
    if precision == "fp64":
        assert abs(G.plaquette() - H.mean_plaquette(links)) < 1e-12 and abs(G.polyakov() - H.polyakov(links)) < 1e-12
    # lock-step sub-steps on links the oracle has ordered a little (cold start + one sweep)
    O.init_cold(5)
    O.sweep(_beta(Nc), 1, 1)
    lo = O.export_links()
    G.import_links(lo)
    G.set_rng(5, 1)
    flipped = 0
    for kind, pass_, parity, mu in [(0, 0, 0, 0), (0, 2, 1, 3), (1, 0, 1, 1), (1, 0, 0, 2), (0, 0, 1, 2)]:
        ag = G.substep(_beta(Nc), kind, pass_, parity, mu, want_attempts=True)
        ao = O.substep(_beta(Nc), kind, pass_, parity, mu, want_attempts=True)
        lg, lo = G.export_links(), O.export_links()
        d = np.abs(lg - lo).reshape(-1, 4, Nc * Nc).max(axis=2)
        bad = np.zeros(O.V, dtype=bool)
        if kind == 0:
            assert ao.min() >= 1
            mism = (ag != ao).any(axis=0)
            bad[_sites_of_parity(DIMS, parity)[mism]] = True
            if precision == "fp64":
                assert not mism.any()
            flipped += int(mism.sum())
        assert d[~bad].max() <= tol, (kind, parity, mu, float(d[~bad].max()))
        G.import_links(lo)
    assert flipped <= 1
    # reunitarisation of slightly damaged links
    noisy = lo + 1e-6 * (rng.standard_normal(lo.shape) + 1j * rng.standard_normal(lo.shape))
    G.import_links(noisy)
    O.import_links(noisy)
    G.reunitarize()
    O.reunitarize()
    lg, lo = G.export_links(), O.export_links()
    assert np.abs(lg - lo).max() <= (1e-11 if precision == "fp64" else 2e-5)
    assert H.unitarity_defect(lg) < (1e-12 if precision == "fp64" else 1e-5)
    assert G.counters()[1] == 0


@pytest.mark.parametrize("Nc", [9, 16])
def test_big_nc_whole_sweep_and_slabs(mods, Nc):
    su, oracle = mods
    from paper_1112_4533_b200.slab import SlabGroup
    dims = (8, 2, 4, 4)                                   # Lx Ly Lz / 2 = 32: whole tiles per time slice (slab mode)
    O = oracle.OracleLattice(Nc, dims, "fp64")
    O.init_cold(2)
    for _ in range(3):
        O.sweep(_beta(Nc), 1, 2)
        O.reunitarize()
    start = O.export_links()
    G = su.Lattice(Nc, dims, "fp64")
    G.import_links(start)
    G.set_rng(2, 3)
    S = SlabGroup(Nc, dims, 2, "fp64")
    S.import_links(start)
    S.set_rng(2, 3)
    att0 = O.counters()[0]
    G.sweep(_beta(Nc), 1, 2)
    S.sweep(_beta(Nc), 1, 2)
    O.sweep(_beta(Nc), 1, 2)
    assert np.abs(G.export_links() - O.export_links()).max() <= 1e-11
    assert np.array_equal(G.export_links(), S.export_links())
    assert G.counters()[0] == O.counters()[0] - att0
    assert abs(G.plaquette() - O.plaquette()) < 1e-12 and abs(S.plaquette() - G.plaquette()) < 1e-13
    S.close()


def test_nc_limits(mods):
    su, _ = mods
    with pytest.raises(su.SuError) as e:
        su.Lattice(33, (2, 2, 2, 2))
    assert e.value.status == su.SU_EUNSUPPORTED
    G = su.Lattice(32, (2, 2, 2, 2), "fp32")
    G.init_cold(0)
    G.sweep(_beta(32), 1, 1)
    assert abs(G.plaquette() - 1.0) < 0.5
