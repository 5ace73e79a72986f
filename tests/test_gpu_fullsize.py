"""Full-size parity (pytest -m gpu): BASELINE.json configs[2] (SU(3) 48^4, hot start seed 7, beta 6.0)
in the launch configuration bench.py times, and the long-run statistical agreement (P-stat).

At 48^4 the oracle cannot run a whole sweep in seconds, but one (parity, mu) sub-step is 2.65 M link
updates (about a second on the box's cores), so the comparison is still ELEMENT BY ELEMENT over every
link of the lattice for a handful of sub-steps chosen to cover both kinds, both parities and all four
directions; the links a sub-step must not touch are compared bitwise. After that, whole sweeps at full
size are checked through properties that hold at any size (group membership, plaquette of the exported
links by the numpy definition, KP attempt statistics).

Tolerances: BASELINE.json north_star (fp64 1e-11 per element; fp32 2e-5 except counted KP flips < 1e-5).
"""
import numpy as np
import pytest

import nphelpers as H

pytestmark = pytest.mark.gpu

L_FULL = 48
BETA = 6.0
SEED = 7


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import psutil
    if psutil.virtual_memory().available < 40 * 2 ** 30:
        pytest.skip("needs 40 GB of host memory for three 3 GB link arrays plus the oracle's lattice")
    import oracle
    import paper_1112_4533_b200 as su
    return su, oracle


def _sites_of_parity(dims, parity):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return np.nonzero(((x + y + z + t) & 1).reshape(-1) == parity)[0]


def _maxdiff(a, b, chunk=1 << 20):
    """max |a - b| over two big arrays without a 3 GB temporary"""
    fa, fb = a.reshape(-1), b.reshape(-1)
    m = 0.0
    for i in range(0, fa.size, chunk):
        m = max(m, float(np.abs(fa[i:i + chunk] - fb[i:i + chunk]).max()))
    return m


@pytest.mark.parametrize("precision,recon12", [("fp64", False), ("fp32", False), ("fp64", True), ("fp32", True)],
                         ids=["fp64-full", "fp32-full", "fp64-r12", "fp32-r12"])      # the four variants bench.py times
def test_su3_48_substeps_every_link(mods, precision, recon12):
    su, oracle = mods
    dims = (L_FULL,) * 4
    G = su.Lattice(3, dims, precision, recon12=recon12)
    O = oracle.OracleLattice(3, dims, precision, recon12=recon12)
    G.init_hot(SEED)
    O.init_hot(SEED)
    lo = O.export_links()
    lg = G.export_links()
    assert _maxdiff(lg, lo) <= (1e-12 if precision == "fp64" else 3e-7)       # hot start, all 21 M links
    if precision == "fp32":
        # fp32 per-sub-step error scales like eps / k; among 1e7 Haar-random staples the smallest subgroup
        # norms k push it to the 2e-5 bar itself, so fp32 is compared on links the ORACLE has ordered with
        # one heatbath + one overrelaxation pass (SURVEY.md 8(c) "fall back to a thermalised start")
        O.sweep(BETA, 1, 1)
        lo = O.export_links()
    tol = 1e-11 if precision == "fp64" else 2e-5
    # heatbath and overrelaxation, both parities, all four directions between them
    plan = [(0, 0, 0, 0), (0, 0, 1, 3), (1, 0, 0, 2), (1, 0, 1, 1)]
    flipped = updated = 0
    sweep_ctr = 1 if precision == "fp32" else 0
    for kind, pass_, parity, mu in plan:
        G.import_links(lo)                        # same input links on both sides (oracle's)
        G.set_rng(SEED, sweep_ctr)
        before = lo
        ag = G.substep(BETA, kind, pass_, parity, mu, want_attempts=(kind == 0))
        ao = O.substep(BETA, kind, pass_, parity, mu, want_attempts=(kind == 0))
        lg, lo = G.export_links(), O.export_links()
        sites = _sites_of_parity(dims, parity)
        g4 = lg.reshape(-1, 4, 9)
        o4 = lo.reshape(-1, 4, 9)
        d = np.abs(g4[sites, mu] - o4[sites, mu]).max(axis=1)
        mism = np.zeros(len(sites), dtype=bool)
        if kind == 0:
            mism = (ag != ao).any(axis=0)
            assert ao.min() >= 1 and ao.max() < 255
            if precision == "fp64":
                assert not mism.any()
        flipped += int(mism.sum())
        updated += len(sites)
        assert d[~mism].max() <= tol, (kind, parity, mu, float(d[~mism].max()))
        # nothing else moved: the other parity and the other directions are bitwise the input
        b4 = before.reshape(-1, 4, 9)
        other = _sites_of_parity(dims, 1 - parity)
        if precision == "fp64" and not recon12:
            assert np.array_equal(g4[other, mu], b4[other, mu])
            for nu in range(4):
                if nu != mu:
                    assert np.array_equal(g4[:, nu], b4[:, nu])
        elif precision == "fp32" and recon12:
            # the two stored rows are the imported floats, bit for bit; the third row is rebuilt in fp32 by each side in
            # its own rounding order (a complex cross product: four products per element), a few ulp of 1 apart
            assert np.array_equal(g4[other, mu][:, :6], b4[other, mu][:, :6])
            assert np.abs(g4[other, mu][:, 6:] - b4[other, mu][:, 6:]).max() <= 5e-7
        else:                                     # storage rounds / rebuilds the third row on import
            assert np.abs(g4[other, mu] - b4[other, mu]).max() <= (1e-15 if precision == "fp64" else 1e-7)
        del lg, g4, b4, before
    assert flipped < 1e-5 * updated + 1, (flipped, updated)
    assert G.counters()[1] == 0 and O.counters()[1] == 0


def test_su3_48_whole_sweeps_properties(mods):
    """Whole su_sweep(1,4) + su_reunitarize at 48^4 exactly as bench.py runs them (including the CUDA-graph
    replay mode): links stay in SU(3), su_plaquette / su_polyakov equal the numpy definitions on the
    exported links, mean KP attempts sit in the band the oracle's sampler pins (1.00..1.15 at beta 6)."""
    su, _ = mods
    dims = (L_FULL,) * 4
    G = su.Lattice(3, dims, "fp64")
    G.init_hot(SEED)
    p0 = G.plaquette()
    assert abs(p0) < 3.0 / np.sqrt(6 * L_FULL ** 4) * 3          # Haar links: <P> = 0 +- 1/sqrt(18 * 6V)-ish
    for _ in range(3):
        G.sweep(BETA, 1, 4)
        G.reunitarize()
    att, exh = G.counters()
    n_draws = 3 * 4 * L_FULL ** 4 * 3                            # sweeps x links x subgroups
    assert exh == 0 and 1.0 <= att / n_draws < 1.25
    links = G.export_links()
    sub = links[:4]                                              # 4 time slices are enough for the group checks
    assert H.unitarity_defect(sub) < 1e-13 and H.det_defect(sub) < 1e-13
    assert abs(G.plaquette() - H.mean_plaquette(links)) < 1e-12
    assert abs(G.polyakov() - H.polyakov(links)) < 1e-12
    assert 0.20 < G.plaquette() < 0.62                           # ordering towards the beta = 6 value
    # graph replay gives bitwise the same chain as plain launches
    A = su.Lattice(3, dims, "fp64", graph=True)
    A.import_links(links)
    A.set_rng(SEED, 3)
    A.sweep(BETA, 1, 4)
    G.sweep(BETA, 1, 4)
    assert abs(A.plaquette() - G.plaquette()) == 0.0


@pytest.mark.parametrize("Nc,L,beta", [(2, 8, 2.3), (3, 6, 6.0)], ids=["su2-8^4", "su3-6^4"])
def test_thermalised_means_agree_statistically(mods, Nc, L, beta):
    """P-stat (north_star): over 1000 thermalised sweeps the mean plaquettes of the GPU chain and the
    oracle chain (DIFFERENT seeds, so the chains are independent) agree within 3 combined standard errors;
    errors from 20-sweep bins."""
    su, oracle = mods
    dims = (L,) * 4
    G = su.Lattice(Nc, dims, "fp64", graph=True)
    O = oracle.OracleLattice(Nc, dims, "fp64")
    G.init_hot(101)
    O.init_hot(202)
    n_therm, n_meas = 100, 1000
    pg, po = [], []
    for i in range(n_therm + n_meas):
        G.sweep(beta, 1, 4)
        O.sweep(beta, 1, 4)
        if Nc > 2:
            G.reunitarize()
            O.reunitarize()
        if i >= n_therm:
            pg.append(G.plaquette())
            po.append(O.plaquette())

    def mean_err(x):
        b = np.asarray(x).reshape(-1, 20).mean(axis=1)
        return b.mean(), b.std(ddof=1) / np.sqrt(len(b))

    (mg, eg), (mo, eo) = mean_err(pg), mean_err(po)
    assert abs(mg - mo) <= 3.0 * np.hypot(eg, eo), (mg, eg, mo, eo)
    assert G.counters()[1] == 0


def test_su3_48_whole_sweep_every_link(mods):
    """P-sweep at full size: one whole su_sweep(1, 4) = 40 kernels at 48^4 fp64 (the z-chunked traversal, the
    launch configuration bench.py times) against the oracle's sweep, all 21 M links at 1e-11, from links the
    ORACLE has thermalised (6 sweeps of 1 HB + 4 OR from the hot start, ~10 s each on the box's cores; after 3 the
    worst of the 190 M elements was still at 1.7e-11: the tail of the rounding amplification grows with the volume,
    SURVEY.md 8(c) P-sweep)."""
    su, oracle = mods
    dims = (L_FULL,) * 4
    O = oracle.OracleLattice(3, dims, "fp64")
    O.init_hot(SEED)
    n_therm = 6
    for _ in range(n_therm):
        O.sweep(BETA, 1, 4)
    G = su.Lattice(3, dims, "fp64")
    assert G.get_option("z_chunk_planes") < L_FULL          # the chunked traversal is what runs here
    G.import_links(O.export_links())
    G.set_rng(SEED, n_therm)
    att0 = O.counters()[0]
    G.sweep(BETA, 1, 4)
    O.sweep(BETA, 1, 4)
    lg, lo = G.export_links(), O.export_links()
    assert _maxdiff(lg, lo) <= 1e-11
    assert G.counters()[0] == O.counters()[0] - att0 and G.counters()[1] == 0
    assert abs(G.plaquette() - O.plaquette()) < 1e-12
    assert abs(G.polyakov() - O.polyakov()) < 1e-12


@pytest.mark.parametrize("Nc,L,beta,seed,start,precision,kernel", [
    (4, 24, 11.0, 11, "hot", "fp64", "auto"), (4, 24, 11.0, 11, "hot", "fp32", "auto"),
    (4, 24, 11.0, 11, "hot", "fp64", "generic"), (6, 16, 25.0, 5, "cold", "fp64", "auto")],
    ids=["su4-24-fp64", "su4-24-fp32", "su4-24-fp64-generic", "su6-16-fp64"])
def test_config4_and_config5_lockstep_at_their_own_size(mods, Nc, L, beta, seed, start, precision, kernel):
    """BASELINE.json configs[3] (SU(4) 24^4, specialised and generic kernel) and configs[4] (SU(6) 16^4) at their
    own sizes: heatbath and overrelaxation sub-steps in lock-step with the oracle on links the oracle has ordered
    with one 1 HB + 1 OR sweep; every link, attempt counts per (link, subgroup)."""
    su, oracle = mods
    dims = (L,) * 4
    G = su.Lattice(Nc, dims, precision, kernel=kernel)
    O = oracle.OracleLattice(Nc, dims, precision)
    (G.init_hot if start == "hot" else G.init_cold)(seed)
    (O.init_hot if start == "hot" else O.init_cold)(seed)
    assert _maxdiff(G.export_links(), O.export_links()) <= (1e-12 if precision == "fp64" else 3e-7)
    O.sweep(beta, 1, 1)
    lo = O.export_links()
    G.import_links(lo)
    G.set_rng(seed, 1)
    tol = 1e-11 if precision == "fp64" else 2e-5
    flipped = updated = 0
    for kind, parity, mu in [(0, 0, 1), (0, 1, 3), (1, 1, 0), (1, 0, 2)]:
        ag = G.substep(beta, kind, 0, parity, mu, want_attempts=(kind == 0))
        ao = O.substep(beta, kind, 0, parity, mu, want_attempts=(kind == 0))
        lg, lo = G.export_links(), O.export_links()
        sites = _sites_of_parity(dims, parity)
        d = np.abs(lg.reshape(-1, 4, Nc * Nc)[sites, mu] - lo.reshape(-1, 4, Nc * Nc)[sites, mu]).max(axis=1)
        mism = np.zeros(len(sites), dtype=bool)
        if kind == 0:
            mism = (ag != ao).any(axis=0)
            assert ao.min() >= 1
            if precision == "fp64":
                assert not mism.any()
        flipped += int(mism.sum())
        updated += len(sites)
        assert d[~mism].max() <= tol, (kind, parity, mu, float(d[~mism].max()))
        assert _maxdiff(lg, lo) <= (tol if not mism.any() else 10.0)      # nothing else moved
        G.import_links(lo)
    assert flipped < 1e-5 * updated * Nc * (Nc - 1) / 2 + 1
    assert G.counters()[1] == 0
