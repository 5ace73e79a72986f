"""Pins for the oracle's geometry, staple, link update, observables, reunitarisation and hot start.

Everything is checked against the paper's definitions restated independently in tests/nphelpers.py
(np.roll / matmul over whole fields), against closed forms, or by brute force on tiny lattices.
"""
import os

import numpy as np
import pytest
from scipy import special

import nphelpers as H
import oracle

DIMS_ANISO = (4, 6, 8, 10)
DIMS_TINY = (2, 2, 2, 2)


def _lat(Nc, dims, links=None, precision="fp64", recon12=False, seed=0):
    L = oracle.OracleLattice(Nc, dims, precision, recon12)
    if links is not None:
        L.import_links(links)
        L.set_rng(seed, 0)
    return L


# ---------------------------------------------------------------- geometry / staple / action

@pytest.mark.parametrize("Nc", [2, 3, 4])
@pytest.mark.parametrize("dims", [DIMS_TINY, DIMS_ANISO, (2, 4, 2, 6)])
def test_plaquette_matches_numpy_definition(Nc, dims):
    rng = np.random.default_rng(10 + Nc)
    links = H.random_links(rng, Nc, dims)
    L = _lat(Nc, dims, links)
    assert abs(L.plaquette() - H.mean_plaquette(links)) < 1e-13
    assert abs(L.polyakov() - H.polyakov(links)) < 1e-13
    assert np.array_equal(L.export_links(), links)          # import/export round trip is exact in fp64


@pytest.mark.parametrize("Nc", [2, 3, 5])
@pytest.mark.parametrize("dims", [DIMS_TINY, DIMS_ANISO])
def test_staple_matches_numpy_and_local_action(Nc, dims):
    """Brute force: the change of the FULL Wilson action (eq 3) when one link is replaced equals
    -(beta/Nc) [ReTr(U' S^dagger) - ReTr(U S^dagger)] with S the oracle's staple (eq 9, reading R1).
    On 2^4, x+nu == x-nu: the degenerate periodic wrap."""
    rng = np.random.default_rng(20 + Nc)
    beta = 2.0 * Nc
    links = H.random_links(rng, Nc, dims)
    L = _lat(Nc, dims, links)
    Lx, Ly, Lz, Lt = dims
    S0 = H.wilson_action(links, beta)
    for trial in range(6):
        x, y, z, t = (int(rng.integers(0, n)) for n in dims)
        if trial == 0:
            x, y, z, t = 0, 0, 0, 0
        if trial == 1:
            x, y, z, t = Lx - 1, Ly - 1, Lz - 1, Lt - 1
        mu = trial % 4
        site = H.site_index(x, y, z, t, dims)
        S = L.staple(site, mu)
        assert np.abs(S - H.staple_field(links, mu)[t, z, y, x]).max() < 1e-13
        U = links[t, z, y, x, mu]
        Unew = H.random_sun(rng, Nc)
        mod = links.copy()
        mod[t, z, y, x, mu] = Unew
        dS_full = H.wilson_action(mod, beta) - S0
        dS_local = -(beta / Nc) * (np.trace(Unew @ H.dag(S)).real - np.trace(U @ H.dag(S)).real)
        assert abs(dS_full - dS_local) < 1e-9 * max(1.0, abs(S0)), (dS_full, dS_local)


def test_staple_footprint_is_18_links(golden_dir):
    """Table 1: a link update loads 19 links = 18 staple links + the link."""
    rows = {}
    with open(os.path.join(golden_dir, "table1_loads.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, reals, phb, reu, plaq = line.split()
            rows[name] = (int(reals), int(phb), int(reu), int(plaq))
    for reals, phb, reu, plaq in rows.values():
        assert phb == 19 * reals and plaq == 24 * reals and reu in (0, 4 * reals)
    Nc, dims = 3, (4, 4, 4, 6)
    rng = np.random.default_rng(3)
    links = H.random_links(rng, Nc, dims)
    L = _lat(Nc, dims, links)
    x, y, z, t, mu = 1, 2, 3, 4, 2
    site = H.site_index(x, y, z, t, dims)
    S0 = L.staple(site, mu)
    touched = []
    Lx, Ly, Lz, Lt = dims
    for tt in range(Lt):
        for zz in range(Lz):
            for yy in range(Ly):
                for xx in range(Lx):
                    if max(min(abs(xx - x), Lx - abs(xx - x)), min(abs(yy - y), Ly - abs(yy - y)),
                           min(abs(zz - z), Lz - abs(zz - z)), min(abs(tt - t), Lt - abs(tt - t))) > 1:
                        continue
                    for nu in range(4):
                        mod = links.copy()
                        mod[tt, zz, yy, xx, nu] = H.random_sun(rng, Nc)
                        L.import_links(mod)
                        if np.abs(L.staple(site, mu) - S0).max() > 1e-9:
                            touched.append((xx, yy, zz, tt, nu))
    assert len(touched) == 18
    assert (x, y, z, t, mu) not in touched


# ---------------------------------------------------------------- link update

def _random_staple_like(rng, Nc):
    return sum(H.random_sun(rng, Nc) for _ in range(6))


@pytest.mark.parametrize("Nc", [2, 3, 4, 6])
def test_overrelaxation_keeps_local_action_and_group(Nc):
    """eq 17 per subgroup: ReTr(U S^dagger) unchanged to 1e-12, U stays in SU(Nc)."""
    rng = np.random.default_rng(30 + Nc)
    for _ in range(20):
        U, S = H.random_sun(rng, Nc), _random_staple_like(rng, Nc)
        W = U @ H.dag(S)
        U1, W1, _ = oracle.update_matrix(U, W, beta=1.0, kind=1)
        assert abs(np.trace(W1).real - np.trace(W).real) < 1e-12 * Nc * 6
        assert np.abs(W1 - U1 @ H.dag(S)).max() < 1e-12            # W is carried along consistently (eq 15)
        assert H.unitarity_defect(U1) < 1e-12 and abs(np.linalg.det(U1) - 1) < 1e-12
        assert np.abs(U1 - U).max() > 1e-3                         # it does move


def test_overrelaxation_su2_is_eq17_and_an_involution():
    rng = np.random.default_rng(31)
    U, S = H.random_sun(rng, 2), _random_staple_like(rng, 2)
    k = np.sqrt(np.linalg.det(S).real)
    U1, _, _ = oracle.update_matrix(U, U @ H.dag(S), beta=1.0, kind=1)
    # eq 17 with Sigma := S^dagger (reading R1): U_new = (S/k) U^dagger (S/k)
    assert np.abs(U1 - (S / k) @ H.dag(U) @ (S / k)).max() < 1e-13
    U2, _, _ = oracle.update_matrix(U1, U1 @ H.dag(S), beta=1.0, kind=1)
    assert np.abs(U2 - U).max() < 1e-13


def test_heatbath_su2_forgets_old_link_and_limits():
    """eq 14: U' = v S/k is independent of U (same RNG counters); beta -> inf gives S/k, the
    minimiser of the single-link action, checked by random search over SU(2)."""
    rng = np.random.default_rng(32)
    S = _random_staple_like(rng, 2)
    k = np.sqrt(np.linalg.det(S).real)
    outs = []
    for _ in range(3):
        U = H.random_sun(rng, 2)
        U1, _, att = oracle.update_matrix(U, U @ H.dag(S), beta=2.3, kind=0, seed=5, c0=17, c1=3)
        assert att[0] >= 1
        outs.append(U1)
    assert np.abs(outs[0] - outs[1]).max() < 1e-13 and np.abs(outs[0] - outs[2]).max() < 1e-13
    U = H.random_sun(rng, 2)
    Uinf, _, _ = oracle.update_matrix(U, U @ H.dag(S), beta=1e12, kind=0, seed=5)
    assert np.abs(Uinf - S / k).max() < 1e-5
    best = max(np.trace(H.random_sun(rng, 2) @ H.dag(S)).real for _ in range(20000))
    assert np.trace((S / k) @ H.dag(S)).real >= best - 1e-12


def test_heatbath_su2_mean_action_is_bessel_ratio():
    """One-link chain with a fixed staple: <ReTr(U S^dagger)>/(2k) = I_2(beta k)/I_1(beta k)
    (moment of eq 13) -- pins alpha = beta k at Nc = 2 through the whole update, not just the sampler."""
    rng = np.random.default_rng(33)
    S = _random_staple_like(rng, 2)
    k = np.sqrt(np.linalg.det(S).real)
    beta = 2.3
    U = H.random_sun(rng, 2)
    vals = []
    for i in range(6000):
        U, _, _ = oracle.update_matrix(U, U @ H.dag(S), beta=beta, kind=0, seed=77, c0=i)
        vals.append(np.trace(U @ H.dag(S)).real / (2 * k))
    vals = np.array(vals)
    exact = special.iv(2, beta * k) / special.iv(1, beta * k)
    assert abs(vals.mean() - exact) < 5 * vals.std() / np.sqrt(len(vals)), (vals.mean(), exact)


@pytest.mark.parametrize("Nc", [3, 4])
def test_subgroup_step_maximises_and_uses_alpha_2betak_over_nc(Nc):
    """For Nc >= 3 the weight of a subgroup element a is exp[(beta/Nc) ReTr(a W)] (step 5 with eq 10;
    reading R3: alpha = 2 beta k / Nc). At beta -> inf the heatbath picks a = u~^dagger, the
    maximiser of ReTr(a W) over that SU(2) subgroup (random search), for every subgroup in turn."""
    rng = np.random.default_rng(34 + Nc)
    U, S = H.random_sun(rng, Nc), _random_staple_like(rng, Nc)
    W = U @ H.dag(S)
    U1, W1, att = oracle.update_matrix(U, W, beta=1e12, kind=0, seed=3)
    assert np.all(att >= 1)
    # replay subgroup by subgroup in numpy: after the first subgroup (0,1) the trace cannot be
    # improved by any element of that subgroup
    Wc = W.copy()
    q = 0
    for i in range(Nc - 1):
        for j in range(i + 1, Nc):
            w = Wc[np.ix_([i, j], [i, j])]
            r = np.array([0.5 * (w[0, 0] + w[1, 1]).real, 0.5 * (w[0, 1] + w[1, 0]).imag,
                          0.5 * (w[0, 1] - w[1, 0]).real, 0.5 * (w[0, 0] - w[1, 1]).imag])
            kk = np.linalg.norm(r)
            a = H.quat_to_su2(np.array([r[0], -r[1], -r[2], -r[3]]) / kk)
            A = np.eye(Nc, dtype=complex)
            A[np.ix_([i, j], [i, j])] = a
            best = np.trace(A @ Wc).real
            for _ in range(300):
                B = np.eye(Nc, dtype=complex)
                B[np.ix_([i, j], [i, j])] = H.random_sun(rng, 2)
                assert np.trace(B @ Wc).real <= best + 1e-12
            # and gain = 2k - Tr(w).real
            assert abs(best - np.trace(Wc).real - (2 * kk - np.trace(w).real)) < 1e-12
            Wc = A @ Wc
            q += 1
    assert np.abs(Wc - W1).max() < 1e-5          # beta=1e12: the oracle's heatbath followed the same path


def test_heatbath_su3_one_link_chain_samples_the_single_link_integral():
    """Repeated pseudo-heatbath of ONE link with a fixed staple must sample
    dP(U) ~ exp[(beta/Nc) ReTr(U S^dagger)] dU (eq 10 generalised, steps 1-5 PAPER.md:106-116).
    The exact mean of ReTr(U S^dagger) is computed by reweighting Haar SU(3) samples. A wrong weight
    (alpha = beta k or beta k / Nc instead of 2 beta k / Nc, reading R3) shifts the mean by many sigma."""
    rng = np.random.default_rng(36)
    Nc, beta = 3, 2.0
    S = _random_staple_like(rng, Nc)
    haar = H.random_sun(rng, Nc, (400000,))
    e = np.trace(haar @ H.dag(S), axis1=1, axis2=2).real
    w = np.exp((beta / Nc) * (e - e.max()))
    exact = (w * e).sum() / w.sum()
    ess = w.sum() ** 2 / (w ** 2).sum()
    err_exact = np.sqrt(((w * (e - exact)) ** 2).sum()) / w.sum()
    assert ess > 2000
    U = H.random_sun(rng, Nc)
    vals = []
    for i in range(12000):
        U, _, _ = oracle.update_matrix(U, U @ H.dag(S), beta=beta, kind=0, seed=11, c0=i)
        vals.append(np.trace(U @ H.dag(S)).real)
    vals = np.array(vals[200:])
    # binned error (the chain has a short autocorrelation)
    bins = vals[: len(vals) // 50 * 50].reshape(-1, 50).mean(axis=1)
    err = bins.std(ddof=1) / np.sqrt(len(bins))
    assert abs(vals.mean() - exact) < 5 * np.hypot(err, err_exact), (vals.mean(), exact, err, err_exact)
    # sensitivity: the same chain run at a weight off by a factor 2 would sit far away
    w2 = np.exp((2 * beta / Nc) * (e - e.max()))
    assert abs((w2 * e).sum() / w2.sum() - exact) > 20 * np.hypot(err, err_exact)


@pytest.mark.parametrize("Nc", [2, 3, 4])
def test_heatbath_keeps_group(Nc):
    rng = np.random.default_rng(37)
    U, S = H.random_sun(rng, Nc), _random_staple_like(rng, Nc)
    U1, W1, att = oracle.update_matrix(U, U @ H.dag(S), beta=2.0 * Nc, kind=0, seed=1)
    assert np.all(att >= 1)
    assert H.unitarity_defect(U1) < 1e-12 and abs(np.linalg.det(U1) - 1) < 1e-12
    assert np.abs(W1 - U1 @ H.dag(S)).max() < 1e-12


# ---------------------------------------------------------------- lattice-level invariants

@pytest.mark.parametrize("Nc", [2, 3, 4, 6])
def test_cold_start_observables_exact(Nc):
    L = oracle.OracleLattice(Nc, (4, 4, 2, 6))
    L.init_cold(1)
    assert L.plaquette() == 1.0
    assert L.polyakov() == 1.0 + 0j


@pytest.mark.parametrize("Nc", [2, 3, 4])
def test_gauge_and_centre_invariance(Nc):
    dims = (4, 2, 4, 6)
    rng = np.random.default_rng(40 + Nc)
    links = H.random_links(rng, Nc, dims)
    L = _lat(Nc, dims, links)
    p0, l0 = L.plaquette(), L.polyakov()
    G = H.random_sun(rng, Nc, (dims[3], dims[2], dims[1], dims[0]))
    L.import_links(H.gauge_transform(links, G))
    assert abs(L.plaquette() - p0) < 1e-12
    assert abs(L.polyakov() - l0) < 1e-12
    # centre transform: all U_3 on one time slice times exp(2 pi i / Nc)
    z = np.exp(2j * np.pi / Nc)
    mod = links.copy()
    mod[2, ..., 3, :, :] *= z
    L.import_links(mod)
    assert abs(L.plaquette() - p0) < 1e-12
    assert abs(L.polyakov() - z * l0) < 1e-12


@pytest.mark.parametrize("Nc", [2, 3, 4])
def test_sweep_keeps_group_and_or_keeps_total_action(Nc):
    dims = (4, 4, 4, 4)
    L = oracle.OracleLattice(Nc, dims)
    L.init_hot(5)
    L.sweep(2.0 * Nc, 1, 1)
    links = L.export_links()
    assert H.unitarity_defect(links) < 1e-12 and H.det_defect(links) < 1e-12
    p0 = L.plaquette()
    L.sweep(2.0 * Nc, 0, 3)               # overrelaxation only: microcanonical
    assert abs(L.plaquette() - p0) < 1e-12
    assert np.abs(L.export_links() - links).max() > 1e-2


def test_sweep_is_the_documented_sequence_of_substeps():
    """Reading R6: passes (all HB, then all OR) x parity 0,1 x mu 0..3; sweep counter bumps after."""
    Nc, dims, beta = 3, (4, 4, 2, 2), 5.5
    A = oracle.OracleLattice(Nc, dims)
    B = oracle.OracleLattice(Nc, dims)
    A.init_hot(9)
    B.init_hot(9)
    A.sweep(beta, 2, 1)
    A.sweep(beta, 1, 0)
    tot = 0
    for pass_, kind in [(0, 0), (1, 0), (0, 1)]:
        for parity in range(2):
            for mu in range(4):
                att = B.substep(beta, kind, pass_, parity, mu, want_attempts=True)
                tot += int(att.sum())
    B.set_rng(9, 1)
    for parity in range(2):
        for mu in range(4):
            tot += int(B.substep(beta, 0, 0, parity, mu, want_attempts=True).sum())
    assert np.array_equal(A.export_links(), B.export_links())
    assert A.counters() == (tot, 0) and B.counters() == (tot, 0)


def test_substep_only_touches_its_parity_and_direction():
    Nc, dims = 2, (4, 4, 4, 4)
    L = oracle.OracleLattice(Nc, dims)
    L.init_hot(2)
    before = L.export_links()
    L.substep(2.3, 0, 0, 1, 2)
    after = L.export_links()
    changed = np.abs(after - before).max(axis=(-1, -2)) > 0
    t, z, y, x = np.indices(changed.shape[:4])
    par = (x + y + z + t) % 2
    for mu in range(4):
        if mu == 2:
            assert changed[..., mu][par == 1].all() and not changed[..., mu][par == 0].any()
        else:
            assert not changed[..., mu].any()


def test_rng_stream_depends_on_every_key_field():
    Nc, dims = 2, (2, 2, 2, 2)
    ref = None
    outs = []
    for seed, sweep, pass_ in [(1, 0, 0), (2, 0, 0), (1, 1, 0), (1, 0, 1), (1 + (1 << 32), 0, 0)]:
        L = oracle.OracleLattice(Nc, dims)
        L.init_cold(0)
        L.set_rng(seed, sweep)
        L.substep(2.3, 0, pass_, 0, 0)
        outs.append(L.export_links())
    for i in range(1, len(outs)):
        assert np.abs(outs[i] - outs[0]).max() > 1e-3


# ---------------------------------------------------------------- hot start / reunitarise / recon12

@pytest.mark.parametrize("Nc", [2, 3, 4])
def test_hot_start_is_haar_like(Nc):
    dims = (6, 6, 6, 6)
    L = oracle.OracleLattice(Nc, dims)
    L.init_hot(1)
    links = L.export_links()
    assert H.unitarity_defect(links) < 1e-13 and H.det_defect(links) < 1e-13
    n = links.shape[0] * links.shape[1] * links.shape[2] * links.shape[3] * 4
    m = links.reshape(n, Nc, Nc)
    # <|U_ij|^2> = 1/Nc, <|Tr U|^2> = 1, <Tr U> = 0
    a2 = (np.abs(m) ** 2).mean(axis=0)
    assert np.abs(a2 - 1 / Nc).max() < 5 * np.sqrt(1.0 / n)
    tr = np.trace(m, axis1=1, axis2=2)
    assert abs((np.abs(tr) ** 2).mean() - 1) < 6 / np.sqrt(n)
    assert abs(tr.mean()) < 5 / np.sqrt(n)
    # <(ReTr U)^2> = 1 for SU(2) (real trace), 1/2 for Nc >= 3
    assert abs((tr.real ** 2).mean() - (1.0 if Nc == 2 else 0.5)) < 6 / np.sqrt(n)
    V = np.prod(dims)
    assert abs(L.plaquette()) < 4 / np.sqrt(6 * V) / (1 if Nc == 2 else np.sqrt(2)) / Nc * 2
    # different seeds and different links differ
    L2 = oracle.OracleLattice(Nc, dims)
    L2.init_hot(2)
    assert np.abs(L2.export_links() - links).max() > 0.1


def _hot_link_restated(Nc, dims, seed, site, mu):
    """One hot-start link written out from the documented keying (SURVEY.md 8(c) "Hot start"; DESIGN.md "RNG keying";
    PAPER.md:164), sharing nothing with the oracle: Philox counter (c0, c1, c2, c3) = (lexicographic site, 0,
    kind 2 << 28 | parity << 19 | mu << 17, block b), key = (seed low, seed high) through the big-integer Philox of
    tests/test_oracle_rng.py (itself pinned by the published known-answer vectors); the four words of block b are two
    Box-Muller pairs (u_a, u_b) -> sqrt(-2 ln u_a) (cos, sin)(2 pi u_b) with u = (w + 1) / 2^32; the Gaussians fill the
    Nc x Nc complex matrix row-major as (re, im); Gram-Schmidt over ROWS with positive normalisation = the QR
    factorisation of the transpose with a positive diagonal (LAPACK, not the oracle's loop); last row times
    conj(det) / |det|. SU(2): the first four Gaussians, normalised, are (a0..a3) of eq 6."""
    from test_oracle_rng import _philox_bigint
    Lx, Ly, Lz, Lt = dims
    x = site % Lx; y = (site // Lx) % Ly; z = (site // (Lx * Ly)) % Lz; t = site // (Lx * Ly * Lz)
    parity = (x + y + z + t) & 1
    key = (seed & 0xFFFFFFFF, seed >> 32)
    ng = 4 if Nc == 2 else 2 * Nc * Nc
    g = []
    for b in range((ng + 3) // 4):
        w = _philox_bigint((site, 0, (2 << 28) | (parity << 19) | (mu << 17), b), key)
        for ua, ub in ((w[0], w[1]), (w[2], w[3])):
            rad = np.sqrt(-2.0 * np.log((ua + 1) / 2.0 ** 32))
            ang = 2.0 * np.pi * ((ub + 1) / 2.0 ** 32)
            g += [rad * np.cos(ang), rad * np.sin(ang)]
    g = np.array(g)
    if Nc == 2:
        a = g[:4] / np.linalg.norm(g[:4])
        return np.array([[a[0] + 1j * a[3], a[2] + 1j * a[1]], [-a[2] + 1j * a[1], a[0] - 1j * a[3]]])
    M = (g[0:ng:2] + 1j * g[1:ng:2]).reshape(Nc, Nc)
    Q, R = np.linalg.qr(M.T)
    d = np.diagonal(R)
    U = (Q * (d / np.abs(d))).T                       # rows of U: the orthonormalised rows of M, positive normalisation
    det = np.linalg.det(U)
    U[Nc - 1] *= np.conj(det) / abs(det)
    return U


@pytest.mark.parametrize("Nc", [2, 3, 4])
@pytest.mark.parametrize("seed", [1, (1 << 40) + 12345])
def test_hot_start_keying_against_an_independent_restatement(Nc, seed):
    """Pins WHICH random numbers make WHICH link (a hot start that reused one matrix for the four
    directions of a site, or one site's matrix for its neighbour, passed every Haar-moment test)."""
    dims = (4, 6, 2, 4)
    L = oracle.OracleLattice(Nc, dims)
    L.init_hot(seed)
    links = L.export_links()                          # [t][z][y][x][mu][row][col]
    flat = links.reshape(-1, 4, Nc, Nc)               # lexicographic site, x fastest
    V = flat.shape[0]
    rng = np.random.default_rng(5)
    sites = sorted(set([0, 1, dims[0], V - 1] + [int(s) for s in rng.integers(0, V, 8)]))
    for site in sites:
        for mu in range(4):
            want = _hot_link_restated(Nc, dims, seed, site, mu)
            assert np.abs(flat[site, mu] - want).max() < 1e-13, (site, mu)
    # independent draws: the four links of a site, and the same direction on neighbouring sites, are different matrices
    for site in sites:
        for mu in range(4):
            for nu in range(mu + 1, 4):
                assert np.abs(flat[site, mu] - flat[site, nu]).max() > 1e-2
            assert np.abs(flat[site, mu] - flat[(site + 1) % V, mu]).max() > 1e-2
    # the seed's high word is part of the key
    if seed >> 32:
        L2 = oracle.OracleLattice(Nc, dims)
        L2.init_hot(seed & 0xFFFFFFFF)
        assert np.abs(L2.export_links() - links).max() > 0.1
    # fp32 lattices hold the same matrices rounded to float (reading R20)
    L32 = oracle.OracleLattice(Nc, dims, "fp32")
    L32.init_hot(seed)
    assert np.abs(L32.export_links() - links).max() < 1e-7


@pytest.mark.parametrize("Nc", [2, 3, 4, 5])
def test_reunitarize(Nc):
    dims = (2, 2, 2, 4)
    rng = np.random.default_rng(50 + Nc)
    links = H.random_links(rng, Nc, dims)
    L = _lat(Nc, dims, links)
    L.reunitarize()
    assert np.abs(L.export_links() - links).max() < 1e-14     # identity on SU(Nc) input
    noisy = links + 1e-6 * (rng.standard_normal(links.shape) + 1j * rng.standard_normal(links.shape))
    L.import_links(noisy)
    L.reunitarize()
    out = L.export_links()
    assert H.unitarity_defect(out) < 1e-13 and H.det_defect(out) < 1e-13
    assert np.abs(out - links).max() < 1e-5
    # first row only rescaled (Gram-Schmidt from the top)
    r0 = noisy[..., 0, :]
    assert np.abs(out[..., 0, :] - r0 / np.linalg.norm(r0, axis=-1, keepdims=True)).max() < 1e-14
    L.reunitarize()
    assert np.abs(L.export_links() - out).max() < 1e-14       # idempotent


def test_recon12_matches_full_storage():
    dims = (4, 4, 2, 4)
    rng = np.random.default_rng(60)
    links = H.random_links(rng, 3, dims)
    F, R = _lat(3, dims, links, seed=4), _lat(3, dims, links, recon12=True, seed=4)
    # the rebuilt third row equals the stored one on exact SU(3) input
    assert np.abs(R.export_links() - links).max() < 1e-15
    for kind in (0, 1):
        F.substep(6.0, kind, 0, 0, 1)
        R.substep(6.0, kind, 0, 0, 1)
    assert np.abs(F.export_links() - R.export_links()).max() < 1e-13
    # a non-unitary third row is discarded by recon12
    bad = links.copy()
    bad[..., 2, :] *= 1.5
    R.import_links(bad)
    assert np.abs(R.export_links() - links).max() < 1e-15


def test_bad_arguments_are_refused():
    for dims in [(3, 4, 4, 4), (4, 4, 4, 0), (4, 4, 1, 4)]:
        with pytest.raises(oracle.OracleError):
            oracle.OracleLattice(3, dims)
    with pytest.raises(oracle.OracleError):
        oracle.OracleLattice(1, (4, 4, 4, 4))
    with pytest.raises(oracle.OracleError):
        oracle.OracleLattice(4, (4, 4, 4, 4), recon12=True)
    L = oracle.OracleLattice(3, (2, 2, 2, 2))
    with pytest.raises(oracle.OracleError):
        L.sweep(6.0, 1, 1)                # not initialised
    L.init_cold(0)
    with pytest.raises(oracle.OracleError):
        L.sweep(float("nan"), 1, 1)
    with pytest.raises(oracle.OracleError):
        L.substep(6.0, 2, 0, 0, 0)
