"""Fused multi-sub-step launches (su_set_option "fuse"; csrc/fused_schedule.h) on the GPU
(pytest -m gpu): g = 2, 4 or 8 consecutive sub-steps of a pass in one launch must leave BITWISE the links, the KP
attempt totals and the observables of the one-launch-per-sub-step sweep - every update sees exactly the links it
sees there (tests/test_fused_schedule.py proves the schedule; this observes it) - and therefore match the oracle
like the plain sweep does."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DIMS_ANISO = (4, 6, 8, 10)
BETA = {2: 2.3, 3: 6.0, 4: 11.0, 6: 25.0}


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import oracle
    import paper_1112_4533_b200 as su
    return su, oracle


VARIANTS = [(3, "fp64", False, "auto"), (3, "fp32", False, "auto"), (3, "fp64", True, "auto"), (3, "fp32", True, "auto"),
            (4, "fp64", False, "auto"), (4, "fp32", False, "auto"), (2, "fp64", False, "generic"), (3, "fp32", True, "generic")]


def _ids(v):
    return f"su{v[0]}-{v[1]}-{'r12' if v[2] else 'full'}-{v[3]}"


@pytest.mark.parametrize("v", VARIANTS, ids=_ids)
@pytest.mark.parametrize("g", [2, 4, 8])
@pytest.mark.parametrize("dims", [DIMS_ANISO, (2, 2, 2, 2), (8, 8, 4, 6)], ids=["4x6x8x10", "2^4", "8x8x4x6"])
def test_fused_sweep_is_bitwise_the_plain_sweep(mods, v, g, dims):
    su, _ = mods
    Nc, precision, recon12, kernel = v
    A = su.Lattice(Nc, dims, precision, recon12, kernel)
    B = su.Lattice(Nc, dims, precision, recon12, kernel)
    B.set_option("fuse", g)
    assert B.get_option("fuse") == g and B.get_option("fuse_effective") == g and A.get_option("fuse_effective") == 1
    A.init_hot(5)
    B.init_hot(5)
    for _ in range(3):
        A.sweep(BETA[Nc], 2, 3)
        B.sweep(BETA[Nc], 2, 3)
        if Nc > 2:
            A.reunitarize()
            B.reunitarize()
    B.synchronize()
    assert np.array_equal(A.export_links(), B.export_links())
    assert A.counters() == B.counters() and A.counters()[1] == 0
    assert A.plaquette() == B.plaquette()
    assert B.launch_count() < A.launch_count()


@pytest.mark.parametrize("kw", [dict(fuse_cell_planes=1), dict(fuse_cell_planes=2, fuse_chunk_planes=2), dict(fuse_chunk_planes=4, fuse_margin=1),
                                dict(fuse_margin=50), dict(fuse_cell_planes=8)])
@pytest.mark.parametrize("g", [2, 8])
def test_fused_schedule_shape_knobs_do_not_change_results(mods, kw, g):
    su, _ = mods
    A = su.Lattice(3, DIMS_ANISO, "fp64")
    B = su.Lattice(3, DIMS_ANISO, "fp64")
    B.set_option("fuse", g)
    for k, val in kw.items():
        B.set_option(k, val)
    A.init_hot(2)
    B.init_hot(2)
    for _ in range(2):
        A.sweep(6.0, 1, 4)
        B.sweep(6.0, 1, 4)
    assert np.array_equal(A.export_links(), B.export_links())
    with pytest.raises(su.SuError):
        B.set_option("fuse", 3)
    with pytest.raises(su.SuError):
        B.set_option("fuse_cell_planes", 3)


def test_fused_graph_replay_and_option_changes(mods):
    su, _ = mods
    A = su.Lattice(3, DIMS_ANISO, "fp64")
    B = su.Lattice(3, DIMS_ANISO, "fp64", graph=True)
    B.set_option("fuse", 4)
    A.init_hot(3)
    B.init_hot(3)
    for i in range(4):
        A.sweep(6.0, 1, 2)
        B.sweep(6.0, 1, 2)
        if i == 1:
            B.set_option("fuse", 8)                     # drops the captured graphs and the tables
    assert np.array_equal(A.export_links(), B.export_links())
    B.set_option("fuse", 1)
    A.sweep(6.0, 1, 1)
    B.sweep(6.0, 1, 1)
    assert np.array_equal(A.export_links(), B.export_links())


@pytest.mark.parametrize("g", [2, 4, 8])
def test_fused_sweep_matches_the_oracle(mods, g):
    su, oracle = mods
    O = oracle.OracleLattice(3, DIMS_ANISO, "fp64")
    O.init_hot(11)
    for _ in range(6):
        O.sweep(6.0, 1, 4)
    G = su.Lattice(3, DIMS_ANISO, "fp64")
    G.set_option("fuse", g)
    G.import_links(O.export_links())
    G.set_rng(11, 6)
    G.sweep(6.0, 1, 4)
    O.sweep(6.0, 1, 4)
    assert np.abs(G.export_links() - O.export_links()).max() <= 1e-11
    assert abs(G.plaquette() - O.plaquette()) < 1e-12


def test_fusion_is_ignored_where_it_does_not_apply(mods):
    su, _ = mods
    from paper_1112_4533_b200.slab import SlabGroup
    G = su.Lattice(6, (4, 4, 4, 4), "fp64")            # row-per-lane generic kernel: no fused form
    G.set_option("fuse", 4)
    assert G.get_option("fuse_effective") == 1
    G.init_cold(1)
    G.sweep(25.0, 1, 1)
    S = SlabGroup(3, (8, 4, 8, 8), 1, "fp64")
    S.slabs[0].set_option("fuse", 4)
    assert S.slabs[0].get_option("fuse_effective") == 1
    S.close()


@pytest.mark.parametrize("precision,g", [("fp64", 2), ("fp64", 8), ("fp32", 4)])
def test_fused_sweep_at_full_size_is_bitwise_the_plain_sweep(mods, precision, g):
    """48^4 (the z-chunked schedule, 9 tiles per cell, ~21 000 tickets per launch): two whole sweeps."""
    su, _ = mods
    dims = (48,) * 4
    A = su.Lattice(3, dims, precision)
    A.init_hot(7)
    for _ in range(2):
        A.sweep(6.0, 1, 4)
    ref = A.export_links()
    ca = A.counters()
    pa = A.plaquette()
    A.close()
    B = su.Lattice(3, dims, precision)
    B.set_option("fuse", g)
    B.init_hot(7)
    for _ in range(2):
        B.sweep(6.0, 1, 4)
    B.synchronize()
    assert B.counters() == ca and B.plaquette() == pa
    out = B.export_links()
    for i in range(0, 48, 8):
        assert np.array_equal(out[i:i + 8], ref[i:i + 8])


def test_a_dependency_wait_that_gives_up_stores_nothing_more_and_the_handle_recovers(mods):
    """su_set_option "fuse_wait_ns" = 0: a wait that does not find its dependencies complete at its first poll gives
    up, exactly what a wait beyond the 10 s default does. The launch must then be reported (SU_ECUDA at the next
    synchronising call), the handle must refuse to go on with the half-updated links (SU_ESTATE), and after a new
    import with the default limit the fused sweep must again be bitwise the plain one (tables rebuilt and zeroed)."""
    su, _ = mods
    dims = (16, 16, 16, 16)
    A = su.Lattice(3, dims, "fp64")
    A.init_hot(21)
    start = A.export_links()
    A.sweep(6.0, 1, 2)
    want = A.export_links()

    B = su.Lattice(3, dims, "fp64")
    B.set_option("fuse", 8)
    B.set_option("fuse_margin", 1)                   # dependent tiles as close together as the schedule allows: blocks do wait
    default_ns = B.get_option("fuse_wait_ns")
    assert default_ns == 10_000_000_000
    B.set_option("fuse_wait_ns", 0)
    tripped = False
    for _ in range(8):                               # in practice the first sweep already has a block that has to wait
        B.import_links(start)
        B.set_rng(21, 0)
        B.sweep(6.0, 1, 2)
        try:
            B.synchronize()
        except su.SuError as e:
            assert e.status == su.SU_ECUDA and "dependency wait timed out" in str(e)
            tripped = True
            break
    assert tripped, "no fused block ever had to wait: the give-up path was not exercised"
    with pytest.raises(su.SuError) as e:
        B.sweep(6.0, 1, 2)
    assert e.value.status == su.SU_ESTATE
    with pytest.raises(su.SuError) as e:
        B.plaquette()
    assert e.value.status == su.SU_ESTATE
    B.set_option("fuse_wait_ns", default_ns)
    B.import_links(start)
    B.set_rng(21, 0)
    B.sweep(6.0, 1, 2)
    B.synchronize()
    assert np.array_equal(B.export_links(), want)
