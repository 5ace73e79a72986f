"""t-slab decomposition on ONE GPU (pytest -m gpu): a lattice cut
into 1, 2 or 4 slabs, all driven by this process on one stream, must reproduce the single-lattice chain BITWISE
(same kernels, same global Philox site index, halos pushed by the update kernel itself), and hence agree with
the oracle like the single lattice does."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DIMS = (8, 4, 8, 8)          # Lx Ly Lz / 2 = 128 sites per slice and parity = 4 tiles
BETA = {2: 2.3, 3: 6.0, 4: 11.0, 6: 25.0}


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import oracle
    import paper_1112_4533_b200 as su
    from paper_1112_4533_b200 import slab
    return su, slab, oracle


@pytest.mark.parametrize("Nc,precision,recon12,kernel", [
    (2, "fp64", False, "auto"), (3, "fp64", False, "auto"), (3, "fp32", True, "auto"), (4, "fp32", False, "auto"),
    (3, "fp64", False, "generic"), (6, "fp64", False, "auto")])
@pytest.mark.parametrize("n_slabs", [1, 2, 4])
def test_slabs_reproduce_the_single_lattice_bitwise(mods, Nc, precision, recon12, kernel, n_slabs):
    su, slab, _ = mods
    A = su.Lattice(Nc, DIMS, precision, recon12, kernel)
    B = slab.SlabGroup(Nc, DIMS, n_slabs, precision, recon12, kernel)
    A.init_hot(5)
    B.init_hot(5)
    assert np.array_equal(A.export_links(), B.export_links())
    for _ in range(2):
        A.sweep(BETA[Nc], 1, 2)
        B.sweep(BETA[Nc], 1, 2)
        if Nc > 2:
            A.reunitarize()
            B.reunitarize()
    assert np.array_equal(A.export_links(), B.export_links())
    assert abs(A.plaquette() - B.plaquette()) < 1e-13
    assert A.counters() == B.counters()
    B.close()


def test_slabs_import_and_halo_push_then_match_the_oracle(mods):
    su, slab, oracle = mods
    O = oracle.OracleLattice(3, DIMS, "fp64")
    O.init_hot(9)
    for _ in range(3):
        O.sweep(6.0, 1, 4)
    B = slab.SlabGroup(3, DIMS, 2, "fp64")
    B.import_links(O.export_links())
    B.set_rng(9, 3)
    B.sweep(6.0, 1, 4)
    O.sweep(6.0, 1, 4)
    assert np.abs(B.export_links() - O.export_links()).max() <= 1e-11
    assert abs(B.plaquette() - O.plaquette()) < 1e-12
    B.close()


def test_thinnest_slabs_and_two_streams(mods):
    """Lt_local = 2 (every owned slice is both first and last: both halos pushed by every thread), and two
    independent lattices advancing on two different CUDA streams at once."""
    import torch
    su, slab, _ = mods
    A = su.Lattice(3, DIMS, "fp64")
    B = slab.SlabGroup(3, DIMS, 4, "fp64")            # 8 time slices -> 4 slabs of 2
    A.init_hot(2)
    B.init_hot(2)
    A.sweep(6.0, 1, 1)
    B.sweep(6.0, 1, 1)
    assert np.array_equal(A.export_links(), B.export_links())
    B.close()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s1):
        X = su.Lattice(3, DIMS, "fp64")
    with torch.cuda.stream(s2):
        Y = su.Lattice(3, DIMS, "fp64")
    X.init_hot(2)
    Y.init_hot(2)
    for _ in range(3):
        X.sweep(6.0, 1, 1)
        Y.sweep(6.0, 1, 1)
    A.sweep(6.0, 1, 1)
    A.sweep(6.0, 1, 1)
    ref = A.export_links()
    assert np.array_equal(X.export_links(), ref) and np.array_equal(Y.export_links(), ref)


def test_slab_argument_checks(mods):
    su, slab, _ = mods
    with pytest.raises(ValueError):
        slab.slab_starts(8, 3)
    with pytest.raises(su.SuError):                       # odd slab length
        su.Lattice(3, DIMS, slab=(0, 3))
    with pytest.raises(su.SuError) as e:                  # 4*6*8/2 = 96 sites per slice and parity: not whole tiles... 96 = 3 tiles, fine; 4*6*6/2 = 72 is not
        su.Lattice(3, (4, 6, 6, 8), slab=(0, 4))
    assert e.value.status == su.SU_EUNSUPPORTED
    G = su.Lattice(3, DIMS, slab=(0, 4))
    G.init_cold(1)
    with pytest.raises(su.SuError) as e:                  # peers not set
        G.substep(6.0, 1, 0, 0, 0)
    assert e.value.status == su.SU_ESTATE
    H = su.Lattice(3, DIMS, slab=(4, 4))
    H.init_cold(1)
    G.set_peers(H.links_ptr()[0], H.links_ptr()[0])
    H.set_peers(G.links_ptr()[0], G.links_ptr()[0])
    with pytest.raises(su.SuError) as e:                  # one slab of two cannot sweep alone
        G.sweep(6.0, 1, 4)
    assert e.value.status == su.SU_ESTATE
    with pytest.raises(su.SuError) as e:
        G.polyakov()
    assert e.value.status == su.SU_EUNSUPPORTED
    assert abs(G.plaquette() + H.plaquette() - 1.0) < 1e-15
