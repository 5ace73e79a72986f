"""The ticket table of the fused multi-sub-step launches (csrc/fused_schedule.cu, fused_schedule.h), proved on small
lattices without a GPU through the host-only hooks su_fused_schedule_debug / su_fused_dep_debug:

  1. every tile of every stage is handed out exactly once, and together the tiles of a stage are the V/2 sites of
     the stage's parity;
  2. every dependency the kernel waits on (fused_dep, enumerated exactly as the kernel does) belongs to a cell all
     of whose tiles were handed to LOWER tickets - so the unfinished block with the lowest ticket never waits on
     an unfinished block, and the launch cannot deadlock whatever order the hardware starts blocks in;
  3. every link-level conflict between two sub-steps of the group - one reads a link the other writes - is covered
     by such a dependency. The conflicts are computed here from the definition of the update's footprint (eq 9,
     PAPER.md:83,189: the 18 staple links plus the link itself), not from the offsets the library uses.

With 1-3 every update of the fused launch reads exactly the link values it reads when the sub-steps run as separate
launches in schedule order, hence the bitwise equality that tests/test_gpu_fused.py then observes on the GPU.
"""
import ctypes as C
import itertools

import numpy as np
import pytest

import paper_1112_4533_b200 as su

NONE = 0xFFFFFFFF


def _schedule(dims, spb, g, sub0, cell_planes=0, chunk_planes=0, margin=1):
    L = su.lib()
    nt, geom = C.c_int(), (C.c_int * 5)()
    args = (*dims, spb, g, sub0, cell_planes, chunk_planes, margin)
    assert L.su_fused_schedule_debug(*args, None, 0, C.byref(nt), geom) == su.SU_OK
    work = np.empty((nt.value, g), dtype=np.uint32)
    assert L.su_fused_schedule_debug(*args, work.ctypes.data, work.size, C.byref(nt), geom) == su.SU_OK
    U, nzu, nT, cell_sites, plane_sites = list(geom)
    return work, dict(U=U, nzu=nzu, nT=nT, cell_sites=cell_sites, plane_sites=plane_sites)


def _shift(x, dims, d, s):
    y = list(x)
    y[d] = (y[d] + s) % dims[d]
    return tuple(y)


def _reads(x, mu, dims):
    """links (site, direction) the update of U_mu(x) reads: eq 9's two staple terms per nu != mu, and the link itself"""
    out = [(x, mu)]
    for nu in range(4):
        if nu == mu:
            continue
        xm = _shift(x, dims, nu, -1)
        out += [(x, nu), (_shift(x, dims, nu, 1), mu), (_shift(x, dims, mu, 1), nu),
                (xm, nu), (xm, mu), (_shift(xm, dims, mu, 1), nu)]
    return out


def _check(dims, spb, g, sub0, **kw):
    Lx, Ly, Lz, Lt = dims
    work, G = _schedule(dims, spb, g, sub0, **kw)
    U, nzu, nT, cell_sites, plane = G["U"], G["nzu"], G["nT"], G["cell_sites"], G["plane_sites"]
    assert Lz % U == 0 and nzu == Lz // U and plane == (Lx // 2) * Ly and cell_sites == plane * U
    ncells = Lt * nzu
    L = su.lib()
    stage_pm = [(((sub0 + s) >> 2) & 1, (sub0 + s) & 3) for s in range(g)]

    def sites_of(s, tile_id):
        cell, tile = divmod(int(tile_id), nT)
        t, zu = divmod(cell, nzu)
        par = stage_pm[s][0]
        out = []
        for r in range(tile * spb, min((tile + 1) * spb, cell_sites)):
            zi, rem = divmod(r, plane)
            y, xh = divmod(rem, Lx // 2)
            z = zu * U + zi
            out.append((2 * xh + ((y + z + t + par) & 1), y, z, t))
        return cell, tile, out

    # 1. coverage
    ticket_of_tile = np.full((g, ncells * nT), -1, dtype=np.int64)
    owner = [dict() for _ in range(g)]                  # site -> (ticket, cell)
    for k in range(work.shape[0]):
        for s in range(g):
            if work[k, s] == NONE:
                continue
            assert ticket_of_tile[s, work[k, s]] == -1
            ticket_of_tile[s, work[k, s]] = k
            cell, _, sites = sites_of(s, work[k, s])
            for x in sites:
                assert x not in owner[s] and sum(x) % 2 == stage_pm[s][0]
                owner[s][x] = (k, cell)
    assert (ticket_of_tile >= 0).all()
    for s in range(g):
        assert len(owner[s]) == Lx * Ly * Lz * Lt // 2
    last_ticket_of_cell = ticket_of_tile.reshape(g, ncells, nT).max(axis=2)

    # writer of every link, readers of every link, per stage (from the footprint definition)
    readers = [dict() for _ in range(g)]
    for s in range(g):
        for x in owner[s]:
            for link in _reads(x, stage_pm[s][1], dims):
                readers[s].setdefault(link, []).append(x)

    n_conf = 0
    for k in range(work.shape[0]):
        for s in range(g):
            if work[k, s] == NONE:
                continue
            cell, tile, sites = sites_of(s, work[k, s])
            deps = {L.su_fused_dep_debug(*dims, spb, g, sub0, kw.get("cell_planes", 0), s, cell, tile, kk) for kk in range(s * 10)}
            deps.discard(-1)
            # 2. dependencies were all handed to lower tickets
            for idx in deps:
                a, c = divmod(idx, ncells)
                assert a < s and last_ticket_of_cell[a, c] < k, (k, s, cell, tile, a, c)
            # 3. conflicts are covered
            for x in sites:
                mu_b = stage_pm[s][1]
                rd = _reads(x, mu_b, dims)
                for a in range(s):
                    pa, mu_a = stage_pm[a]
                    conf = {y for (y, d) in rd if d == mu_a and sum(y) % 2 == pa}           # a writes what b reads
                    conf |= set(readers[a].get((x, mu_b), []))                               # b writes what a reads
                    for y in conf:
                        n_conf += 1
                        assert a * ncells + owner[a][y][1] in deps, (k, s, x, a, y)
    return work.shape[0], n_conf, G


@pytest.mark.parametrize("dims,spb", [((4, 4, 4, 6), 4), ((4, 4, 4, 6), 8), ((4, 6, 8, 4), 16), ((2, 2, 2, 2), 2),
                                      ((2, 2, 2, 2), 128), ((6, 2, 4, 8), 5)])
@pytest.mark.parametrize("g,sub0", [(2, 0), (2, 2), (2, 4), (2, 6), (4, 0), (4, 4), (8, 0)])
def test_schedule_is_complete_deadlock_free_and_covers_every_conflict(dims, spb, g, sub0):
    nt, n_conf, G = _check(dims, spb, g, sub0)
    assert n_conf > 0
    V2 = int(np.prod(dims)) // 2
    assert nt >= -(-V2 // spb)


@pytest.mark.parametrize("kw", [dict(cell_planes=2), dict(cell_planes=4, chunk_planes=4), dict(chunk_planes=2, margin=5),
                                dict(cell_planes=1, chunk_planes=1, margin=3)])
def test_schedule_shape_knobs(kw):
    for g, sub0 in [(2, 2), (4, 4), (8, 0)]:
        _check((4, 4, 8, 6), 8, g, sub0, **kw)


def test_pipeline_depth_stays_small_at_the_headline_size():
    """48^4, 128 sites per block: the later stages trail stage 0 by about one time slice of a z-chunk per stage that
    needs the slice above (mu = 3, or the other parity), so the launch ends a few hundred tickets after the last
    stage-0 tile - the working set in flight stays a few chunk-slices, far below the 126 MB L2."""
    for g in (2, 4, 8):
        work, G = _schedule((48, 48, 48, 48), 128, g, 0, chunk_planes=12, margin=8)
        n0 = 48 ** 4 // 2 // 128
        assert G["U"] == 1 and G["nT"] == 9
        assert n0 <= work.shape[0] <= n0 + 5000
        first = [int(np.argmax(work[:, s] != NONE)) for s in range(g)]
        assert first[0] == 0 and max(first) < 1500
        # steady state: the tile of stage s handed out at ticket k lies close behind stage 0's (same chunk, <= 3 slices)
        k = n0 // 2 + n0 // 16                          # mid-chunk (the chunks are n0 / 4 tickets long)
        assert (work[k] != NONE).all()
        cells = (work[k] // G["nT"]).astype(np.int64)
        t, zu = cells // G["nzu"], cells % G["nzu"]
        # the chunk's last z-plane waits for the next chunk, so a stage may be busy with the previous chunk's boundary cell
        assert int(t.max() - t.min()) <= 4 and (np.abs(zu // 12 - zu[0] // 12) <= 1).all()


def test_debug_hooks_validate_arguments():
    L = su.lib()
    nt, geom = C.c_int(), (C.c_int * 5)()
    assert L.su_fused_schedule_debug(4, 4, 4, 5, 8, 2, 0, 0, 0, 1, None, 0, C.byref(nt), geom) == su.SU_EINVAL
    assert L.su_fused_schedule_debug(4, 4, 4, 4, 8, 3, 6, 0, 0, 1, None, 0, C.byref(nt), geom) == su.SU_EINVAL
    w = np.empty(4, dtype=np.uint32)
    assert L.su_fused_schedule_debug(4, 4, 4, 4, 8, 2, 0, 0, 0, 1, w.ctypes.data, 4, C.byref(nt), geom) == su.SU_ENOMEM
