"""Host logic of the t-slab decomposition (no GPU): slab boundaries, the ring of neighbours, and the sub-step
schedule the drivers share - which must be the oracle's own sweep order (R6) - plus a world_size-2
gloo run of the rank -> slab mapping."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _slab():
    from paper_1112_4533_b200 import slab      # pure Python import; libsugauge.so is only loaded on use
    return slab


def test_slab_starts_and_ring():
    slab = _slab()
    assert slab.slab_starts(48, 4) == ([0, 12, 24, 36], 12)
    assert slab.slab_starts(8, 1) == ([0], 8)
    for bad in [(48, 5), (12, 4), (8, 0)]:          # not divisible / odd slab length / no slab
        with pytest.raises(ValueError):
            slab.slab_starts(*bad)
    assert slab.ring_neighbours(0, 4) == (3, 1) and slab.ring_neighbours(3, 4) == (2, 0)
    assert slab.ring_neighbours(0, 1) == (0, 0)


def test_schedule_is_the_oracle_sweep_order():
    """Driving the oracle sub-step by sub-step in the drivers' order reproduces the oracle's own sweep."""
    import oracle
    slab = _slab()
    dims = (4, 4, 4, 4)
    A, B = oracle.OracleLattice(3, dims), oracle.OracleLattice(3, dims)
    A.init_hot(3)
    B.init_hot(3)
    A.sweep(6.0, 2, 3)
    steps = list(slab.schedule(2, 3))
    assert len(steps) == 40 and steps[0] == (0, 0, 0, 0) and steps[8] == (0, 1, 0, 0) and steps[16] == (1, 0, 0, 0)
    for kind, pass_, parity, mu in steps:
        B.substep(6.0, kind, pass_, parity, mu)
    assert np.array_equal(A.export_links(), B.export_links())


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    from paper_1112_4533_b200 import slab
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    starts, lt = slab.slab_starts(16, dist.get_world_size())
    mine = (starts[dist.get_rank()], lt)
    gathered = [None] * world
    dist.all_gather_object(gathered, (mine, slab.ring_neighbours(rank, world)))
    q.put((rank, gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_rank_to_slab_mapping_over_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out[0] == out[1] == [((0, 8), (1, 1)), ((8, 8), (0, 0))]
