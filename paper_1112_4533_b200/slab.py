"""Drivers of the t-slab decomposition (include/su_gauge.h "t-slab decomposition"; Fig. 2).

Argument marshalling and ordering only: the arithmetic, including the halo push, runs in the CUDA kernels
(the update kernel stores the links of a slab's first / last owned time slice straight into the neighbour
slab's halo - peer memory over NVLink when the slabs sit on different GPUs).

  SlabGroup           n slabs driven by ONE process (one device, or several with peer access): used by the
                      tests to prove that n slabs reproduce the single-lattice chain exactly.
  DistributedLattice  one slab per torch.distributed rank (one process per GPU): peers through CUDA IPC, the
                      ordering between sub-steps through a stream-ordered NCCL all-reduce of one element.

The sweep schedule is the single-lattice one (R6): every sub-step (pass, parity, mu) on all slabs,
then the next; the handles' sweep counters advance together.
"""
import numpy as np

from . import Lattice


def slab_starts(Lt_global, n_slabs):
    """t0 of every slab; Lt_global must split into n equal even pieces."""
    if n_slabs < 1 or Lt_global % n_slabs or (Lt_global // n_slabs) % 2:
        raise ValueError(f"Lt = {Lt_global} does not split into {n_slabs} slabs of equal even length")
    lt = Lt_global // n_slabs
    return [r * lt for r in range(n_slabs)], lt


def ring_neighbours(rank, world):
    """(rank of the slab below in t, rank of the slab above), periodic"""
    return (rank - 1) % world, (rank + 1) % world


def schedule(n_hb, n_or):
    """(kind, heatbath pass number, parity, mu) of the 8 (n_hb + n_or) sub-steps of a sweep, in order."""
    for p in range(n_hb + n_or):
        kind = 0 if p < n_hb else 1
        for parity in range(2):
            for mu in range(4):
                yield kind, (p if kind == 0 else 0), parity, mu


class SlabGroup:
    """A lattice cut into n_slabs t-slabs, all driven from this process on one stream (same-stream order is
    the ordering the ABI asks for). devices: one CUDA ordinal per slab (default: all on `device`)."""

    def __init__(self, Nc, dims, n_slabs, precision="fp64", recon12=False, kernel="auto", device=0, devices=None):
        starts, lt = slab_starts(dims[3], n_slabs)
        devices = devices or [device] * n_slabs
        self.Nc, self.dims, self.n = Nc, tuple(dims), n_slabs
        self.slabs = [Lattice(Nc, dims, precision, recon12, kernel, device=devices[r], slab=(starts[r], lt))
                      for r in range(n_slabs)]
        ptrs = [s.links_ptr()[0] for s in self.slabs]
        for r, s in enumerate(self.slabs):
            below, above = ring_neighbours(r, n_slabs)
            s.set_peers(ptrs[below], ptrs[above])
        self.sweep_counter = 0
        self.seed = 0

    def close(self):
        for s in self.slabs:
            s.close()

    def init_cold(self, seed):
        for s in self.slabs:
            s.init_cold(seed)
        self.seed, self.sweep_counter = seed, 0

    def init_hot(self, seed):
        for s in self.slabs:
            s.init_hot(seed)
        self.seed, self.sweep_counter = seed, 0

    def set_rng(self, seed, sweep_counter):
        for s in self.slabs:
            s.set_rng(seed, sweep_counter)
        self.seed, self.sweep_counter = seed, sweep_counter

    def sweep(self, beta, n_hb=1, n_or=4):
        for kind, pass_, parity, mu in schedule(n_hb, n_or):
            for s in self.slabs:
                s.substep(beta, kind, pass_, parity, mu)
        self.set_rng(self.seed, self.sweep_counter + 1)

    def reunitarize(self):
        for s in self.slabs:
            s.reunitarize()

    def plaquette(self):
        return sum(s.plaquette() for s in self.slabs)

    def export_links(self):
        return np.concatenate([s.export_links() for s in self.slabs], axis=0)

    def import_links(self, links):
        lt = self.dims[3] // self.n
        for r, s in enumerate(self.slabs):
            s.import_links(links[r * lt:(r + 1) * lt])
        for s in self.slabs:
            s.halo_push()

    def counters(self):
        c = [s.counters() for s in self.slabs]
        return sum(x[0] for x in c), sum(x[1] for x in c)


class DistributedLattice:
    """One t-slab per rank of an initialised torch.distributed process group (backend nccl, one process per
    GPU of one node). Neighbours' link buffers are mapped with CUDA IPC; between two sub-steps a one-element
    all-reduce, enqueued on the lattice's stream, orders the ranks without blocking the host."""

    def __init__(self, Nc, dims, precision="fp64", recon12=False, kernel="auto", device=None):
        import torch
        import torch.distributed as dist
        self.dist, self.torch = dist, torch
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        starts, lt = slab_starts(dims[3], self.world)
        device = torch.cuda.current_device() if device is None else device
        self.lat = Lattice(Nc, dims, precision, recon12, kernel, device=device, slab=(starts[self.rank], lt),
                           library_buffer=True)
        handles = [None] * self.world
        dist.all_gather_object(handles, self.lat.ipc_export())
        self._opened = []
        ptr = {self.rank: self.lat.links_ptr()[0]}
        below, above = ring_neighbours(self.rank, self.world)
        for r in {below, above}:
            if r not in ptr:
                ptr[r] = self.lat.ipc_open(handles[r])
                self._opened.append(ptr[r])
        self.lat.set_peers(ptr[below], ptr[above])
        self._token = torch.zeros(1, device=self.lat.device)
        self.seed, self.sweep_counter = 0, 0

    def _order(self):
        # stream-ordered: the collective waits for the kernels already enqueued on the current stream
        # (the lattice's stream) and later kernels on that stream wait for it
        self.dist.all_reduce(self._token)

    def close(self):
        self._order()
        self.torch.cuda.synchronize()
        for p in self._opened:
            self.lat.ipc_close(p)
        self._opened = []
        self.lat.close()

    def init_cold(self, seed):
        self.lat.init_cold(seed)
        self.seed, self.sweep_counter = seed, 0
        self._order()

    def init_hot(self, seed):
        self.lat.init_hot(seed)
        self.seed, self.sweep_counter = seed, 0
        self._order()

    def sweep(self, beta, n_hb=1, n_or=4):
        for kind, pass_, parity, mu in schedule(n_hb, n_or):
            self.lat.substep(beta, kind, pass_, parity, mu)
            self._order()
        self.sweep_counter += 1
        self.lat.set_rng(self.seed, self.sweep_counter)

    def reunitarize(self):
        self.lat.reunitarize()

    def plaquette(self):
        t = self.torch.tensor([self.lat.plaquette()], dtype=self.torch.float64, device=self.lat.device)
        self.dist.all_reduce(t)
        return float(t.item())

    def import_links(self, local_links):
        self.lat.import_links(local_links)
        self._order()
        self.lat.halo_push()
        self._order()

    def export_links(self):
        return self.lat.export_links()
