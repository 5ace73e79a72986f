"""Drivers of the t-slab decomposition (include/su_gauge.h "t-slab decomposition"; Fig. 2).

Argument marshalling and ordering only: the arithmetic, including the halo push, runs in the CUDA kernels
(the update kernel stores the links of a slab's first / last owned time slice straight into the neighbour
slab's halo - peer memory over NVLink when the slabs sit on different GPUs).

  SlabGroup           n slabs driven by ONE process on ONE device and one stream: used by the tests to prove
                      that n slabs reproduce the single-lattice chain exactly.
  DistributedLattice  one slab per torch.distributed rank (one process per GPU): peers through CUDA IPC, the
                      ordering between sub-steps through a stream-ordered NCCL all-reduce of one element
                      (order="nccl"), or through su_synchronize + a host barrier (order="host": any backend,
                      e.g. gloo when two test ranks share one GPU).

The sweep schedule is the single-lattice one (R6): every sub-step (pass, parity, mu) on all slabs,
then the next; the handles' sweep counters advance together.
"""
import ctypes as C

import numpy as np

from . import Lattice, SuError, SU_OK, lib


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
    """A lattice cut into n_slabs t-slabs, all on ONE device and driven from this process on one stream
    (same-stream order is the ordering the ABI asks for). Slabs on several devices need one process per device:
    DistributedLattice."""

    def __init__(self, Nc, dims, n_slabs, precision="fp64", recon12=False, kernel="auto", device=0):
        starts, lt = slab_starts(dims[3], n_slabs)
        self.Nc, self.dims, self.n = Nc, tuple(dims), n_slabs
        self.slabs = [Lattice(Nc, dims, precision, recon12, kernel, device=device, slab=(starts[r], lt))
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
        handles = (C.c_void_p * self.n)(*[s._h for s in self.slabs])
        out = C.c_double()
        st = lib().su_slab_plaquette_sum(handles, self.n, C.byref(out))
        if st != SU_OK:
            raise SuError(st, "su_slab_plaquette_sum")
        return out.value

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
    """One t-slab per rank of an initialised torch.distributed process group (one process per GPU of one
    node). Neighbours' link buffers are mapped with CUDA IPC. Ordering between sub-steps (and after every call
    that rewrites halo slices: init, reunitarise, halo push):
      order="nccl"  a one-element all-reduce enqueued on the lattice's stream: stream-ordered, the host never blocks;
      order="host"  su_synchronize + dist.barrier(): works with any backend (gloo), used when NCCL cannot run,
                    e.g. two test ranks sharing one GPU."""

    def __init__(self, Nc, dims, precision="fp64", recon12=False, kernel="auto", device=None, order="nccl"):
        import torch
        import torch.distributed as dist
        if order not in ("nccl", "host"):
            raise ValueError("order must be 'nccl' or 'host'")
        self.dist, self.torch, self.order = dist, torch, order
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
        self._token = torch.zeros(1, device=self.lat.device) if order == "nccl" else None
        self.seed, self.sweep_counter = 0, 0

    def _order(self):
        if self.order == "nccl":
            # stream-ordered: the collective waits for the kernels already enqueued on the lattice's stream and later
            # kernels on that stream wait for it. NCCL enqueues on torch's CURRENT stream, which need not be the one
            # the Lattice captured at construction (a caller inside `with torch.cuda.stream(...)`): select it here,
            # or the all-reduce would order nothing and the peer halo stores would race
            with self.torch.cuda.stream(self.lat.stream):
                self.dist.all_reduce(self._token)
        else:
            self.lat.synchronize()
            self.dist.barrier()

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
        # su_reunitarize rewrites the halo slices too (consistently: the same links, the same arithmetic); a
        # neighbour must not start pushing the next sub-step's links into them before that is finished
        self.lat.reunitarize()
        self._order()

    def plaquette(self):
        dev = self.lat.device if self.order == "nccl" else "cpu"
        t = self.torch.tensor([self.lat.plaquette()], dtype=self.torch.float64, device=dev)
        self.dist.all_reduce(t)
        return float(t.item())

    def import_links(self, local_links):
        self.lat.import_links(local_links)
        self._order()
        self.lat.halo_push()
        self._order()

    def export_links(self):
        return self.lat.export_links()
