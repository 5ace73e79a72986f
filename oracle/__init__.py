"""ctypes wrapper of the CPU oracle (oracle/su_oracle.cpp).

TEST INFRASTRUCTURE ONLY: import from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs. The product package never imports this module.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        P = C.c_void_p
        L.so_create.argtypes = [C.c_int] * 7 + [C.POINTER(P)]
        L.so_destroy.argtypes = [P]
        L.so_destroy.restype = None
        L.so_init_cold.argtypes = [P, C.c_uint64]
        L.so_init_hot.argtypes = [P, C.c_uint64]
        L.so_set_rng.argtypes = [P, C.c_uint64, C.c_uint32]
        L.so_sweep.argtypes = [P, C.c_double, C.c_int, C.c_int]
        L.so_substep.argtypes = [P, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.so_plaquette.argtypes = [P, C.POINTER(C.c_double)]
        L.so_polyakov.argtypes = [P, C.POINTER(C.c_double)]
        L.so_reunitarize.argtypes = [P]
        L.so_export_links.argtypes = [P, C.c_void_p, C.c_size_t]
        L.so_import_links.argtypes = [P, C.c_void_p, C.c_size_t]
        L.so_get_counters.argtypes = [P, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.so_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.so_philox4x32_10.restype = None
        L.so_uniform.argtypes = [C.c_uint32, C.c_int]
        L.so_uniform.restype = C.c_double
        L.so_staple.argtypes = [P, C.c_size_t, C.c_int, C.c_void_p]
        L.so_kp_sample.argtypes = [C.c_int, C.c_double, C.c_uint64, C.c_size_t, C.c_void_p, C.c_void_p]
        L.so_update_matrix.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int, C.c_uint64, C.c_uint32,
                                       C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.so_num_threads.restype = C.c_int
        _lib = L
    return _lib


class OracleError(RuntimeError):
    pass


def _ck(rc, what):
    if rc != 0:
        raise OracleError(f"{what} failed with status {rc}")


class OracleLattice:
    """Same surface as paper_1112_4533_b200.Lattice so one harness drives both."""

    def __init__(self, Nc, dims, precision="fp64", recon12=False):
        self.Nc, self.dims = int(Nc), tuple(int(d) for d in dims)
        self.precision = precision
        self.recon12 = bool(recon12)
        self.V = int(np.prod(self.dims))
        self.n_sub = self.Nc * (self.Nc - 1) // 2
        self._h = C.c_void_p()
        _ck(lib().so_create(self.Nc, *self.dims, 1 if precision == "fp64" else 0, int(self.recon12),
                            C.byref(self._h)), "so_create")

    def close(self):
        if self._h:
            lib().so_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init_cold(self, seed):
        _ck(lib().so_init_cold(self._h, seed), "so_init_cold")

    def init_hot(self, seed):
        _ck(lib().so_init_hot(self._h, seed), "so_init_hot")

    def set_rng(self, seed, sweep_counter):
        _ck(lib().so_set_rng(self._h, seed, sweep_counter), "so_set_rng")

    def sweep(self, beta, n_hb, n_or):
        _ck(lib().so_sweep(self._h, beta, n_hb, n_or), "so_sweep")

    def substep(self, beta, kind, pass_, parity, mu, want_attempts=False):
        att = None
        ptr = None
        if want_attempts:
            att = np.zeros((self.n_sub, self.V // 2), dtype=np.uint8)
            ptr = att.ctypes.data
        _ck(lib().so_substep(self._h, beta, kind, pass_, parity, mu, ptr), "so_substep")
        return att

    def plaquette(self):
        out = C.c_double()
        _ck(lib().so_plaquette(self._h, C.byref(out)), "so_plaquette")
        return out.value

    def polyakov(self):
        out = (C.c_double * 2)()
        _ck(lib().so_polyakov(self._h, out), "so_polyakov")
        return complex(out[0], out[1])

    def reunitarize(self):
        _ck(lib().so_reunitarize(self._h), "so_reunitarize")

    def export_links(self):
        """-> complex128 array [t][z][y][x][mu][row][col]"""
        Lx, Ly, Lz, Lt = self.dims
        out = np.empty((Lt, Lz, Ly, Lx, 4, self.Nc, self.Nc), dtype=np.complex128)
        _ck(lib().so_export_links(self._h, out.ctypes.data, out.size * 2), "so_export_links")
        return out

    def import_links(self, links):
        a = np.ascontiguousarray(links, dtype=np.complex128)
        _ck(lib().so_import_links(self._h, a.ctypes.data, a.size * 2), "so_import_links")

    def counters(self):
        a, e = C.c_uint64(), C.c_uint64()
        _ck(lib().so_get_counters(self._h, C.byref(a), C.byref(e)), "so_get_counters")
        return a.value, e.value

    def staple(self, site, mu):
        out = np.empty((self.Nc, self.Nc), dtype=np.complex128)
        _ck(lib().so_staple(self._h, site, mu, out.ctypes.data), "so_staple")
        return out


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().so_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def uniform(w, precision="fp64"):
    return lib().so_uniform(w, 1 if precision == "fp64" else 0)


def kp_sample(alpha, seed, n, precision="fp64"):
    v = np.empty((n, 4), dtype=np.float64)
    att = np.empty(n, dtype=np.uint8)
    _ck(lib().so_kp_sample(1 if precision == "fp64" else 0, alpha, seed, n, v.ctypes.data, att.ctypes.data),
        "so_kp_sample")
    return v, att


def update_matrix(U, W, beta, kind, seed=0, c0=0, c1=0, c2_base=0, precision="fp64"):
    """Subgroup loop on one (U, W) pair; returns (U', W', attempts)."""
    N = U.shape[0]
    u = np.ascontiguousarray(U, dtype=np.complex128).copy()
    w = np.ascontiguousarray(W, dtype=np.complex128).copy()
    att = np.zeros(N * (N - 1) // 2, dtype=np.uint8)
    _ck(lib().so_update_matrix(N, 1 if precision == "fp64" else 0, beta, kind, seed, c0, c1, c2_base,
                               u.ctypes.data, w.ctypes.data, att.ctypes.data), "so_update_matrix")
    return u, w, att


def num_threads():
    return lib().so_num_threads()
