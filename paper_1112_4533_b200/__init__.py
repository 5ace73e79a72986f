"""paper_1112_4533_b200 — thin Python binding of libsugauge (include/su_gauge.h).

Argument marshalling only: every step of the path (staple, Cabibbo-Marinari heatbath with
Kennedy-Pendleton draws, overrelaxation, plaquette / Polyakov reductions, reunitarisation, init,
import / export layout conversion) runs in the CUDA kernels under csrc/. PyTorch supplies device
memory (a uint8 tensor that backs the links) and the stream; nothing here computes, and there is
no CPU fallback: a missing library or a missing GPU raises.

Method: Cardoso & Bicudo, arXiv:1112.4533.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# SU_GAUGE_LIB selects an ablation build (python -m paper_1112_4533_b200.build with SUG_BUILD_VARIANT); default: the product library
LIB_PATH = os.environ.get("SU_GAUGE_LIB") or os.path.join(_HERE, "libsugauge.so")

SU_OK, SU_EINVAL, SU_EUNSUPPORTED, SU_ENOMEM, SU_ECUDA, SU_ESTATE = range(6)
_STATUS = {0: "SU_OK", 1: "SU_EINVAL", 2: "SU_EUNSUPPORTED", 3: "SU_ENOMEM", 4: "SU_ECUDA", 5: "SU_ESTATE"}
SU_FP32, SU_FP64 = 0, 1
SU_STORE_FULL, SU_STORE_RECON12 = 0, 1
SU_KERNEL_AUTO, SU_KERNEL_SPECIALISED, SU_KERNEL_GENERIC = 0, 1, 2
SU_MAX_NC = 32

# every entry point include/su_gauge.h and include/su_gauge_test.h declare (tests check the library exports exactly these)
ABI_SYMBOLS = (
    "su_lattice_bytes", "su_lattice_create", "su_lattice_create_ex", "su_lattice_destroy",
    "su_init_cold", "su_init_hot", "su_sweep", "su_plaquette", "su_polyakov", "su_reunitarize",
    "su_export_links", "su_import_links", "su_set_rng", "su_substep", "su_get_counters",
    "su_synchronize", "su_set_graph_mode", "su_set_timing", "su_get_timing", "su_get_launch_count", "su_last_error",
    "su_lattice_create_slab", "su_slab_bytes", "su_slab_links", "su_slab_set_peers", "su_slab_halo_push",
    "su_ipc_export", "su_ipc_open", "su_ipc_close", "su_slab_plaquette_sum", "su_set_option", "su_get_option",
    "su_measure_fma_peak", "su_measure_l2_peak", "su_debug_kp_math", "su_save_config", "su_load_config", "su_fused_schedule_debug", "su_fused_dep_debug",
    "su_plaquette_static", "su_static_last_error",
)


class su_options(C.Structure):
    _fields_ = [("storage", C.c_int), ("kernel", C.c_int), ("device", C.c_int), ("stream", C.c_void_p),
                ("buffer", C.c_void_p), ("buffer_bytes", C.c_size_t)]


class SuError(RuntimeError):
    def __init__(self, status, what, detail=""):
        self.status = status
        super().__init__(f"{what}: {_STATUS.get(status, status)}" + (f" ({detail})" if detail else ""))


_lib = None


def lib():
    """Load libsugauge.so (built in-tree by `python -m paper_1112_4533_b200.build`). Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1112_4533_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    P, I, D = C.c_void_p, C.c_int, C.c_double
    L.su_lattice_bytes.argtypes = [I] * 7
    L.su_lattice_bytes.restype = C.c_size_t
    L.su_lattice_create.argtypes = [I] * 6 + [C.POINTER(P)]
    L.su_lattice_create_ex.argtypes = [I] * 6 + [C.POINTER(su_options), C.POINTER(P)]
    L.su_lattice_destroy.argtypes = [P]
    L.su_init_cold.argtypes = [P, C.c_uint64]
    L.su_init_hot.argtypes = [P, C.c_uint64]
    L.su_sweep.argtypes = [P, D, I, I]
    L.su_plaquette.argtypes = [P, C.POINTER(D)]
    L.su_polyakov.argtypes = [P, C.POINTER(D)]
    L.su_reunitarize.argtypes = [P]
    L.su_export_links.argtypes = [P, C.c_void_p, C.c_size_t]
    L.su_import_links.argtypes = [P, C.c_void_p, C.c_size_t]
    L.su_set_rng.argtypes = [P, C.c_uint64, C.c_uint32]
    L.su_substep.argtypes = [P, D, I, I, I, I, C.c_void_p]
    L.su_get_counters.argtypes = [P, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.su_synchronize.argtypes = [P]
    L.su_set_graph_mode.argtypes = [P, I]
    L.su_set_timing.argtypes = [P, I]
    L.su_get_timing.argtypes = [P, C.POINTER(D), C.POINTER(C.c_uint64), C.POINTER(D), C.POINTER(C.c_uint64)]
    L.su_get_launch_count.argtypes = [P, C.POINTER(C.c_uint64)]
    L.su_last_error.argtypes = [P]
    L.su_last_error.restype = C.c_char_p
    L.su_lattice_create_slab.argtypes = [I] * 8 + [C.POINTER(su_options), C.POINTER(P)]
    L.su_slab_bytes.argtypes = [I] * 7
    L.su_slab_bytes.restype = C.c_size_t
    L.su_slab_links.argtypes = [P, C.POINTER(P), C.POINTER(C.c_size_t)]
    L.su_slab_set_peers.argtypes = [P, P, P]
    L.su_slab_halo_push.argtypes = [P]
    L.su_ipc_export.argtypes = [P, C.c_char_p]
    L.su_ipc_open.argtypes = [P, C.c_char_p, C.POINTER(P)]
    L.su_ipc_close.argtypes = [P, P]
    L.su_slab_plaquette_sum.argtypes = [C.POINTER(P), I, C.POINTER(D)]
    L.su_fused_schedule_debug.argtypes = [I] * 10 + [C.c_void_p, C.c_size_t, C.POINTER(I), C.POINTER(I)]
    L.su_fused_dep_debug.argtypes = [I] * 12
    L.su_save_config.argtypes = [P, C.c_char_p]
    L.su_load_config.argtypes = [P, C.c_char_p]
    L.su_measure_fma_peak.argtypes = [I, I, C.POINTER(D), C.POINTER(D)]
    L.su_debug_kp_math.argtypes = [I, C.c_void_p, C.c_size_t, C.c_void_p]
    L.su_measure_l2_peak.argtypes = [I, I, C.POINTER(D), C.POINTER(D), C.POINTER(D)]
    L.su_set_option.argtypes = [P, C.c_char_p, C.c_longlong]
    L.su_get_option.argtypes = [P, C.c_char_p, C.POINTER(C.c_longlong)]
    for name in ABI_SYMBOLS:
        if name not in ("su_lattice_bytes", "su_slab_bytes", "su_last_error"):
            getattr(L, name).restype = I
    L.su_plaquette_static.argtypes = [I] * 8 + [P, P, C.c_size_t, P]
    L.su_static_last_error.argtypes = []
    L.su_static_last_error.restype = C.c_char_p
    _lib = L
    return L


def _prec(precision):
    if precision in ("fp64", "f64", "double"):
        return SU_FP64
    if precision in ("fp32", "f32", "float"):
        return SU_FP32
    raise ValueError(f"precision must be 'fp32' or 'fp64', got {precision!r}")


def lattice_bytes(Nc, dims, precision="fp64", recon12=False):
    return lib().su_lattice_bytes(Nc, *dims, _prec(precision), SU_STORE_RECON12 if recon12 else SU_STORE_FULL)


def measure_fma_peak(precision="fp64", device=-1):
    """-> (TFLOP/s, ms of the best launch) of the device's FP32 / FP64 FMA pipe (su_measure_fma_peak)"""
    t, ms = C.c_double(), C.c_double()
    st = lib().su_measure_fma_peak(device, _prec(precision), C.byref(t), C.byref(ms))
    if st != SU_OK:
        raise SuError(st, "su_measure_fma_peak")
    return t.value, ms.value


def debug_kp_math(words, device=-1):
    """-> array [n, 5]: ln u, sin 2 pi u, cos 2 pi u, sqrt u, 1 / sqrt(100 u + 0.001) for u = (w + 1) / 2^32 (su_debug_kp_math)"""
    import numpy as np
    w = np.ascontiguousarray(words, dtype=np.uint32)
    out = np.empty((w.size, 5), dtype=np.float64)
    st = lib().su_debug_kp_math(device, w.ctypes.data, w.size, out.ctypes.data)
    if st != SU_OK:
        raise SuError(st, "su_debug_kp_math")
    return out


def measure_l2_peak(device=-1, through_l1=False):
    """-> (GB/s, ms of the best launch, bytes per SM clock) of the device's L2 -> SM read path (su_measure_l2_peak)"""
    g, ms, bpc = C.c_double(), C.c_double(), C.c_double()
    st = lib().su_measure_l2_peak(device, 1 if through_l1 else 0, C.byref(g), C.byref(ms), C.byref(bpc))
    if st != SU_OK:
        raise SuError(st, "su_measure_l2_peak")
    return g.value, ms.value, bpc.value


SU_STATIC_MAX_SITES = 64 ** 4


def plaquette_static(Nc, dims, precision, recon12, links_ptr, links_bytes, out_ptr, stream_ptr=None, device=-1):
    """su_plaquette_static: enqueue the mean plaquette of the DEVICE link buffer `links_ptr` (library layout, whole
    lattice) into the DEVICE double at `out_ptr`, on the cudaStream_t `stream_ptr`. For callers that must not
    allocate GPU memory (their pool owns it all, or they sit in a running loop where cudaMalloc would stall the
    device): the library allocates nothing here; its partial sums go to a fixed 1 MiB array inside the library, which
    limits the lattice to SU_STATIC_MAX_SITES = 64^4 sites and is shared by every call on the device, so calls that
    could overlap on the GPU must be ordered by the caller. Asynchronous; raises SuError with the library's text."""
    st = lib().su_plaquette_static(int(Nc), *[int(d) for d in dims], _prec(precision),
                                   SU_STORE_RECON12 if recon12 else SU_STORE_FULL, int(device),
                                   C.c_void_p(stream_ptr), C.c_void_p(links_ptr), int(links_bytes), C.c_void_p(out_ptr))
    if st != SU_OK:
        raise SuError(st, "su_plaquette_static", (lib().su_static_last_error() or b"").decode())


class Lattice:
    """One SU(Nc) gauge field on the GPU. Same method names as the C ABI without the su_ prefix.

    dims = (Lx, Ly, Lz, Lt). kernel: 'auto' | 'specialised' | 'generic'. The link storage is a torch
    uint8 tensor on `device`, kernels run on torch's current stream at construction time.
    """

    def __init__(self, Nc, dims, precision="fp64", recon12=False, kernel="auto", device=0, graph=False, slab=None,
                 library_buffer=False):
        """slab = (t0, Lt_local): this handle owns the global time slices [t0, t0 + Lt_local) of the lattice
        `dims` (su_lattice_create_slab); see SlabGroup / DistributedLattice in .slab for the drivers.
        library_buffer: let the library cudaMalloc the links (needed for CUDA IPC) instead of a torch tensor."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1112_4533_b200 needs a CUDA device (there is no CPU fallback)")
        L = lib()
        self.Nc, self.dims = int(Nc), tuple(int(d) for d in dims)
        self.precision = "fp64" if _prec(precision) == SU_FP64 else "fp32"
        self.recon12 = bool(recon12)
        self.slab = None if slab is None else (int(slab[0]), int(slab[1]))
        self.local_dims = self.dims if slab is None else self.dims[:3] + (self.slab[1],)
        self.V = int(np.prod(self.local_dims))              # owned sites
        self.n_sub = self.Nc * (self.Nc - 1) // 2
        self._h = C.c_void_p()
        self._torch = torch
        self.device = torch.device("cuda", device) if isinstance(device, int) else torch.device(device)
        storage = SU_STORE_RECON12 if recon12 else SU_STORE_FULL
        if slab is None:
            nbytes = L.su_lattice_bytes(self.Nc, *self.dims, _prec(precision), storage)
        else:
            nbytes = L.su_slab_bytes(self.Nc, *self.dims[:3], self.slab[1], _prec(precision), storage)
        if nbytes == 0:
            raise SuError(SU_EINVAL, "su_lattice_bytes", "invalid Nc / extents / storage")
        self.links_bytes = int(nbytes)
        with torch.cuda.device(self.device):
            self.buffer = None if library_buffer else torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device)
        opt = su_options(storage, {"auto": 0, "specialised": 1, "generic": 2}[kernel], self.device.index or 0,
                         C.c_void_p(self.stream.cuda_stream),
                         C.c_void_p(self.buffer.data_ptr()) if self.buffer is not None else None,
                         nbytes if self.buffer is not None else 0)
        if slab is None:
            st = L.su_lattice_create_ex(self.Nc, *self.dims, _prec(precision), C.byref(opt), C.byref(self._h))
        else:
            st = L.su_lattice_create_slab(self.Nc, *self.dims, self.slab[0], self.slab[1], _prec(precision),
                                          C.byref(opt), C.byref(self._h))
        if st != SU_OK:
            self._h = C.c_void_p()
            raise SuError(st, "su_lattice_create_slab" if slab else "su_lattice_create_ex")
        if graph:
            self.set_graph_mode(True)

    # ---- plumbing ----
    def _ck(self, st, what):
        if st != SU_OK:
            msg = lib().su_last_error(self._h)
            raise SuError(st, what, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_h", None):
            lib().su_lattice_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- the C ABI, one to one ----
    def init_cold(self, seed):
        self._ck(lib().su_init_cold(self._h, seed), "su_init_cold")

    def init_hot(self, seed):
        self._ck(lib().su_init_hot(self._h, seed), "su_init_hot")

    def set_rng(self, seed, sweep_counter):
        self._ck(lib().su_set_rng(self._h, seed, sweep_counter), "su_set_rng")

    def sweep(self, beta, n_hb=1, n_or=4):
        self._ck(lib().su_sweep(self._h, beta, n_hb, n_or), "su_sweep")

    def substep(self, beta, kind, pass_, parity, mu, want_attempts=False):
        att = np.zeros((self.n_sub, self.V // 2), dtype=np.uint8) if want_attempts else None
        self._ck(lib().su_substep(self._h, beta, kind, pass_, parity, mu, att.ctypes.data if want_attempts else None),
                 "su_substep")
        return att

    def plaquette(self):
        out = C.c_double()
        self._ck(lib().su_plaquette(self._h, C.byref(out)), "su_plaquette")
        return out.value

    def polyakov(self):
        out = (C.c_double * 2)()
        self._ck(lib().su_polyakov(self._h, out), "su_polyakov")
        return complex(out[0], out[1])

    def reunitarize(self):
        self._ck(lib().su_reunitarize(self._h), "su_reunitarize")

    def export_links(self, out=None):
        """-> complex128 array [t][z][y][x][mu][row][col] (host)"""
        Lx, Ly, Lz, Lt = self.local_dims
        if out is None:
            out = np.empty((Lt, Lz, Ly, Lx, 4, self.Nc, self.Nc), dtype=np.complex128)
        self._ck(lib().su_export_links(self._h, out.ctypes.data, out.size * 2), "su_export_links")
        return out

    def import_links(self, links):
        a = np.ascontiguousarray(links, dtype=np.complex128)
        self._ck(lib().su_import_links(self._h, a.ctypes.data, a.size * 2), "su_import_links")

    def save_config(self, path):
        self._ck(lib().su_save_config(self._h, str(path).encode()), "su_save_config")

    def load_config(self, path):
        self._ck(lib().su_load_config(self._h, str(path).encode()), "su_load_config")

    def counters(self):
        a, e = C.c_uint64(), C.c_uint64()
        self._ck(lib().su_get_counters(self._h, C.byref(a), C.byref(e)), "su_get_counters")
        return a.value, e.value

    def synchronize(self):
        self._ck(lib().su_synchronize(self._h), "su_synchronize")

    def set_graph_mode(self, enabled):
        self._ck(lib().su_set_graph_mode(self._h, int(bool(enabled))), "su_set_graph_mode")

    def set_timing(self, enabled):
        self._ck(lib().su_set_timing(self._h, int(bool(enabled))), "su_set_timing")

    def timing(self):
        """-> dict(hb_ms, hb_launches, or_ms, or_launches) accumulated since set_timing(True)"""
        a, b = C.c_double(), C.c_double()
        na, nb = C.c_uint64(), C.c_uint64()
        self._ck(lib().su_get_timing(self._h, C.byref(a), C.byref(na), C.byref(b), C.byref(nb)), "su_get_timing")
        return {"hb_ms": a.value, "hb_launches": na.value, "or_ms": b.value, "or_launches": nb.value}

    # ---- t-slab decomposition (include/su_gauge.h "t-slab decomposition") ----
    def links_ptr(self):
        p, n = C.c_void_p(), C.c_size_t()
        self._ck(lib().su_slab_links(self._h, C.byref(p), C.byref(n)), "su_slab_links")
        return p.value, n.value

    def set_peers(self, below_ptr, above_ptr):
        self._ck(lib().su_slab_set_peers(self._h, C.c_void_p(below_ptr), C.c_void_p(above_ptr)), "su_slab_set_peers")

    def halo_push(self):
        self._ck(lib().su_slab_halo_push(self._h), "su_slab_halo_push")

    def ipc_export(self):
        buf = C.create_string_buffer(64)
        self._ck(lib().su_ipc_export(self._h, buf), "su_ipc_export")
        return buf.raw

    def ipc_open(self, handle):
        p = C.c_void_p()
        self._ck(lib().su_ipc_open(self._h, C.create_string_buffer(handle, 64), C.byref(p)), "su_ipc_open")
        return p.value

    def ipc_close(self, ptr):
        self._ck(lib().su_ipc_close(self._h, C.c_void_p(ptr)), "su_ipc_close")

    def set_option(self, name, value):
        self._ck(lib().su_set_option(self._h, name.encode(), int(value)), "su_set_option")

    def get_option(self, name):
        v = C.c_longlong()
        self._ck(lib().su_get_option(self._h, name.encode(), C.byref(v)), "su_get_option")
        return v.value

    def launch_count(self):
        n = C.c_uint64()
        self._ck(lib().su_get_launch_count(self._h, C.byref(n)), "su_get_launch_count")
        return n.value
