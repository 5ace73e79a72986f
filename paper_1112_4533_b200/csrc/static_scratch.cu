// static_scratch.cu — su_plaquette_static: the mean plaquette of a link buffer WITHOUT any allocation.
//
// Why it exists. Every other measurement of this library goes through a su_lattice handle, and creating a handle
// calls cudaMalloc five times (per-block partial sums, result, counters, ...) and cudaMallocHost once. Some users of
// the library cannot afford that, or cannot do it at all:
//   * a generation job that sized its lattices to fill the GPU, or that runs inside a program whose own memory pool
//     (PyTorch's caching allocator, for one) has already taken the free HBM: a cudaMalloc issued by the library then
//     fails, or takes memory behind that pool's back;
//   * monitoring code that wants a plaquette value from inside a running production loop: cudaMalloc / cudaFree may
//     synchronise the whole device, so an allocation there stalls the update sweeps on the other streams;
//   * a process that only holds a mapping of somebody else's link buffer (su_ipc_open, a torch tensor handed over by a
//     host framework) and has no handle of its own to measure with.
// For them the per-block partial sums — the only scratch memory the plaquette reduction needs — live in a file-scope
// __device__ array of fixed size that is part of the loaded library image: 1 MiB on every GPU that loads libsugauge,
// from the moment the module is loaded there until the process exits, whether or not this entry point is ever called.
// That size covers lattices up to SU_STATIC_MAX_SITES = 64^4 sites; larger ones are refused (SU_EUNSUPPORTED).
//
// The kernel is k_plaquette of aux_kernels.cu (eq 4) restated for a partial-sum pointer that is not
// part of AuxArgs; thread -> site mapping, product order, block sum and final pass are the same, so under the default
// traversal rule the value equals su_plaquette's bit for bit (tests/test_zz_no_alloc.py). Nothing else in the
// library calls into this file and this file changes no other path.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <mutex>

#include "su_internal.h"

// One partial sum per block of the plaquette kernel: 2 * ceil(V / 2 / PLAQ_BLOCK) doubles at V = SU_STATIC_MAX_SITES = 131072.
#define SUG_STATIC_MAX_PARTIALS (2u * (unsigned)((SU_STATIC_MAX_SITES / 2 + sug::PLAQ_BLOCK - 1) / sug::PLAQ_BLOCK))

// The scratch itself (1 MiB). In HOST code the name `s_plaq_partials` is only a stand-in for the symbol (taking its
// address there does not give a device address); the device address is looked up once per device by
// cudaGetSymbolAddress in scratch_of() below and handed to the kernels as an ordinary pointer argument.
static __device__ __align__(256) double s_plaq_partials[SUG_STATIC_MAX_PARTIALS];

namespace sug {
namespace {

constexpr unsigned STATIC_MAX_PARTIALS = SUG_STATIC_MAX_PARTIALS;
static_assert(STATIC_MAX_PARTIALS * sizeof(double) == (1u << 20), "the static scratch is documented as 1 MiB");

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_lock;
double* g_scratch_ptr[MAX_DEVICES] = {nullptr};      // device address of s_plaq_partials on device d; nullptr: not looked up yet

thread_local char t_err[256] = "";

su_status sfail(su_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return st;
}

// First call on a device: resolve the array's device address with that device current. cudaGetSymbolAddress loads
// the module on the device if it is not loaded yet, which is why the first call per device belongs outside any
// stream capture and outside latency-critical code; later calls only read the cached pointer.
cudaError_t scratch_of(int device, double** out) {
    std::lock_guard<std::mutex> lk(g_setup_lock);
    if (!g_scratch_ptr[device]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, s_plaq_partials);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[device] = p;
    }
    *out = g_scratch_ptr[device];
    return cudaSuccess;
}

// k_plaquette (aux_kernels.cu) with the partial sums going to `partials` (the static array) instead of AuxArgs::partials.
// One block = both parities of PLAQ_BLOCK / 2 consecutive sites of the z-chunked traversal; block b writes partials[b].
template <int NC, class T, int STORE>
__global__ void __launch_bounds__(PLAQ_BLOCK, (sizeof(T) == 8 ? PLAQ_MINB_F64 : PLAQ_MINB_F32))
k_plaquette_static(const void* __restrict__ links, const Geom g, double* __restrict__ partials) {
    typedef LinkIO<NC, T, STORE, true> IO;
    typedef Mat<NC, T, true> M;
    typedef cx<T> C;
    const int p = (int)(threadIdx.x / (PLAQ_BLOCK / 2));
    const unsigned tix = blockIdx.x * (PLAQ_BLOCK / 2) + (threadIdx.x % (PLAQ_BLOCK / 2));
    double acc = 0.0;
    if (tix < g.Vh_int) {
        SiteNbr s;
        site_of_thread(g, tix, p, s);
        const unsigned cb = s.cb;
        if (NC <= 3) {
            C Uo[4][NC * NC], B[NC * NC], D[NC * NC], P[NC * NC], Q[NC * NC];
#pragma unroll
            for (int d = 0; d < 4; ++d) IO::template load<LD_RO>(IO::plane(links, g, d, p), cb, Uo[d]);
#pragma unroll
            for (int mu = 0; mu < 3; ++mu)
#pragma unroll
                for (int nu = mu + 1; nu < 4; ++nu) {
                    IO::template load<LD_RO>(IO::plane(links, g, nu, 1 - p), cb + (unsigned)s.dp[mu], B);
                    IO::template load<LD_RO>(IO::plane(links, g, mu, 1 - p), cb + (unsigned)s.dp[nu], D);
                    M::mul_nn(Uo[mu], B, P);
                    M::mul_nn(Uo[nu], D, Q);
                    acc += (double)M::retr_nd(P, Q);
                }
        } else {
            C A[NC * NC], B[NC * NC], P[NC * NC], Q[NC * NC];
#pragma unroll 1
            for (int mu = 0; mu < 3; ++mu)
#pragma unroll 1
                for (int nu = mu + 1; nu < 4; ++nu) {
                    const unsigned fmu = cb + (unsigned)sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
                    const unsigned fnu = cb + (unsigned)sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
                    IO::template load<LD_RO>(IO::plane(links, g, mu, p), cb, A);
                    IO::template load<LD_RO>(IO::plane(links, g, nu, 1 - p), fmu, B);
                    M::mul_nn(A, B, P);
                    IO::template load<LD_RO>(IO::plane(links, g, nu, p), cb, A);
                    IO::template load<LD_RO>(IO::plane(links, g, mu, 1 - p), fnu, B);
                    M::mul_nn(A, B, Q);
                    acc += (double)M::retr_nd(P, Q);
                }
        }
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// out[0] = scale * sum_b partials[b], one block, the fixed order of k_reduce_final (aux_kernels.cu)
__global__ void __launch_bounds__(REDUCE_BLOCK) k_reduce_static(const double* __restrict__ partials, unsigned nb, double scale,
                                                                double* __restrict__ out) {
    double s = 0.0;
    for (unsigned i = threadIdx.x; i < nb; i += REDUCE_BLOCK) s += partials[i];
    s = block_sum(s);
    if (threadIdx.x == 0) out[0] = s * scale;
}

// The default traversal rule of su_lattice_create (su_api.cu traversal_z_chunk), restated: the largest divisor of Lz
// whose chunk of one time slice stays under 16 MB (SU_GAUGE_ZCHUNK_MB overrides, as there).
int default_z_chunk(int Lx, int Ly, int Lz, size_t link_bytes) {
    const size_t plane = (size_t)Lx * Ly * 4 * link_bytes;
    size_t limit = (size_t)16 << 20;
    if (const char* e = getenv("SU_GAUGE_ZCHUNK_MB")) {
        const long v = atol(e);
        if (v > 0) limit = (size_t)v << 20;
    }
    int zc = 1;
    for (int d = 1; d <= Lz; ++d)
        if (Lz % d == 0 && plane * (size_t)d <= limit) zc = d;
    return zc;
}

struct DeviceScope {       // make `dev` current for the duration of the call, then restore
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceScope(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) { err = cudaSetDevice(dev); switched = (err == cudaSuccess); }
    }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};

}  // namespace
}  // namespace sug

using namespace sug;

extern "C" {

su_status su_plaquette_static(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_storage s, int device,
                              void* stream, const void* device_links, size_t links_bytes, double* device_out) {
    t_err[0] = 0;
    if (!device_links || !device_out) return sfail(SU_EINVAL, "su_plaquette_static: null link or output pointer");
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2 || (L[d] & 1)) return sfail(SU_EINVAL, "su_plaquette_static: every extent must be even and >= 2 (got %d in direction %d)", L[d], d);
    if (p != SU_FP32 && p != SU_FP64) return sfail(SU_EINVAL, "su_plaquette_static: precision must be SU_FP32 or SU_FP64");
    if (s != SU_STORE_FULL && s != SU_STORE_RECON12) return sfail(SU_EINVAL, "su_plaquette_static: unknown storage mode");
    if (Nc < 2 || (s == SU_STORE_RECON12 && Nc != 3)) return sfail(SU_EINVAL, "su_plaquette_static: Nc must be >= 2, two-row storage is SU(3) only");
    if (Nc > 4)
        return sfail(SU_EUNSUPPORTED, "su_plaquette_static: only the register layouts of Nc = 2, 3, 4 have a no-allocation form (Nc = %d)", Nc);
    const double sites = (double)Lx * Ly * Lz * Lt;
    if (sites > (double)SU_STATIC_MAX_SITES)
        return sfail(SU_EUNSUPPORTED,
                     "su_plaquette_static: %.0f sites exceed the static scratch limit of %lld sites (64^4); use su_plaquette on a handle",
                     sites, (long long)SU_STATIC_MAX_SITES);
    const size_t need = su_lattice_bytes(Nc, Lx, Ly, Lz, Lt, p, s);
    if (need == 0) return sfail(SU_EINVAL, "su_plaquette_static: invalid lattice");
    if (links_bytes < need) return sfail(SU_EINVAL, "su_plaquette_static: link buffer of %zu bytes, su_lattice_bytes says %zu", links_bytes, need);
    if (((uintptr_t)device_links & 15u) || ((uintptr_t)device_out & 7u))
        return sfail(SU_EINVAL, "su_plaquette_static: links must be 16-byte and the output 8-byte aligned");

    int dev = device;
    if (dev < 0) {
        const cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return sfail(SU_ECUDA, "su_plaquette_static: cudaGetDevice: %s", cudaGetErrorString(e));
    }
    if (dev >= MAX_DEVICES) return sfail(SU_EUNSUPPORTED, "su_plaquette_static: device ordinal %d above %d", dev, MAX_DEVICES - 1);
    DeviceScope scope(dev);
    if (scope.err != cudaSuccess) return sfail(SU_ECUDA, "su_plaquette_static: selecting device %d: %s", dev, cudaGetErrorString(scope.err));
    double* partials = nullptr;
    if (const cudaError_t e = scratch_of(dev, &partials))
        return sfail(SU_ECUDA, "su_plaquette_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));

    // the geometry of a whole (non-slab) lattice, as su_lattice_create sets it
    Geom g{};
    g.L[0] = Lx; g.L[1] = Ly; g.L[2] = Lz; g.L[3] = Lt;
    g.Lxh = Lx / 2;
    const size_t V = (size_t)Lx * Ly * Lz * Lt;
    g.t_halo = 0; g.Lt_int = Lt; g.Lt_glob = Lt; g.t0g = 0;
    g.Vsh = (unsigned)((size_t)Lx * Ly * Lz / 2);
    g.Vh_int = g.Vsh * (unsigned)Lt;
    g.Vh = (unsigned)(V / 2);
    g.Vhp = (unsigned)((V / 2 + LINK_TILE - 1) / LINK_TILE * LINK_TILE);
    const int elems = Nc == 2 ? 2 : (s == SU_STORE_RECON12 ? 6 : Nc * Nc);
    g.Zc = default_z_chunk(Lx, Ly, Lz, (size_t)elems * 2 * (p == SU_FP64 ? 8 : 4));

    const unsigned nb = plaquette_blocks(g.Vh_int);      // <= STATIC_MAX_PARTIALS by the size check above
    const cudaStream_t st = (cudaStream_t)stream;
    const bool f64 = p == SU_FP64;
#define SUG_STATIC_LAUNCH(NC, STORE)                                                                       \
    do {                                                                                                   \
        if (f64) k_plaquette_static<NC, double, STORE><<<nb, PLAQ_BLOCK, 0, st>>>(device_links, g, partials); \
        else     k_plaquette_static<NC, float,  STORE><<<nb, PLAQ_BLOCK, 0, st>>>(device_links, g, partials); \
    } while (0)
    if (Nc == 2) SUG_STATIC_LAUNCH(2, STORE_QUAT);
    else if (Nc == 3 && s == SU_STORE_RECON12) SUG_STATIC_LAUNCH(3, STORE_RECON12);
    else if (Nc == 3) SUG_STATIC_LAUNCH(3, STORE_FULL);
    else SUG_STATIC_LAUNCH(4, STORE_FULL);
#undef SUG_STATIC_LAUNCH
    const double scale = 1.0 / (6.0 * 2.0 * (double)g.Vsh * (double)Lt * (double)Nc);
    k_reduce_static<<<1, REDUCE_BLOCK, 0, st>>>(partials, nb, scale, device_out);
    if (const cudaError_t e = cudaGetLastError())
        return sfail(SU_ECUDA, "su_plaquette_static: kernel launch: %s", cudaGetErrorString(e));
    return SU_OK;
}

const char* su_static_last_error(void) { return t_err; }

}  // extern "C"
