// su_api.cu — the C ABI of libsugauge (include/su_gauge.h): handle, validation, sweep schedule,
// reductions' host side, import/export staging. All arithmetic of the method runs in the kernels
// of update_kernels.cu / aux_kernels.cu; nothing here falls back to the CPU.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <tuple>
#include <vector>

#include "su_internal.h"

using namespace sug;

struct su_lattice {
    int Nc = 0;
    Geom g{};
    size_t V = 0;
    su_precision prec = SU_FP64;
    Variant var{};
    int device = 0;
    cudaStream_t stream = nullptr;
    void* links = nullptr;
    void* peer_lo = nullptr;       // slab mode: link buffers of the slabs below / above (su_slab_set_peers)
    void* peer_hi = nullptr;
    bool owns_links = false;
    size_t links_bytes = 0;
    size_t link_bytes = 0;         // bytes of one stored link
    double* d_partials = nullptr;
    double* d_result = nullptr;
    double* h_result = nullptr;    // pinned host copy of d_result (2 doubles): the read-back of a reduction is one async copy + sync
    unsigned long long* d_counters = nullptr;
    uint32_t* d_sweep = nullptr;
    uint8_t* d_attempts = nullptr;
    double* d_staging[2] = {nullptr, nullptr};   // import / export staging, double-buffered against the PCIe copies
    size_t staging_bytes = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_filled[2] = {nullptr, nullptr}, ev_drained[2] = {nullptr, nullptr};
    bool halos_valid = true;
    // fused launches of g consecutive sub-steps (fused_schedule.h): tables per (g, stage pattern, tile size)
    struct FusedTable { FusedGeom fg; unsigned n_tickets; uint32_t* d_work; unsigned* d_done; FusedCtrl* d_ctrl; };
    std::map<std::tuple<int, int, int>, FusedTable> fused;
    int fuse_g = 1;                  // sub-steps per launch: 1 (plain), 2, 4 or 8
    int fuse_chunk_planes = 0;       // z-planes per chunk of the fused traversal (0: the plain kernel's Zc)
    int fuse_margin = 8;             // tickets between a cell's last tile and the first tile that depends on it
    int fuse_cell_planes = 0;        // z-planes per cell (0: chosen by fused_make_geom)
    unsigned long long fuse_wait_ns = 10000000000ull;   // fused launches: a dependency wait longer than this aborts the launch (10 s)
    int prefetch_slices = 0;         // update kernels: L2 prefetch distance in time slices (0: off)
    int blocks_per_sm = 0;           // update kernels: cap on the resident blocks per SM (0: whatever fits)
    int tile_z = 1, tile_t = 1;      // register update kernels: z-planes x time slices per block tile (Geom::Bz, Bt)
    bool coop_sweep = false;         // su_sweep: one cooperative launch per kind (all its passes) when the lattice fits the device at once
    long long coop_sites[2] = {-1, -1};   // cached capacity (sites of one parity) of the cooperative kernel per kind; -1: not queried
    bool substep_reunit = false;     // test hook: su_substep runs the reunitarise-before-store kernel instances (the last pass of a reunit_on_store sweep)
    bool reunit_on_store = false;    // su_sweep leaves reunitarised links (in its last pass; see su_set_option)                     // slab mode: false between su_import_links and su_slab_halo_push
    uint64_t seed = 0;
    uint32_t sweep = 0;
    bool ready = false;
    bool graph_mode = false;
    std::map<std::tuple<double, int, int>, cudaGraphExec_t> graphs;
    std::map<std::tuple<double, int, int>, uint64_t> graph_launches;    // kernels per replay of each graph
    uint64_t n_launch = 0;
    // per-kind device timing of su_sweep (su_set_timing): events before / between / after the pass groups
    bool timing = false;
    struct SweepEvents { cudaEvent_t e[3]; int n_hb, n_or; };
    std::vector<SweepEvents> pending;
    std::vector<cudaEvent_t> free_events;
    double hb_ms = 0, or_ms = 0;
    uint64_t hb_launches = 0, or_launches = 0;
    char err[512] = {0};
};

namespace {

#ifndef SUG_ZCHUNK_MB
#define SUG_ZCHUNK_MB 16
#endif

const char* kNullHandle = "null lattice handle";

struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) { cudaSetDevice(dev); switched = true; }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

su_status fail(su_lattice* h, su_status st, const char* fmt, const char* detail = "") {
    if (h) snprintf(h->err, sizeof(h->err), fmt, detail);
    return st;
}
su_status cuda_fail(su_lattice* h, cudaError_t e, const char* where) {
    if (h) snprintf(h->err, sizeof(h->err), "CUDA error in %s: %s", where, cudaGetErrorString(e));
    return SU_ECUDA;
}
#define SU_CUDA(h, call, where)                                   \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, where);  \
    } while (0)

bool dims_ok(int Nc, int Lx, int Ly, int Lz, int Lt) {
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int d = 0; d < 4; ++d) if (L[d] < 2 || (L[d] & 1)) return false;     // reading R7
    if (Nc < 2) return false;
    return (double)Lx * Ly * Lz * Lt <= 4294967295.0;   // the site index is one 32-bit RNG counter word
}
// The kernels index links (8 V/2 of them) and checkerboard offsets in 32 bits: V < 2^30 keeps every such product
// in range (176^4 = 0.96e9 sites; SU(2) fp32 at that size is 61 GB). Larger lattices: SU_EUNSUPPORTED.
bool size_supported(int Lx, int Ly, int Lz, int Lt) { return (double)Lx * Ly * Lz * Lt <= 1073741824.0 - 1024.0; }

int elems_per_link(int Nc, su_storage s) { return Nc == 2 ? 2 : (s == SU_STORE_RECON12 ? 6 : Nc * Nc); }
// sites stored per (mu, parity) plane: V/2 rounded up to whole tiles of LINK_TILE sites
size_t plane_sites(size_t Vh) { return (Vh + LINK_TILE - 1) / LINK_TILE * LINK_TILE; }

// Traversal order of the update kernel: the largest divisor Zc of Lz for
// which one (Zc z-planes) x (one time slice) x (all 8 link planes) chunk stays under 16 MB, so that the
// three chunks in flight (t-1, t, t+1) sit in L2 together. Measured at 48^4: DRAM traffic 1.34x -> 1.08x
// of the algorithmic bytes (profiles/r01a, r01b).
int traversal_z_chunk(const Geom& g, size_t link_bytes) {
    const size_t plane = (size_t)g.L[0] * g.L[1] * 4 * link_bytes;   // one z-plane of one time slice, 4 directions
    size_t limit = (size_t)SUG_ZCHUNK_MB << 20;
    if (const char* e = getenv("SU_GAUGE_ZCHUNK_MB")) {              // tuning knob
        const long v = atol(e);
        if (v > 0) limit = (size_t)v << 20;
    }
    int zc = 1;
    for (int d = 1; d <= g.L[2]; ++d)
        if (g.L[2] % d == 0 && plane * (size_t)d <= limit) zc = d;
    return zc;
}

#define SU_BY_NC(h, FN, ...)                                                   \
    ([&]() -> cudaError_t {                                                    \
        switch ((h)->Nc) {                                                     \
            case 2: return FN##2(__VA_ARGS__);                                 \
            case 3: return FN##3(__VA_ARGS__);                                 \
            case 4: return FN##4(__VA_ARGS__);                                 \
            case 5: return FN##5(__VA_ARGS__);                                 \
            case 6: return FN##6(__VA_ARGS__);                                 \
            case 7: return FN##7(__VA_ARGS__);                                 \
            case 8: return FN##8(__VA_ARGS__);                                 \
            default: return FN##_big(__VA_ARGS__);        /* 9 .. SU_MAX_NC */ \
        }                                                                      \
    })()

AuxArgs aux_args(su_lattice* h) {
    AuxArgs a{};
    a.links = h->links; a.g = h->g; a.partials = h->d_partials; a.result = h->d_result;
    a.staging = h->d_staging[0]; a.site0 = 0; a.nsites = 0;
    a.k0 = (uint32_t)h->seed; a.k1 = (uint32_t)(h->seed >> 32);
    return a;
}

__global__ void k_set_u32(uint32_t* p, uint32_t v) { *p = v; }

// FMA-rate micro-benchmark (su_measure_fma_peak): 16 independent accumulator chains per thread, so the pipe is
// never latency-bound; the operands come from memory so nothing folds at compile time.
template <class T>
__global__ void __launch_bounds__(256) k_fma_peak(T* out, const T* in, int iters) {
    T a[16];
    const T x = in[0], y = in[1];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = in[2] + (T)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 16; ++i) a[i] = a[i] * x + y;
        }
    }
    T s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == (T)123456789) out[blockIdx.x * blockDim.x + threadIdx.x] = s;     // never true: keeps the chains alive
}

// L2 -> SM throughput micro-benchmark (su_measure_l2_peak): every block streams the whole L2-resident buffer with
// 128-bit loads that bypass L1 (ld.global.cg), 8 independent loads per thread in flight; the sum keeps them alive.
template <int MODE>      // 0: ld.global.cg (L2 only), 1: ld.global.nc (through L1, as the update kernels' neighbour loads)
__global__ void __launch_bounds__(256) k_l2_peak(double* out, const double2* __restrict__ buf, size_t n16, int passes) {
    double acc = 0;
    const long long c0 = clock64();
    const size_t stride = (size_t)blockDim.x * 8;
    for (int p = 0; p < passes; ++p) {
        // blocks start at different offsets so that the L2 slices are hit evenly at any instant
        size_t i = ((size_t)blockIdx.x * 40503u * stride + threadIdx.x) % n16;
        for (size_t done = 0; done < n16; done += stride) {
            double2 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) { size_t j = i + (size_t)k * blockDim.x; if (j >= n16) j -= n16; v[k] = MODE == 0 ? __ldcg(buf + j) : __ldg(buf + j); }
#pragma unroll
            for (int k = 0; k < 8; ++k) acc += v[k].x + v[k].y;
            i += stride; if (i >= n16) i -= n16;
        }
    }
    if (acc == 123456789.0) out[blockIdx.x * blockDim.x + threadIdx.x] = acc;       // never true
    if (blockIdx.x == 0 && threadIdx.x == 0) out[0] = (double)(clock64() - c0);     // SM clocks of a block that ran start to end
}

// su_debug_kp_math: the elementary functions of the Kennedy-Pendleton draw as the fp64 kernels evaluate them
__global__ void k_debug_kp_math(const uint32_t* w, size_t n, double* out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double u = ((double)w[i] + 1.0) * (1.0 / 4294967296.0);
    double sn, cs;
    Fn<double>::sincos2pi_w(w[i], &sn, &cs);
    out[5 * i + 0] = Fn<double>::log_w(w[i]);
    out[5 * i + 1] = sn;
    out[5 * i + 2] = cs;
    out[5 * i + 3] = Fn<double>::sqrt01(u);
    out[5 * i + 4] = Fn<double>::rsqrt_pos(100.0 * u + 1e-3);
}

void free_graphs(su_lattice* h);

void free_fused(su_lattice* h) {
    for (auto& kv : h->fused) {
        cudaFree(kv.second.d_work); cudaFree(kv.second.d_done); cudaFree(kv.second.d_ctrl);
    }
    h->fused.clear();
}

int update_spb(su_lattice* h, int kind) {
    switch (h->Nc) {
        case 2: return update_spb_nc2(h->var, kind);
        case 3: return update_spb_nc3(h->var, kind);
        case 4: return update_spb_nc4(h->var, kind);
        case 5: return update_spb_nc5(h->var, kind);
        case 6: return update_spb_nc6(h->var, kind);
        case 7: return update_spb_nc7(h->var, kind);
        case 8: return update_spb_nc8(h->var, kind);
        default: return 0;
    }
}

// "coop_sweep": the whole-pass cooperative kernel can be used when it exists for this variant, the handle is not a slab
// and every block of a sub-step is resident at once
bool coop_fits(su_lattice* h, int kind) {
    if (!h->coop_sweep || h->g.t_halo) return false;
    if (h->coop_sites[kind] < 0) {
        switch (h->Nc) {
            case 2: h->coop_sites[kind] = update_coop_sites_nc2(h->var, kind); break;
            case 3: h->coop_sites[kind] = update_coop_sites_nc3(h->var, kind); break;
            case 4: h->coop_sites[kind] = update_coop_sites_nc4(h->var, kind); break;
            default: h->coop_sites[kind] = 0;
        }
    }
    return (long long)h->g.Vh_int <= h->coop_sites[kind];
}

// fused launches need the whole lattice in one buffer with periodic t (no slab halos) and a kernel that has the fused form
int effective_fuse(su_lattice* h, int kind) {
    if (h->fuse_g <= 1 || h->g.t_halo || update_spb(h, kind) <= 0) return 1;
    return h->fuse_g;
}

// the table of the group of g sub-steps that starts at sub-step sub0 (built and uploaded on first use)
su_status fused_table(su_lattice* h, int kind, int sub0, su_lattice::FusedTable** out) {
    const int g = h->fuse_g, spb = update_spb(h, kind);
    const auto key = std::make_tuple(g, sub0 % 4, spb);
    auto it = h->fused.find(key);
    if (it == h->fused.end()) {
        su_lattice::FusedTable t{};
        t.fg = fused_make_geom(h->g.L[0], h->g.L[1], h->g.L[2], h->g.L[3], spb, g, sub0 % 4, h->fuse_cell_planes);
        const int chunk_planes = h->fuse_chunk_planes > 0 ? h->fuse_chunk_planes : h->g.Zc;
        std::vector<uint32_t> work;
        int nt = 0;
        if (!fused_build_schedule(t.fg, chunk_planes / t.fg.U > 0 ? chunk_planes / t.fg.U : 1, h->fuse_margin, work, nt))
            return fail(h, SU_ESTATE, "fused schedule construction failed");
        t.n_tickets = (unsigned)nt;
        const size_t ncnt = (size_t)g * t.fg.Lt * t.fg.nzu;
        cudaError_t e = cudaMalloc(&t.d_work, work.size() * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMalloc(&t.d_done, ncnt * sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMalloc(&t.d_ctrl, sizeof(FusedCtrl));
        if (e == cudaSuccess) e = cudaMemcpy(t.d_work, work.data(), work.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemset(t.d_done, 0, ncnt * sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMemset(t.d_ctrl, 0, sizeof(FusedCtrl));
        if (e != cudaSuccess) {
            cudaFree(t.d_work); cudaFree(t.d_done); cudaFree(t.d_ctrl); cudaGetLastError();
            return fail(h, SU_ENOMEM, "fused schedule upload failed");
        }
        it = h->fused.emplace(key, t).first;
    }
    *out = &it->second;
    return SU_OK;
}

// A dependency wait that gave up (fused_wait) means a broken schedule or a wedged device: the launch stopped half way,
// so the links are a mixture of old and new and the tables' counters are inconsistent. Report it, and leave the handle
// in a state from which the caller can go on: captured graphs and fused tables are dropped (rebuilt and zeroed on the
// next use) and the lattice counts as uninitialised until su_init_* / su_import_links / su_load_config.
// Called only after the stream has been synchronised.
su_status check_fused_error(su_lattice* h) {
    bool tripped = false;
    for (auto& kv : h->fused) {
        FusedCtrl c{};
        SU_CUDA(h, cudaMemcpy(&c, kv.second.d_ctrl, sizeof(c), cudaMemcpyDeviceToHost), "fused control read-back");
        if (c.error) tripped = true;
    }
    if (!tripped) return SU_OK;
    free_graphs(h);
    free_fused(h);
    h->ready = false;
    return fail(h, SU_ECUDA, "fused launch: a dependency wait timed out; the links are not valid (initialise or import them again)");
}

// the register kernels of Nc <= 4 can reunitarise the link they have just updated before they store it
bool reunit_in_kernel(const su_lattice* h) { return !h->var.generic && h->Nc <= 4; }

// "blocks_per_sm" = n: every update launch asks for so much (unused) dynamic shared memory that only n blocks fit an SM
int occupancy_cap_bytes(const su_lattice* h) {
    if (h->blocks_per_sm <= 0) return 0;
    const int per_sm = 227 * 1024, reserve = 1024 + 8 * 1024;     // 1 KB per block is the system's; headroom for static shared memory
    const int bytes = per_sm / h->blocks_per_sm - reserve;
    return bytes > 0 ? bytes : 0;                                  // more blocks than shared memory could ever limit: no cap
}

// Block tiles (Geom::Bz, Bt, Wb) for the launch of one sub-step, if the register kernel of this variant and kind can
// take them: whole warps per x-y plane, whole tiles per z-chunk and per owned time range, whole blocks per segment row.
void set_block_tile(const su_lattice* h, int kind, Geom& g) {
    g.Bz = g.Bt = 1; g.Wb = 0;
    const int spb = h->Nc <= 4 && !h->var.generic && h->Nc > 2 ? update_spb(const_cast<su_lattice*>(h), kind) : 0;
    const int bz = h->tile_z, bt = h->tile_t, pl = g.Lxh * g.L[1];
    if (bz * bt <= 1 || spb <= 0 || spb % 32 || pl % 32) return;
    const int wb = spb / 32;
    if (wb % (bz * bt) || g.Zc % bz || g.Lt_int % bt || (pl / 32) % (wb / (bz * bt))) return;
    g.Bz = bz; g.Bt = bt; g.Wb = wb;
}

su_status launch_fused_group(su_lattice* h, double beta, int kind, int pass, int sub0, const uint32_t* d_sweep, bool reunit) {
    su_lattice::FusedTable* t = nullptr;
    su_status st = fused_table(h, kind, sub0, &t);
    if (st != SU_OK) return st;
    UpdateArgs a{};
    a.links = h->links; a.g = h->g; a.parity = sub0 >> 2; a.mu = sub0 & 3; a.beta = beta;
    a.k0 = (uint32_t)h->seed; a.k1 = (uint32_t)(h->seed >> 32);
    a.sweep = h->sweep; a.sweep_ptr = d_sweep; a.pass = (uint32_t)pass;
    a.attempts = nullptr; a.counters = h->d_counters; a.reunit = reunit ? 1 : 0;
    a.pf_slices = h->prefetch_slices; a.dyn_smem = occupancy_cap_bytes(h);
    a.fz.work = t->d_work; a.fz.done = t->d_done; a.fz.ctrl = t->d_ctrl; a.fz.fg = t->fg; a.fz.fg.sub0 = sub0;
    a.fz.n_tickets = t->n_tickets;
    a.fz.wait_ns = h->fuse_wait_ns;
    SU_CUDA(h, SU_BY_NC(h, update_nc, h->var, kind, a, h->stream, &h->n_launch), "fused update kernel launch");
    return SU_OK;
}

su_status launch_substep(su_lattice* h, double beta, int kind, int pass, int parity, int mu,
                         uint8_t* d_attempts, const uint32_t* d_sweep, bool reunit = false) {
    UpdateArgs a{};
    a.links = h->links; a.g = h->g; a.parity = parity; a.mu = mu; a.beta = beta;
    a.k0 = (uint32_t)h->seed; a.k1 = (uint32_t)(h->seed >> 32);
    a.sweep = h->sweep; a.sweep_ptr = d_sweep; a.pass = (uint32_t)pass;
    a.attempts = d_attempts; a.counters = h->d_counters; a.reunit = reunit ? 1 : 0;
    a.peer_lo = h->peer_lo; a.peer_hi = h->peer_hi;
    a.pf_slices = h->prefetch_slices; a.dyn_smem = occupancy_cap_bytes(h);
    set_block_tile(h, kind, a.g);
    if (h->g.t_halo && (!h->peer_lo || !h->peer_hi)) return fail(h, SU_ESTATE, "slab lattice: su_slab_set_peers first");
    SU_CUDA(h, SU_BY_NC(h, update_nc, h->var, kind, a, h->stream, &h->n_launch), "update kernel launch");
    return SU_OK;
}

cudaEvent_t take_event(su_lattice* h) {
    cudaEvent_t e = nullptr;
    if (!h->free_events.empty()) { e = h->free_events.back(); h->free_events.pop_back(); }
    else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }
    return e;
}

// Fold finished sweeps' event pairs into the per-kind totals (synchronises on the last event).
void drain_timing(su_lattice* h) {
    for (auto& s : h->pending) {
        float a = 0, b = 0;
        if (cudaEventSynchronize(s.e[2]) == cudaSuccess && cudaEventElapsedTime(&a, s.e[0], s.e[1]) == cudaSuccess &&
            cudaEventElapsedTime(&b, s.e[1], s.e[2]) == cudaSuccess) {
            h->hb_ms += a; h->or_ms += b;
            h->hb_launches += (uint64_t)s.n_hb * 8; h->or_launches += (uint64_t)s.n_or * 8;
        } else {
            cudaGetLastError();
        }
        for (int i = 0; i < 3; ++i) h->free_events.push_back(s.e[i]);
    }
    h->pending.clear();
}

su_status enqueue_sweep(su_lattice* h, double beta, int n_hb, int n_or, const uint32_t* d_sweep, bool timed) {
    // reading R6: all heatbath passes, then all overrelaxation passes; parity outer, mu inner
    su_lattice::SweepEvents ev{};
    if (timed) {
        if (h->pending.size() >= 256) drain_timing(h);
        for (int i = 0; i < 3; ++i) if (!(ev.e[i] = take_event(h))) return fail(h, SU_ECUDA, "cudaEventCreate failed");
        ev.n_hb = n_hb; ev.n_or = n_or;
        SU_CUDA(h, cudaEventRecord(ev.e[0], h->stream), "timing event");
    }
    // "reunit_on_store": every link is updated exactly once in the LAST pass of the sweep; there the Nc <= 4 register
    // kernels project it back to SU(Nc) before they store it (the other kernels get the reunitarisation kernel below)
    const bool reunit_store = h->reunit_on_store && h->Nc > 2 - 1 && reunit_in_kernel(h) && n_hb + n_or > 0;
    for (int pass = 0; pass < n_hb + n_or; ++pass) {
        const int kind = pass < n_hb ? KIND_HB : KIND_OR;
        const bool ru = reunit_store && pass == n_hb + n_or - 1;
        if (timed && pass == n_hb) SU_CUDA(h, cudaEventRecord(ev.e[1], h->stream), "timing event");
        if (coop_fits(h, kind)) {
            // all the passes of this kind in ONE cooperative launch (grid barriers between the sub-steps)
            const int n_kind = kind == KIND_HB ? n_hb : n_or, last = n_hb + n_or - 1;
            UpdateArgs a{};
            a.links = h->links; a.g = h->g; a.parity = 0; a.mu = 0; a.beta = beta;
            a.k0 = (uint32_t)h->seed; a.k1 = (uint32_t)(h->seed >> 32);
            a.sweep = h->sweep; a.sweep_ptr = d_sweep; a.pass = kind == KIND_HB ? (uint32_t)pass : 0u;
            a.attempts = nullptr; a.counters = h->d_counters;
            a.reunit = (reunit_store && pass + n_kind - 1 == last) ? 1 : 0;
            a.coop_passes = n_kind;
            SU_CUDA(h, SU_BY_NC(h, update_nc, h->var, kind, a, h->stream, &h->n_launch), "cooperative update kernel launch");
            pass += n_kind - 1;
            continue;
        }
        const int g = effective_fuse(h, kind);
        if (g > 1) {
            for (int sub0 = 0; sub0 < 8; sub0 += g) {        // sub-step index = 4 parity + mu (reading R6)
                su_status st = launch_fused_group(h, beta, kind, kind == KIND_HB ? pass : 0, sub0, d_sweep, ru);
                if (st != SU_OK) return st;
            }
            continue;
        }
        for (int parity = 0; parity < 2; ++parity)
            for (int mu = 0; mu < 4; ++mu) {
                su_status st = launch_substep(h, beta, kind, kind == KIND_HB ? pass : 0, parity, mu, nullptr, d_sweep, ru);
                if (st != SU_OK) return st;
            }
    }
    if (h->reunit_on_store && !reunit_store && n_hb + n_or > 0) {
        AuxArgs ra = aux_args(h);
        SU_CUDA(h, SU_BY_NC(h, reunit_nc, h->var, ra, h->stream, &h->n_launch), "reunitarise kernel");
    }
    if (timed) {
        if (n_or == 0) SU_CUDA(h, cudaEventRecord(ev.e[1], h->stream), "timing event");
        SU_CUDA(h, cudaEventRecord(ev.e[2], h->stream), "timing event");
        h->pending.push_back(ev);
    }
    return SU_OK;
}

// slab mode: after su_import_links the halo slices are stale until every slab has called su_slab_halo_push
su_status halos_ok(su_lattice* h, const char* who) {
    if (h->g.t_halo && !h->halos_valid) return fail(h, SU_ESTATE, "%s after su_import_links on a slab: su_slab_halo_push first", who);
    return SU_OK;
}

su_status ensure_staging(su_lattice* h, size_t bytes) {
    if (!h->copy_stream) {
        SU_CUDA(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking), "copy stream");
        for (int b = 0; b < 2; ++b) {
            SU_CUDA(h, cudaEventCreateWithFlags(&h->ev_filled[b], cudaEventDisableTiming), "staging event");
            SU_CUDA(h, cudaEventCreateWithFlags(&h->ev_drained[b], cudaEventDisableTiming), "staging event");
        }
    }
    if (h->staging_bytes >= bytes) return SU_OK;
    for (int b = 0; b < 2; ++b) {
        if (h->d_staging[b]) { cudaFree(h->d_staging[b]); h->d_staging[b] = nullptr; }
        h->staging_bytes = 0;
        if (cudaMalloc(&h->d_staging[b], bytes) != cudaSuccess) { cudaGetLastError(); return fail(h, SU_ENOMEM, "device staging allocation failed"); }
    }
    h->staging_bytes = bytes;
    return SU_OK;
}

void free_graphs(su_lattice* h) {
    for (auto& kv : h->graphs) cudaGraphExecDestroy(kv.second);
    h->graphs.clear();
}

}  // namespace

extern "C" {

size_t su_lattice_bytes(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_storage s) {
    if (!dims_ok(Nc, Lx, Ly, Lz, Lt) || !size_supported(Lx, Ly, Lz, Lt) || (p != SU_FP32 && p != SU_FP64)) return 0;
    if (s != SU_STORE_FULL && s != SU_STORE_RECON12) return 0;
    if (s == SU_STORE_RECON12 && Nc != 3) return 0;
    const size_t Vhp = plane_sites((size_t)Lx * Ly * Lz * Lt / 2);
    const size_t b = 8 * Vhp * (size_t)elems_per_link(Nc, s) * 2 * (p == SU_FP64 ? 8 : 4);
    return (b + 255) / 256 * 256;
}

su_status su_lattice_create(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_lattice** out) {
    return su_lattice_create_ex(Nc, Lx, Ly, Lz, Lt, p, nullptr, out);
}

// Lt_glob / t0 / Lt_loc: the handle owns global time slices [t0, t0 + Lt_loc); slab = false: the whole lattice.
static su_status create_common(int Nc, int Lx, int Ly, int Lz, int Lt_glob, bool slab, int t0, int Lt_loc, su_precision p,
                               const su_options* opt, su_lattice** out) {
    if (!out) return SU_EINVAL;
    su_options o{};
    o.storage = SU_STORE_FULL; o.kernel = SU_KERNEL_AUTO; o.device = -1;
    if (opt) o = *opt;
    if (!dims_ok(Nc, Lx, Ly, Lz, Lt_glob)) return SU_EINVAL;
    if (p != SU_FP32 && p != SU_FP64) return SU_EINVAL;
    if (o.storage != SU_STORE_FULL && o.storage != SU_STORE_RECON12) return SU_EINVAL;
    if (o.storage == SU_STORE_RECON12 && Nc != 3) return SU_EINVAL;
    if (o.kernel != SU_KERNEL_AUTO && o.kernel != SU_KERNEL_SPECIALISED && o.kernel != SU_KERNEL_GENERIC) return SU_EINVAL;
    if (Nc > SU_MAX_NC) return SU_EUNSUPPORTED;
    if (!size_supported(Lx, Ly, Lz, slab ? Lt_loc + 2 : Lt_glob)) return SU_EUNSUPPORTED;
    if (o.kernel == SU_KERNEL_SPECIALISED && Nc > 4) return SU_EUNSUPPORTED;
    if (slab) {
        // whole 32-site tiles per time slice and parity, so that a halo slice of a plane is one contiguous range
        if (Lt_loc < 2 || (Lt_loc & 1) || t0 < 0 || t0 + Lt_loc > Lt_glob) return SU_EINVAL;
        if (((size_t)Lx * Ly * Lz / 2) % LINK_TILE) return SU_EUNSUPPORTED;
    }
    const int Lt = slab ? Lt_loc + 2 : Lt_glob;      // stored time slices

    su_lattice* h = new (std::nothrow) su_lattice;
    if (!h) return SU_ENOMEM;
    h->Nc = Nc;
    h->g.L[0] = Lx; h->g.L[1] = Ly; h->g.L[2] = Lz; h->g.L[3] = Lt;
    h->g.Lxh = Lx / 2;
    const size_t Vstore = (size_t)Lx * Ly * Lz * Lt;
    h->g.t_halo = slab ? 1 : 0;
    h->g.Lt_int = slab ? Lt_loc : Lt_glob;
    h->g.Lt_glob = Lt_glob;
    h->g.t0g = slab ? (t0 - 1 + Lt_glob) % Lt_glob : 0;
    h->g.Vsh = (unsigned)((size_t)Lx * Ly * Lz / 2);
    h->g.Vh_int = h->g.Vsh * (unsigned)h->g.Lt_int;
    h->V = (size_t)Lx * Ly * Lz * h->g.Lt_int;          // owned sites: what import / export move
    h->g.Vh = (unsigned)(Vstore / 2);
    h->g.Vhp = (unsigned)plane_sites(Vstore / 2);
    h->var.store = Nc == 2 ? STORE_QUAT : (o.storage == SU_STORE_RECON12 ? STORE_RECON12 : STORE_FULL);
    h->link_bytes = (size_t)elems_per_link(Nc, o.storage) * 2 * (p == SU_FP64 ? 8 : 4);
    h->g.Zc = traversal_z_chunk(h->g, h->link_bytes);
    h->prec = p;
    h->var.Nc = Nc; h->var.prec = (int)p;
    h->var.generic = (o.kernel == SU_KERNEL_GENERIC) || (o.kernel == SU_KERNEL_AUTO && Nc > 4);
    h->stream = (cudaStream_t)o.stream;

    cudaError_t e = cudaSuccess;
    if (o.device < 0) e = cudaGetDevice(&h->device); else h->device = o.device;
    if (e != cudaSuccess) { delete h; return SU_ECUDA; }
    DeviceGuard guard(h->device);
    h->links_bytes = su_lattice_bytes(Nc, Lx, Ly, Lz, Lt, p, o.storage);
    su_status st = SU_OK;
    if (o.buffer) {
        if (o.buffer_bytes < h->links_bytes || ((uintptr_t)o.buffer & 255u)) st = SU_ENOMEM;
        h->links = o.buffer;
    } else {
        if (cudaMalloc(&h->links, h->links_bytes) != cudaSuccess) st = SU_ENOMEM;
        h->owns_links = (st == SU_OK);
    }
    const unsigned Vs = (unsigned)Lx * Ly * Lz;
    // partial sums of the reductions: one per block; the row-per-lane kernels have as few as 4 sites per block
    const size_t npart = Nc > SUG_MAX_TEMPLATE_NC ? 2 * (size_t)h->g.Vh + 2 :
                         (h->var.generic ? 2 * ((size_t)h->g.Vh / ROWS_MIN_LINKS_PER_BLOCK + 1)
                                         : (size_t)plaquette_blocks(h->g.Vh) + 2 * (size_t)reduce_blocks(Vs)) + 2;
    if (st == SU_OK && cudaMalloc(&h->d_partials, npart * sizeof(double)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK && cudaMalloc(&h->d_result, 2 * sizeof(double)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK && cudaMallocHost(&h->h_result, 2 * sizeof(double)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK && cudaMalloc(&h->d_counters, 2 * sizeof(unsigned long long)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK && cudaMalloc(&h->d_sweep, sizeof(uint32_t)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK && cudaMemset(h->d_counters, 0, 2 * sizeof(unsigned long long)) != cudaSuccess) st = SU_ECUDA;
    if (st != SU_OK) { cudaGetLastError(); su_lattice_destroy(h); return st; }
    *out = h;
    return SU_OK;
}

su_status su_lattice_create_ex(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, const su_options* opt,
                               su_lattice** out) {
    return create_common(Nc, Lx, Ly, Lz, Lt, false, 0, Lt, p, opt, out);
}

su_status su_lattice_create_slab(int Nc, int Lx, int Ly, int Lz, int Lt_global, int t0, int Lt_local, su_precision p,
                                 const su_options* opt, su_lattice** out) {
    return create_common(Nc, Lx, Ly, Lz, Lt_global, true, t0, Lt_local, p, opt, out);
}

size_t su_slab_bytes(int Nc, int Lx, int Ly, int Lz, int Lt_local, su_precision p, su_storage s) {
    if (Lt_local < 2 || (Lt_local & 1)) return 0;
    return su_lattice_bytes(Nc, Lx, Ly, Lz, Lt_local + 2, p, s);
}

su_status su_slab_links(su_lattice* h, void** device_links, size_t* bytes) {
    if (!h || !device_links) return SU_EINVAL;
    *device_links = h->links;
    if (bytes) *bytes = h->links_bytes;
    return SU_OK;
}

su_status su_slab_set_peers(su_lattice* h, void* device_links_below, void* device_links_above) {
    if (!h || !device_links_below || !device_links_above) return SU_EINVAL;
    if (!h->g.t_halo) return fail(h, SU_ESTATE, "su_slab_set_peers on a lattice that is not a slab");
    DeviceGuard guard(h->device);
    free_graphs(h);                      // peer pointers are baked into captured launches
    h->peer_lo = device_links_below; h->peer_hi = device_links_above;
    return SU_OK;
}

su_status su_slab_halo_push(su_lattice* h) {
    if (!h) return SU_EINVAL;
    if (!h->g.t_halo) return fail(h, SU_ESTATE, "su_slab_halo_push on a lattice that is not a slab");
    if (!h->peer_lo || !h->peer_hi) return fail(h, SU_ESTATE, "slab lattice: su_slab_set_peers first");
    if (!h->ready) return fail(h, SU_ESTATE, "su_slab_halo_push before su_init_* / su_import_links");
    DeviceGuard guard(h->device);
    // per (mu, parity) plane a time slice is one contiguous range of whole tiles
    const size_t pair = 2 * (h->prec == SU_FP64 ? 8 : 4);
    const size_t E = (size_t)elems_per_link(h->Nc, h->var.store == STORE_RECON12 ? SU_STORE_RECON12 : SU_STORE_FULL);
    const size_t plane = E * h->g.Vhp * pair, slice = E * h->g.Vsh * pair;
    for (int pl = 0; pl < 8; ++pl) {
        const char* own = (const char*)h->links + pl * plane;
        char* lo = (char*)h->peer_lo + pl * plane;
        char* hi = (char*)h->peer_hi + pl * plane;
        // first owned slice (stored t = 1) -> upper halo of the slab below (their stored t = Lt_int + 1)
        SU_CUDA(h, cudaMemcpyAsync(lo + (size_t)(h->g.Lt_int + 1) * slice, own + slice, slice, cudaMemcpyDefault, h->stream), "halo push");
        // last owned slice (stored t = Lt_int) -> lower halo of the slab above (their stored t = 0)
        SU_CUDA(h, cudaMemcpyAsync(hi, own + (size_t)h->g.Lt_int * slice, slice, cudaMemcpyDefault, h->stream), "halo push");
    }
    h->halos_valid = true;
    return SU_OK;
}

su_status su_ipc_export(su_lattice* h, unsigned char handle[64]) {
    if (!h || !handle) return SU_EINVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
    if (!h->owns_links) return fail(h, SU_ESTATE, "su_ipc_export needs a library-owned link buffer (no caller buffer)");
    DeviceGuard guard(h->device);
    cudaIpcMemHandle_t m;
    SU_CUDA(h, cudaIpcGetMemHandle(&m, h->links), "cudaIpcGetMemHandle");
    memcpy(handle, &m, 64);
    return SU_OK;
}

su_status su_ipc_open(su_lattice* h, const unsigned char handle[64], void** device_ptr) {
    if (!h || !handle || !device_ptr) return SU_EINVAL;
    DeviceGuard guard(h->device);
    cudaIpcMemHandle_t m;
    memcpy(&m, handle, 64);
    void* ptr = nullptr;
    SU_CUDA(h, cudaIpcOpenMemHandle(&ptr, m, cudaIpcMemLazyEnablePeerAccess), "cudaIpcOpenMemHandle");
    *device_ptr = ptr;
    return SU_OK;
}

su_status su_ipc_close(su_lattice* h, void* device_ptr) {
    if (!h || !device_ptr) return SU_EINVAL;
    DeviceGuard guard(h->device);
    SU_CUDA(h, cudaIpcCloseMemHandle(device_ptr), "cudaIpcCloseMemHandle");
    return SU_OK;
}

su_status su_lattice_destroy(su_lattice* h) {
    if (!h) return SU_EINVAL;
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    free_graphs(h);
    free_fused(h);
    drain_timing(h);
    for (cudaEvent_t e : h->free_events) cudaEventDestroy(e);
    if (h->owns_links && h->links) cudaFree(h->links);
    if (h->d_partials) cudaFree(h->d_partials);
    if (h->d_result) cudaFree(h->d_result);
    if (h->h_result) cudaFreeHost(h->h_result);
    if (h->d_counters) cudaFree(h->d_counters);
    if (h->d_sweep) cudaFree(h->d_sweep);
    if (h->d_attempts) cudaFree(h->d_attempts);
    for (int b = 0; b < 2; ++b) {
        if (h->d_staging[b]) cudaFree(h->d_staging[b]);
        if (h->ev_filled[b]) cudaEventDestroy(h->ev_filled[b]);
        if (h->ev_drained[b]) cudaEventDestroy(h->ev_drained[b]);
    }
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    cudaGetLastError();
    delete h;
    return SU_OK;
}

static su_status init_common(su_lattice* h, uint64_t seed, bool hot) {
    if (!h) return SU_EINVAL;
    DeviceGuard guard(h->device);
    if (seed != h->seed) free_graphs(h);             // the Philox key is baked into captured launches
    h->seed = seed; h->sweep = 0; h->halos_valid = true;
    SU_CUDA(h, cudaMemsetAsync(h->d_counters, 0, 2 * sizeof(unsigned long long), h->stream), "counter reset");
    AuxArgs a = aux_args(h);
    if (hot) SU_CUDA(h, SU_BY_NC(h, init_hot_nc, h->var, a, h->stream, &h->n_launch), "hot start");
    else     SU_CUDA(h, SU_BY_NC(h, init_cold_nc, h->var, a, h->stream, &h->n_launch), "cold start");
    h->ready = true;
    return SU_OK;
}
su_status su_init_cold(su_lattice* h, uint64_t seed) { return init_common(h, seed, false); }
su_status su_init_hot(su_lattice* h, uint64_t seed) { return init_common(h, seed, true); }

su_status su_set_rng(su_lattice* h, uint64_t seed, uint32_t sweep_counter) {
    if (!h) return SU_EINVAL;
    if (seed != h->seed) { DeviceGuard guard(h->device); free_graphs(h); }   // the key is baked into captured launches
    h->seed = seed; h->sweep = sweep_counter;
    return SU_OK;
}

su_status su_sweep(su_lattice* h, double beta, int n_hb, int n_or) {
    if (!h) return SU_EINVAL;
    if (!(beta >= 0.0) || !std::isfinite(beta) || n_hb < 0 || n_or < 0 || n_hb > 255)
        return fail(h, SU_EINVAL, "su_sweep: beta must be finite and >= 0, 0 <= n_heatbath <= 255, n_overrelax >= 0");
    if (!h->ready) return fail(h, SU_ESTATE, "su_sweep before su_init_* / su_import_links");
    if (h->g.t_halo && !(h->peer_lo == h->links && h->peer_hi == h->links))
        return fail(h, SU_ESTATE, "su_sweep on one slab of several: drive su_substep on all slabs, one sub-step at a time");
    if (su_status hs = halos_ok(h, "su_sweep")) return hs;
    if (h->graph_mode && h->timing) return fail(h, SU_EUNSUPPORTED, "su_sweep: per-kind timing is not available in graph mode");
    DeviceGuard guard(h->device);
    for (int kind = 0; kind < 2; ++kind) {           // build the fused tables outside any stream capture
        if ((kind == KIND_HB ? n_hb : n_or) == 0 || effective_fuse(h, kind) <= 1) continue;
        for (int sub0 = 0; sub0 < 8; sub0 += h->fuse_g) {
            su_lattice::FusedTable* t = nullptr;
            su_status st = fused_table(h, kind, sub0, &t);
            if (st != SU_OK) return st;
        }
    }
    if (!h->graph_mode) {
        su_status st = enqueue_sweep(h, beta, n_hb, n_or, nullptr, h->timing);
        if (st != SU_OK) return st;
    } else {
        // the captured kernels read the sweep counter from device memory, so one graph serves every sweep
        auto key = std::make_tuple(beta, n_hb, n_or);
        auto it = h->graphs.find(key);
        if (it == h->graphs.end()) {
            if (h->graphs.size() >= 16) free_graphs(h);      // e.g. annealing over many beta: bound the cache
            cudaStream_t cap;
            SU_CUDA(h, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking), "graph capture stream");
            cudaStream_t user = h->stream;
            h->stream = cap;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
            su_status st = SU_OK;
            const uint64_t before = h->n_launch;
            if (e == cudaSuccess) st = enqueue_sweep(h, beta, n_hb, n_or, h->d_sweep, false);
            if (e == cudaSuccess) e = cudaStreamEndCapture(cap, &graph);
            h->graph_launches[key] = h->n_launch - before;
            h->n_launch = before;
            h->stream = user;
            cudaGraphExec_t exec = nullptr;
            if (e == cudaSuccess && st == SU_OK) e = cudaGraphInstantiate(&exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            cudaStreamDestroy(cap);
            if (st != SU_OK) return st;
            if (e != cudaSuccess) return cuda_fail(h, e, "graph capture");
            it = h->graphs.emplace(key, exec).first;
        }
        k_set_u32<<<1, 1, 0, h->stream>>>(h->d_sweep, h->sweep);
        SU_CUDA(h, cudaGetLastError(), "sweep counter upload");
        SU_CUDA(h, cudaGraphLaunch(it->second, h->stream), "graph launch");
        h->n_launch += 1 + h->graph_launches[key];
    }
    ++h->sweep;
    return SU_OK;
}

su_status su_substep(su_lattice* h, double beta, int kind, int pass, int parity, int mu, uint8_t* host_attempts) {
    if (!h) return SU_EINVAL;
    if (!(beta >= 0.0) || !std::isfinite(beta) || kind < 0 || kind > 1 || pass < 0 || pass > 255 || parity < 0 ||
        parity > 1 || mu < 0 || mu > 3)
        return fail(h, SU_EINVAL, "su_substep: argument out of range");
    if (!h->ready) return fail(h, SU_ESTATE, "su_substep before su_init_* / su_import_links");
    if (host_attempts && h->g.t_halo) return fail(h, SU_EUNSUPPORTED, "attempt counts are not exported in slab mode");
    if (su_status hs = halos_ok(h, "su_substep")) return hs;
    DeviceGuard guard(h->device);
    const size_t nsub = (size_t)h->Nc * (h->Nc - 1) / 2, nbytes = nsub * h->g.Vh;
    if (host_attempts) {
        if (!h->d_attempts && cudaMalloc(&h->d_attempts, nbytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(h, SU_ENOMEM, "attempt buffer allocation failed");
        }
        SU_CUDA(h, cudaMemsetAsync(h->d_attempts, 0, nbytes, h->stream), "attempt buffer reset");
    }
    su_status st = launch_substep(h, beta, kind, pass, parity, mu, host_attempts ? h->d_attempts : nullptr, nullptr, h->substep_reunit);
    if (st != SU_OK) return st;
    if (host_attempts) {
        SU_CUDA(h, cudaMemcpyAsync(host_attempts, h->d_attempts, nbytes, cudaMemcpyDeviceToHost, h->stream), "attempt copy");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_substep synchronise");
    }
    return SU_OK;
}

su_status su_plaquette(su_lattice* h, double* out) {
    if (!h || !out) return SU_EINVAL;
    if (!h->ready) return fail(h, SU_ESTATE, "su_plaquette before su_init_* / su_import_links");
    if (su_status hs = halos_ok(h, "su_plaquette")) return hs;
    DeviceGuard guard(h->device);
    AuxArgs a = aux_args(h);
    SU_CUDA(h, SU_BY_NC(h, plaquette_nc, h->var, a, h->stream, &h->n_launch), "plaquette kernels");
    double v = 0;
    SU_CUDA(h, cudaMemcpyAsync(h->h_result, h->d_result, sizeof(double), cudaMemcpyDeviceToHost, h->stream), "plaquette copy");
    SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_plaquette synchronise");
    v = h->h_result[0];
    if (su_status fs = check_fused_error(h)) return fs;
    *out = v;
    return SU_OK;
}

su_status su_polyakov(su_lattice* h, double out[2]) {
    if (!h || !out) return SU_EINVAL;
    if (!h->ready) return fail(h, SU_ESTATE, "su_polyakov before su_init_* / su_import_links");
    if (h->g.t_halo) return fail(h, SU_EUNSUPPORTED, "the Polyakov loop crosses slabs: not available in slab mode");
    DeviceGuard guard(h->device);
    AuxArgs a = aux_args(h);
    SU_CUDA(h, SU_BY_NC(h, polyakov_nc, h->var, a, h->stream, &h->n_launch), "polyakov kernels");
    double v[2] = {0, 0};
    SU_CUDA(h, cudaMemcpyAsync(h->h_result, h->d_result, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream), "polyakov copy");
    SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_polyakov synchronise");
    v[0] = h->h_result[0]; v[1] = h->h_result[1];
    out[0] = v[0]; out[1] = v[1];
    return SU_OK;
}

su_status su_reunitarize(su_lattice* h) {
    if (!h) return SU_EINVAL;
    if (!h->ready) return fail(h, SU_ESTATE, "su_reunitarize before su_init_* / su_import_links");
    if (su_status hs = halos_ok(h, "su_reunitarize")) return hs;
    DeviceGuard guard(h->device);
    AuxArgs a = aux_args(h);
    SU_CUDA(h, SU_BY_NC(h, reunit_nc, h->var, a, h->stream, &h->n_launch), "reunitarise kernel");
    return SU_OK;
}

// Layout conversion runs on the lattice's stream, the PCIe copy on a second stream; two staging buffers, so the
// conversion kernel of chunk i+1 overlaps the copy of chunk i (events order the hand-over in both directions).
static su_status transfer_links(su_lattice* h, double* host, size_t n_doubles, bool to_host) {
    const size_t per_site = 4 * 2 * (size_t)h->Nc * h->Nc;                  // doubles per site
    if (n_doubles != h->V * per_site) return fail(h, SU_EINVAL, "link array size must be 4 V * 2 Nc^2 doubles");
    DeviceGuard guard(h->device);
    const size_t chunk_sites_max = (size_t)(32u << 20) / (per_site * sizeof(double)) + 1;
    const size_t chunk_sites = chunk_sites_max < h->V ? chunk_sites_max : h->V;
    su_status st = ensure_staging(h, chunk_sites * per_site * sizeof(double));
    if (st != SU_OK) return st;
    int i = 0;
    for (size_t s0 = 0; s0 < h->V; s0 += chunk_sites, ++i) {
        const int b = i & 1;
        const size_t ns = (h->V - s0 < chunk_sites) ? h->V - s0 : chunk_sites;
        AuxArgs a = aux_args(h);
        a.staging = h->d_staging[b];
        a.site0 = (unsigned)s0; a.nsites = (unsigned)ns;
        double* hp = host + s0 * per_site;
        if (to_host) {
            if (i >= 2) SU_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_drained[b], 0), "export ordering");
            SU_CUDA(h, SU_BY_NC(h, export_nc, h->var, a, h->stream, &h->n_launch), "export kernel");
            SU_CUDA(h, cudaEventRecord(h->ev_filled[b], h->stream), "export ordering");
            SU_CUDA(h, cudaStreamWaitEvent(h->copy_stream, h->ev_filled[b], 0), "export ordering");
            SU_CUDA(h, cudaMemcpyAsync(hp, h->d_staging[b], ns * per_site * sizeof(double), cudaMemcpyDeviceToHost, h->copy_stream), "export copy");
            SU_CUDA(h, cudaEventRecord(h->ev_drained[b], h->copy_stream), "export ordering");
        } else {
            if (i >= 2) SU_CUDA(h, cudaStreamWaitEvent(h->copy_stream, h->ev_drained[b], 0), "import ordering");
            SU_CUDA(h, cudaMemcpyAsync(h->d_staging[b], hp, ns * per_site * sizeof(double), cudaMemcpyHostToDevice, h->copy_stream), "import copy");
            SU_CUDA(h, cudaEventRecord(h->ev_filled[b], h->copy_stream), "import ordering");
            SU_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_filled[b], 0), "import ordering");
            SU_CUDA(h, SU_BY_NC(h, import_nc, h->var, a, h->stream, &h->n_launch), "import kernel");
            SU_CUDA(h, cudaEventRecord(h->ev_drained[b], h->stream), "import ordering");
        }
    }
    SU_CUDA(h, cudaStreamSynchronize(h->copy_stream), "link transfer synchronise");
    SU_CUDA(h, cudaStreamSynchronize(h->stream), "link transfer synchronise");
    return SU_OK;
}

su_status su_export_links(su_lattice* h, double* host_dst, size_t n_doubles) {
    if (!h || !host_dst) return SU_EINVAL;
    if (!h->ready) return fail(h, SU_ESTATE, "su_export_links before su_init_* / su_import_links");
    return transfer_links(h, host_dst, n_doubles, true);
}

su_status su_import_links(su_lattice* h, const double* host_src, size_t n_doubles) {
    if (!h || !host_src) return SU_EINVAL;
    su_status st = transfer_links(h, const_cast<double*>(host_src), n_doubles, false);
    if (st == SU_OK) { h->ready = true; if (h->g.t_halo) h->halos_valid = false; }
    return st;
}

// ---- configuration files ("file storing ... configurations") ----
namespace {
struct ConfigHeader {          // 64 bytes, little-endian
    char magic[8];             // "SUGCONF1"
    int32_t Nc, L[4], precision, storage, reserved;
    uint64_t seed;
    uint32_t sweep, pad;
    double plaquette;          // of the stored configuration, recomputed and compared on load
};
static_assert(sizeof(ConfigHeader) == 64, "configuration file header");
uint64_t fnv1a(const void* p, size_t n, uint64_t h) {
    const unsigned char* b = (const unsigned char*)p;
    for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    return h;
}
}  // namespace

su_status su_save_config(su_lattice* h, const char* path) {
    if (!h || !path) return SU_EINVAL;
    if (!h->ready) return fail(h, SU_ESTATE, "su_save_config before su_init_* / su_import_links");
    if (h->g.t_halo) return fail(h, SU_EUNSUPPORTED, "su_save_config: export the slabs and write them from the driver");
    ConfigHeader hd{};
    memcpy(hd.magic, "SUGCONF1", 8);
    hd.Nc = h->Nc; for (int d = 0; d < 4; ++d) hd.L[d] = h->g.L[d];
    hd.precision = (int)h->prec; hd.storage = h->var.store == STORE_RECON12 ? 1 : 0;
    hd.seed = h->seed; hd.sweep = h->sweep;
    su_status st = su_plaquette(h, &hd.plaquette);
    if (st != SU_OK) return st;
    const size_t n = h->V * 4 * 2 * (size_t)h->Nc * h->Nc;
    std::vector<double> buf;
    try { buf.resize(n); } catch (...) { return fail(h, SU_ENOMEM, "su_save_config: host buffer"); }
    st = su_export_links(h, buf.data(), n);
    if (st != SU_OK) return st;
    FILE* f = fopen(path, "wb");
    if (!f) return fail(h, SU_EINVAL, "su_save_config: cannot open '%s' for writing", path);
    const uint64_t sum = fnv1a(buf.data(), n * sizeof(double), fnv1a(&hd, sizeof(hd), 14695981039346656037ull));
    const bool ok = fwrite(&hd, sizeof(hd), 1, f) == 1 && fwrite(buf.data(), sizeof(double), n, f) == n && fwrite(&sum, 8, 1, f) == 1;
    if (fclose(f) != 0 || !ok) return fail(h, SU_EINVAL, "su_save_config: write to '%s' failed", path);
    return SU_OK;
}

su_status su_load_config(su_lattice* h, const char* path) {
    if (!h || !path) return SU_EINVAL;
    if (h->g.t_halo) return fail(h, SU_EUNSUPPORTED, "su_load_config: read the file in the driver and import the slabs");
    FILE* f = fopen(path, "rb");
    if (!f) return fail(h, SU_EINVAL, "su_load_config: cannot open '%s'", path);
    ConfigHeader hd{};
    const size_t n = h->V * 4 * 2 * (size_t)h->Nc * h->Nc;
    std::vector<double> buf;
    uint64_t sum = 0;
    bool ok = fread(&hd, sizeof(hd), 1, f) == 1 && !memcmp(hd.magic, "SUGCONF1", 8);
    if (ok && (hd.Nc != h->Nc || hd.L[0] != h->g.L[0] || hd.L[1] != h->g.L[1] || hd.L[2] != h->g.L[2] || hd.L[3] != h->g.L[3])) {
        fclose(f);
        return fail(h, SU_EINVAL, "su_load_config: '%s' holds another group or lattice", path);
    }
    if (ok) { try { buf.resize(n); } catch (...) { fclose(f); return fail(h, SU_ENOMEM, "su_load_config: host buffer"); } }
    ok = ok && fread(buf.data(), sizeof(double), n, f) == n && fread(&sum, 8, 1, f) == 1;
    fclose(f);
    if (!ok) return fail(h, SU_EINVAL, "su_load_config: '%s' is not a complete configuration file", path);
    if (sum != fnv1a(buf.data(), n * sizeof(double), fnv1a(&hd, sizeof(hd), 14695981039346656037ull)))
        return fail(h, SU_EINVAL, "su_load_config: checksum mismatch in '%s'", path);
    if ((hd.precision != (int)SU_FP32 && hd.precision != (int)SU_FP64) || (hd.storage != (int)SU_STORE_FULL && hd.storage != (int)SU_STORE_RECON12) ||
        (hd.storage == (int)SU_STORE_RECON12 && hd.Nc != 3) || hd.reserved != 0 || !std::isfinite(hd.plaquette))
        return fail(h, SU_EINVAL, "su_load_config: header of '%s' holds values outside their range", path);
    // Up to here the handle is untouched. The links have to be on the device before their plaquette can be measured,
    // so a file that fails this last check does overwrite them: the lattice then counts as uninitialised (SU_ESTATE
    // until su_init_* / su_import_links / another load) instead of silently holding the rejected configuration.
    // RNG seed and sweep counter are only taken over once everything has passed.
    su_status st = su_import_links(h, buf.data(), n);
    if (st != SU_OK) return st;
    // the stored plaquette was measured in the writer's precision and storage; a reader in fp32 / two-row storage rounds the links
    double plaq = 0;
    st = su_plaquette(h, &plaq);
    if (st != SU_OK) { h->ready = false; return st; }
    const double tol = (h->prec == SU_FP64 && hd.precision == (int)SU_FP64) ? 1e-12 : 1e-5;
    if (!(std::fabs(plaq - hd.plaquette) <= tol)) {
        h->ready = false;
        return fail(h, SU_EINVAL, "su_load_config: plaquette of '%s' does not match its header; the lattice is now uninitialised", path);
    }
    return su_set_rng(h, hd.seed, hd.sweep);
}

su_status su_get_counters(su_lattice* h, uint64_t* kp_attempts_total, uint64_t* kp_exhausted) {
    if (!h) return SU_EINVAL;
    DeviceGuard guard(h->device);
    unsigned long long v[2] = {0, 0};
    SU_CUDA(h, cudaMemcpyAsync(v, h->d_counters, sizeof(v), cudaMemcpyDeviceToHost, h->stream), "counter copy");
    SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_get_counters synchronise");
    if (su_status fs = check_fused_error(h)) return fs;
    if (kp_attempts_total) *kp_attempts_total = v[0];
    if (kp_exhausted) *kp_exhausted = v[1];
    return SU_OK;
}

su_status su_synchronize(su_lattice* h) {
    if (!h) return SU_EINVAL;
    DeviceGuard guard(h->device);
    SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_synchronize");
    return check_fused_error(h);
}

su_status su_set_graph_mode(su_lattice* h, int enabled) {
    if (!h) return SU_EINVAL;
    if (enabled && h->timing) return fail(h, SU_EUNSUPPORTED, "su_set_graph_mode: per-kind timing is on (events cannot be read back from a replayed graph)");
    h->graph_mode = enabled != 0;
    return SU_OK;
}

su_status su_set_timing(su_lattice* h, int enabled) {
    if (!h) return SU_EINVAL;
    if (enabled && h->graph_mode) return fail(h, SU_EUNSUPPORTED, "su_set_timing: not available in graph mode");
    DeviceGuard guard(h->device);
    drain_timing(h);
    h->timing = enabled != 0;
    h->hb_ms = h->or_ms = 0; h->hb_launches = h->or_launches = 0;
    return SU_OK;
}

su_status su_get_timing(su_lattice* h, double* hb_ms, uint64_t* hb_launches, double* or_ms, uint64_t* or_launches) {
    if (!h) return SU_EINVAL;
    DeviceGuard guard(h->device);
    drain_timing(h);
    if (hb_ms) *hb_ms = h->hb_ms;
    if (or_ms) *or_ms = h->or_ms;
    if (hb_launches) *hb_launches = h->hb_launches;
    if (or_launches) *or_launches = h->or_launches;
    return SU_OK;
}

su_status su_get_launch_count(su_lattice* h, uint64_t* out) {
    if (!h || !out) return SU_EINVAL;
    *out = h->n_launch;
    return SU_OK;
}

su_status su_set_option(su_lattice* h, const char* name, long long value) {
    if (!h || !name) return SU_EINVAL;
    DeviceGuard guard(h->device);
    if (!strcmp(name, "z_chunk_planes")) {
        // traversal order of the update / plaquette kernels: planes per z-chunk, a divisor of Lz (0 = the default rule)
        if (value < 0 || value > h->g.L[2] || (value > 0 && h->g.L[2] % value)) return fail(h, SU_EINVAL, "z_chunk_planes must divide Lz");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        free_fused(h);
        h->g.Zc = value > 0 ? (int)value : traversal_z_chunk(h->g, h->link_bytes);
        return SU_OK;
    }
    if (!strcmp(name, "reunit_on_store")) {
        if (value != 0 && value != 1) return fail(h, SU_EINVAL, "reunit_on_store must be 0 or 1");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        h->reunit_on_store = value != 0;
        return SU_OK;
    }
    if (!strcmp(name, "coop_sweep")) {
        if (value != 0 && value != 1) return fail(h, SU_EINVAL, "coop_sweep must be 0 or 1");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        h->coop_sweep = value != 0;
        return SU_OK;
    }
    if (!strcmp(name, "block_tile_z") || !strcmp(name, "block_tile_t")) {
        if (value < 1 || value > 8) return fail(h, SU_EINVAL, "%s must be in 1...8", name);
        if (!SUG_BLOCK_TILES && value != 1) return fail(h, SU_EUNSUPPORTED, "%s: this library was built without -DSUG_BLOCK_TILES=1", name);
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        (name[11] == 'z' ? h->tile_z : h->tile_t) = (int)value;
        return SU_OK;
    }
    if (!strcmp(name, "prefetch_slices") || !strcmp(name, "blocks_per_sm")) {
        if (value < 0 || value > 64) return fail(h, SU_EINVAL, "%s must be in 0...64", name);
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        (name[0] == 'p' ? h->prefetch_slices : h->blocks_per_sm) = (int)value;
        return SU_OK;
    }
    if (!strcmp(name, "substep_reunit")) {
        if (value != 0 && value != 1) return fail(h, SU_EINVAL, "substep_reunit must be 0 or 1");
        if (value && !reunit_in_kernel(h)) return fail(h, SU_EUNSUPPORTED, "substep_reunit: only the register kernels of Nc <= 4 reunitarise before the store");
        h->substep_reunit = value != 0;
        return SU_OK;
    }
    if (!strcmp(name, "fuse_wait_ns")) {
        if (value < 0) return fail(h, SU_EINVAL, "fuse_wait_ns must be >= 0");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);                  // the limit is an argument of the captured launches
        h->fuse_wait_ns = (unsigned long long)value;
        return SU_OK;
    }
    const bool is_fuse = !strcmp(name, "fuse"), is_chunk = !strcmp(name, "fuse_chunk_planes"), is_margin = !strcmp(name, "fuse_margin"),
               is_cell = !strcmp(name, "fuse_cell_planes");
    if (is_fuse || is_chunk || is_margin || is_cell) {
        if (is_fuse && value != 1 && value != 2 && value != 4 && value != 8) return fail(h, SU_EINVAL, "fuse must be 1, 2, 4 or 8");
        if ((is_chunk || is_cell) && (value < 0 || value > h->g.L[2] || (value > 0 && h->g.L[2] % value)))
            return fail(h, SU_EINVAL, "%s must divide Lz", name);
        if (is_margin && (value < 1 || value > 1000000)) return fail(h, SU_EINVAL, "fuse_margin must be >= 1");
        SU_CUDA(h, cudaStreamSynchronize(h->stream), "su_set_option");
        free_graphs(h);
        free_fused(h);
        if (is_fuse) h->fuse_g = (int)value;
        if (is_chunk) h->fuse_chunk_planes = (int)value;
        if (is_margin) h->fuse_margin = (int)value;
        if (is_cell) h->fuse_cell_planes = (int)value;
        return SU_OK;
    }
    return fail(h, SU_EINVAL, "su_set_option: unknown option '%s'", name);
}

su_status su_get_option(su_lattice* h, const char* name, long long* value) {
    if (!h || !name || !value) return SU_EINVAL;
    if (!strcmp(name, "z_chunk_planes")) { *value = h->g.Zc; return SU_OK; }
    if (!strcmp(name, "reunit_on_store")) { *value = h->reunit_on_store ? 1 : 0; return SU_OK; }
    if (!strcmp(name, "coop_sweep")) { *value = h->coop_sweep ? 1 : 0; return SU_OK; }
    if (!strcmp(name, "coop_sweep_effective")) { *value = (coop_fits(h, 0) ? 1 : 0) | (coop_fits(h, 1) ? 2 : 0); return SU_OK; }
    if (!strcmp(name, "block_tiles_supported")) { *value = SUG_BLOCK_TILES; return SU_OK; }
    if (!strcmp(name, "block_tile_z")) { *value = h->tile_z; return SU_OK; }
    if (!strcmp(name, "block_tile_t")) { *value = h->tile_t; return SU_OK; }
    if (!strcmp(name, "prefetch_slices")) { *value = h->prefetch_slices; return SU_OK; }
    if (!strcmp(name, "blocks_per_sm")) { *value = h->blocks_per_sm; return SU_OK; }
    if (!strcmp(name, "fuse")) { *value = h->fuse_g; return SU_OK; }
    if (!strcmp(name, "fuse_chunk_planes")) { *value = h->fuse_chunk_planes; return SU_OK; }
    if (!strcmp(name, "fuse_margin")) { *value = h->fuse_margin; return SU_OK; }
    if (!strcmp(name, "fuse_wait_ns")) { *value = (long long)h->fuse_wait_ns; return SU_OK; }
    if (!strcmp(name, "substep_reunit")) { *value = h->substep_reunit ? 1 : 0; return SU_OK; }
    if (!strcmp(name, "fuse_cell_planes")) { *value = h->fuse_cell_planes; return SU_OK; }
    if (!strcmp(name, "fuse_effective")) { *value = std::max(effective_fuse(h, 0), effective_fuse(h, 1)); return SU_OK; }
    return fail(h, SU_EINVAL, "su_get_option: unknown option '%s'", name);
}

su_status su_slab_plaquette_sum(su_lattice* const* slabs, int n_slabs, double* out) {
    if (!slabs || n_slabs < 1 || !out) return SU_EINVAL;
    double sum = 0;
    for (int r = 0; r < n_slabs; ++r) {
        double share = 0;
        su_status st = su_plaquette(slabs[r], &share);
        if (st != SU_OK) return st;
        sum += share;
    }
    *out = sum;
    return SU_OK;
}

su_status su_measure_fma_peak(int device, su_precision p, double* tflops, double* ms) {
    if (!tflops || (p != SU_FP32 && p != SU_FP64)) return SU_EINVAL;
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return SU_ECUDA;
    DeviceGuard guard(dev);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SU_ECUDA;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = p == SU_FP64 ? 4096 : 16384;
    void *in = nullptr, *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    su_status st = SU_OK;
    const double host_in64[3] = {1.0000001, 1e-9, 0.5};
    const float host_in32[3] = {1.0000001f, 1e-9f, 0.5f};
    if (cudaMalloc(&in, 3 * sizeof(double)) != cudaSuccess || cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) != cudaSuccess ||
        cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) st = SU_ENOMEM;
    float best = 0;
    if (st == SU_OK) {
        cudaMemcpy(in, p == SU_FP64 ? (const void*)host_in64 : (const void*)host_in32, p == SU_FP64 ? 24 : 12, cudaMemcpyHostToDevice);
        for (int rep = 0; rep < 6 && st == SU_OK; ++rep) {          // first repetition = warm-up
            cudaEventRecord(e0, 0);
            if (p == SU_FP64) k_fma_peak<double><<<blocks, threads>>>((double*)out, (const double*)in, iters);
            else              k_fma_peak<float><<<blocks, threads>>>((float*)out, (const float*)in, iters);
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess) { st = SU_ECUDA; break; }
            float t = 0;
            cudaEventElapsedTime(&t, e0, e1);
            if (rep > 0 && (best == 0 || t < best)) best = t;
        }
    }
    if (in) cudaFree(in);
    if (out) cudaFree(out);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (st != SU_OK) { cudaGetLastError(); return st; }
    const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;     // 64 FMAs per iteration per thread
    *tflops = flops / ((double)best * 1e-3) / 1e12;
    if (ms) *ms = best;
    return SU_OK;
}

su_status su_measure_l2_peak(int device, int through_l1, double* gbs, double* ms, double* bytes_per_clock) {
    if (!gbs) return SU_EINVAL;
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return SU_ECUDA;
    DeviceGuard guard(dev);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SU_ECUDA;
    const size_t bytes = 24u << 20, n16 = bytes / 16;           // 24 MB: a fifth of L2, far beyond the SMs' L1
    const int blocks = prop.multiProcessorCount * 4, threads = 256, passes = 1;
    void *buf = nullptr, *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    su_status st = SU_OK;
    if (cudaMalloc(&buf, bytes) != cudaSuccess || cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) != cudaSuccess ||
        cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) st = SU_ENOMEM;
    float best = 0;
    double clocks = 0;
    if (st == SU_OK) {
        cudaMemset(buf, 0, bytes);
        for (int rep = 0; rep < 6 && st == SU_OK; ++rep) {          // first repetition = warm-up (brings the buffer into L2)
            cudaEventRecord(e0, 0);
            if (through_l1) k_l2_peak<1><<<blocks, threads>>>((double*)out, (const double2*)buf, n16, passes);
            else            k_l2_peak<0><<<blocks, threads>>>((double*)out, (const double2*)buf, n16, passes);
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess) { st = SU_ECUDA; break; }
            float t = 0;
            cudaEventElapsedTime(&t, e0, e1);
            if (rep > 0 && (best == 0 || t < best)) {
                best = t;
                cudaMemcpy(&clocks, out, sizeof(double), cudaMemcpyDeviceToHost);
            }
        }
    }
    if (buf) cudaFree(buf);
    if (out) cudaFree(out);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (st != SU_OK) { cudaGetLastError(); return st; }
    // every block reads ceil(n16 / (8 * threads)) * 8 * threads elements per pass
    const double per_block = (double)((n16 + (size_t)threads * 8 - 1) / ((size_t)threads * 8)) * threads * 8 * 16.0 * passes;
    *gbs = per_block * blocks / ((double)best * 1e-3) / 1e9;
    if (ms) *ms = best;
    if (bytes_per_clock) *bytes_per_clock = clocks > 0 ? per_block * blocks / clocks : 0.0;
    return SU_OK;
}

su_status su_debug_kp_math(int device, const uint32_t* words, size_t n, double* out) {
    if (!words || !out || n == 0) return SU_EINVAL;
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return SU_ECUDA;
    DeviceGuard guard(dev);
    uint32_t* d_w = nullptr;
    double* d_o = nullptr;
    su_status st = SU_OK;
    if (cudaMalloc(&d_w, n * sizeof(uint32_t)) != cudaSuccess || cudaMalloc(&d_o, n * 5 * sizeof(double)) != cudaSuccess) st = SU_ENOMEM;
    if (st == SU_OK) {
        cudaMemcpy(d_w, words, n * sizeof(uint32_t), cudaMemcpyHostToDevice);
        k_debug_kp_math<<<(unsigned)((n + 255) / 256), 256>>>(d_w, n, d_o);
        if (cudaMemcpy(out, d_o, n * 5 * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) st = SU_ECUDA;
    }
    if (d_w) cudaFree(d_w);
    if (d_o) cudaFree(d_o);
    if (st != SU_OK) cudaGetLastError();
    return st;
}

const char* su_last_error(const su_lattice* h) { return h ? h->err : kNullHandle; }

}  // extern "C"
