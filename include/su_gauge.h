/*
 * su_gauge.h — C ABI of libsugauge: B200 (sm_100a) Monte Carlo generation of 4-D SU(Nc) pure-gauge
 * (Wilson action) configurations: Cabibbo-Marinari pseudo-heatbath with Kennedy-Pendleton SU(2)
 * draws + microcanonical overrelaxation on even/odd checkerboards, plaquette and Polyakov-loop
 * reductions. Method: Cardoso & Bicudo, arXiv:1112.4533 ("PAPER.md" below = its text, cited by line).
 *
 * Conventions
 *  - Every call returns su_status; nothing throws, aborts or exits across this boundary.
 *    Out-parameters are written only on SU_OK. su_last_error() gives a text for the last failure.
 *  - Pointers are HOST pointers unless the name/documentation says "device".
 *  - A lattice handle is bound to one CUDA device and one stream; calls on one handle must not be
 *    made concurrently from several host threads. Kernels are enqueued on the handle's stream.
 *  - Geometry: periodic Lx x Ly x Lz x Lt lattice, every extent even and >= 2
 *    (checkerboard + periodic boundary), site index i = x + Lx (y + Ly (z + Lz t)), directions
 *    mu = 0..3 <-> x,y,z,t, parity = (x+y+z+t) mod 2.
 *  - Device storage: structure of arrays
 *        links[mu][parity][elem][cb],  cb = i / 2  (checkerboard index, x fastest),
 *    one array of (re,im) pairs per matrix element: Nc=2 -> 2 pairs (a0,a1),(a2,a3) of eq 6
 *    (PAPER.md:70,153); Nc=3 -> 9 pairs, or 6 pairs (first two rows) in RECON12;
 *    Nc>=4 -> Nc^2 pairs.
 *  - Randomness: counter-based Philox4x32-10 keyed by (seed; site, sweep, kind, pass, parity, mu,
 *    subgroup, attempt). No RNG state is stored; (seed, sweep counter, links) determine the chain.
 */
#ifndef SU_GAUGE_H
#define SU_GAUGE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default) /* the library itself is built with -fvisibility=hidden */
#endif

typedef struct su_lattice su_lattice; /* opaque, owned by the library */

typedef enum {
    SU_OK = 0,
    SU_EINVAL = 1,       /* NULL pointer, odd or <2 extent, Nc<2, bad beta/pass counts/sizes, RECON12 with Nc!=3 */
    SU_EUNSUPPORTED = 2, /* Nc above the generic kernel's limit (SU_MAX_NC); V >= 2^30 sites (32-bit link indices) */
    SU_ENOMEM = 3,       /* host or device allocation failed / caller buffer too small */
    SU_ECUDA = 4,        /* CUDA error (sticky; text via su_last_error) */
    SU_ESTATE = 5        /* sweep / measurement / export before init or import */
} su_status;

typedef enum { SU_FP32 = 0, SU_FP64 = 1 } su_precision;
typedef enum { SU_STORE_FULL = 0, SU_STORE_RECON12 = 1 } su_storage; /* RECON12: Nc == 3 only */
typedef enum {
    SU_KERNEL_AUTO = 0,        /* specialised for Nc = 2,3,4, generic otherwise */
    SU_KERNEL_SPECIALISED = 1, /* register-resident kernels; SU_EUNSUPPORTED for Nc > 4 */
    SU_KERNEL_GENERIC = 2      /* the generic SU(Nc) kernel at any supported Nc */
} su_kernel;

#define SU_MAX_NC 32 /* Nc <= 8: kernels compiled per Nc; 9..32: the runtime-Nc warp-per-link kernels */

typedef struct {
    su_storage storage;
    su_kernel kernel;
    int device;          /* CUDA device ordinal; -1 = current device */
    void* stream;        /* cudaStream_t to enqueue on; NULL = the legacy default stream */
    void* buffer;        /* DEVICE pointer to caller-owned link storage (e.g. a torch uint8 tensor),
                            256-byte aligned, or NULL: the library allocates. Must outlive the handle. */
    size_t buffer_bytes; /* size of buffer; must be >= su_lattice_bytes(...) */
} su_options;

/* Bytes of device link storage for this lattice: 4 V * R * sizeof(real), R = reals per link
 * (4 / 18 / 12 / 2 Nc^2), rounded up to 256. Returns 0 on invalid arguments. */
size_t su_lattice_bytes(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_storage s);

/* Create a lattice. The links are undefined until su_init_* / su_import_links. */
su_status su_lattice_create(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_lattice** out);
su_status su_lattice_create_ex(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p,
                               const su_options* opt, su_lattice** out);
su_status su_lattice_destroy(su_lattice*); /* synchronises the stream; frees what the library owns */

/* Cold start: all links = identity. Sets the RNG seed, sweep counter = 0. */
su_status su_init_cold(su_lattice*, uint64_t seed);
/* Hot start: independent Haar-random SU(Nc) links drawn from Philox(seed);
 * sweep counter = 0. Asynchronous on the stream. */
su_status su_init_hot(su_lattice*, uint64_t seed);

/* One Monte Carlo sweep: n_heatbath (pseudo-)heatbath passes
 * (eqs 9-16) followed by n_overrelax overrelaxation passes (eq 17); each pass updates every link
 * once, as 8 sub-steps: parity 0,1 (outer) x mu 0..3 (inner). Wilson coupling beta = 2Nc/g^2
 * (eq 3). Asynchronous on the stream. Uses, then increments, the handle's sweep counter.
 * Never reunitarises (unless su_set_option "reunit_on_store" asks for it). 0 <= n_heatbath <= 255, n_overrelax >= 0, beta finite and >= 0. */
su_status su_sweep(su_lattice*, double beta, int n_heatbath, int n_overrelax);

/* Mean plaquette <ReTr P>/Nc over the 6V plaquettes (eq 4); fp64 accumulation.
 * Synchronises the stream. Cold start gives exactly 1. */
su_status su_plaquette(su_lattice*, double* out);
/* Polyakov loop: mean over spatial sites of Tr prod_{t} U_3(x,t) / Nc; out = {re, im}. Synchronises. */
su_status su_polyakov(su_lattice*, double out[2]);
/* Project every link back to SU(Nc): Nc=2 normalise; Nc=3 Gram-Schmidt on
 * rows 0,1 + cross product; Nc>=4 Gram-Schmidt + phase on the last row. Asynchronous. */
su_status su_reunitarize(su_lattice*);

/* Copy the links to / from a HOST array of doubles in the canonical layout
 * [t][z][y][x][mu][row][col][re,im]; n_doubles must equal 4 V * 2 Nc^2. RECON12 rebuilds / drops
 * the third row. Synchronise. su_import_links marks the lattice initialised. */
su_status su_export_links(su_lattice*, double* host_dst, size_t n_doubles);
su_status su_import_links(su_lattice*, const double* host_src, size_t n_doubles);

/* Configuration files ("file storing ... configurations"): a 64-byte header ("SUGCONF1", Nc, extents,
 * precision, storage, RNG seed and sweep counter, plaquette), the links as canonical doubles (the su_export_links
 * layout), and a 64-bit FNV-1a checksum of both. su_load_config needs a handle of the same Nc and extents (any
 * precision / storage), verifies the checksum and that the plaquette it measures after the import matches the
 * header, and restores the RNG seed and sweep counter: load + su_sweep continues the writer's chain exactly when
 * precision and storage agree. Host-side I/O; both synchronise. Not available on slab handles.
 * A file that cannot be opened, is truncated, belongs to another lattice, has header fields out of range or a wrong
 * checksum is refused (SU_EINVAL) with the handle untouched. The plaquette can only be compared after the links are on
 * the device: a file that fails that last check has overwritten the links, and the handle is then uninitialised
 * (SU_ESTATE until su_init_* / su_import_links / a successful load); its RNG seed and sweep counter are unchanged. */
su_status su_save_config(su_lattice*, const char* path);
su_status su_load_config(su_lattice*, const char* path);

/* ---- test / resume hooks ---- */
/* Set the RNG seed and sweep counter: export + su_set_rng + import is an exact resume. */
su_status su_set_rng(su_lattice*, uint64_t seed, uint32_t sweep_counter);
/* One sub-step of a sweep: kind 0 = heatbath, 1 = overrelaxation; pass = heatbath pass number
 * (RNG counter field); parity 0/1; mu 0..3. host_attempts: NULL, or n_sub * V/2 bytes receiving
 * the Kennedy-Pendleton attempts used per [subgroup][cb] (0 = none / exhausted); when given the
 * call synchronises. Does not touch the sweep counter. */
su_status su_substep(su_lattice*, double beta, int kind, int pass, int parity, int mu, uint8_t* host_attempts);
/* Totals since the last init: KP attempts used, and subgroup draws abandoned after 1024 attempts
 * or a null projection (those leave the link unchanged for that subgroup). Synchronises. */
su_status su_get_counters(su_lattice*, uint64_t* kp_attempts_total, uint64_t* kp_exhausted);
/* Stream synchronise (surfaces asynchronous errors). */
su_status su_synchronize(su_lattice*);
/* Per-handle toggle: capture each distinct (beta, n_hb, n_or) sweep into a CUDA graph and replay it
 * (launch-bound small lattices). Default off. At most 16 graphs are cached per handle; a new seed
 * (su_init_*, su_set_rng) or new peers drop them. SU_EUNSUPPORTED while su_set_timing is on. */
su_status su_set_graph_mode(su_lattice*, int enabled);
/* Per-kind device timing of su_sweep (for the benchmark's roofline): when enabled (and graph mode
 * is off) su_sweep records CUDA events on the handle's stream before the heatbath passes, between
 * the heatbath and overrelaxation passes, and after; su_get_timing synchronises and returns the
 * accumulated milliseconds and update SUB-STEPS per kind (8 per pass, however many launches ran them) since su_set_timing.
 * SU_EUNSUPPORTED in graph mode (events cannot be read back from a replayed graph). */
su_status su_set_timing(su_lattice*, int enabled);
su_status su_get_timing(su_lattice*, double* hb_ms, uint64_t* hb_launches, double* or_ms, uint64_t* or_launches);
/* Number of kernels this handle has launched so far (for the benchmark's gpu_launches). */
su_status su_get_launch_count(su_lattice*, uint64_t* out);

/* ---- t-slab decomposition over several GPUs (Fig. 2: "each GPU holds Lt/n + 2 slices") ----
 * A slab handle owns the global time slices [t0, t0 + Lt_local) of an Lx x Ly x Lz x Lt_global lattice and
 * stores one halo slice below and one above them. Lt_local even and >= 2, the same on every slab;
 * Lx Ly Lz / 2 a multiple of 32 (else SU_EUNSUPPORTED). The Philox site index is the GLOBAL one, so n slabs
 * reproduce the single-lattice chain exactly.
 *   - su_slab_set_peers: DEVICE pointers (valid on this handle's device: same process, peer access, or
 *     su_ipc_open) to the link buffers of the slabs below (t0 - Lt_local) and above (t0 + Lt_local),
 *     periodically; a lattice cut into one slab names itself twice. The update kernel stores every link of
 *     the first / last owned slice into that neighbour's halo as well (fused halo push: no separate exchange).
 *   - Ordering is the caller's: sub-step k+1 may start on any slab only after sub-step k has finished on
 *     its neighbours (stream order in one process; a stream-ordered collective or event across processes).
 *     su_sweep therefore returns SU_ESTATE on one slab of several; drive su_substep. Sub-step (p, mu) never
 *     reads the halo plane (mu, p), which is the only one its neighbours write meanwhile.
 *   - su_init_cold / su_init_hot / su_reunitarize fill or transform the halos consistently by themselves;
 *     after su_import_links every slab must call su_slab_halo_push once all slabs have imported; until it
 *     has, su_sweep / su_substep / su_plaquette / su_reunitarize on that slab return SU_ESTATE.
 *   - su_plaquette returns this slab's SHARE (sum over slabs = the plaquette); su_polyakov and the
 *     attempt-count output of su_substep are SU_EUNSUPPORTED; import / export move the owned slices,
 *     n_doubles = 4 * Lx Ly Lz Lt_local * 2 Nc^2.
 *   - su_slab_bytes: size of the link buffer (0 on invalid arguments). su_slab_links: its device address.
 *   - su_ipc_export / su_ipc_open / su_ipc_close: CUDA IPC handle (64 bytes) of a library-owned link buffer,
 *     for peers in other processes. */
su_status su_lattice_create_slab(int Nc, int Lx, int Ly, int Lz, int Lt_global, int t0, int Lt_local,
                                 su_precision p, const su_options* opt, su_lattice** out);
size_t    su_slab_bytes(int Nc, int Lx, int Ly, int Lz, int Lt_local, su_precision p, su_storage s);
su_status su_slab_links(su_lattice*, void** device_links, size_t* bytes);
su_status su_slab_set_peers(su_lattice*, void* device_links_below, void* device_links_above);
su_status su_slab_halo_push(su_lattice*);
su_status su_ipc_export(su_lattice*, unsigned char handle[64]);
su_status su_ipc_open(su_lattice*, const unsigned char handle[64], void** device_ptr);
su_status su_ipc_close(su_lattice*, void* device_ptr);

/* Sum of the slabs' plaquette shares, for slabs driven by one process (synchronises every slab's stream). */
su_status su_slab_plaquette_sum(su_lattice* const* slabs, int n_slabs, double* out);

/* ---- tuning knobs (none changes a result bit; DESIGN.md names the measured defaults) ----
 *   "z_chunk_planes"  z-planes per chunk of the update / plaquette kernels' traversal order (a divisor of Lz;
 *                     0 = the default rule: the largest chunk under 16 MB per time slice). Synchronises.
 *   "fuse"            sub-steps of a pass that su_sweep runs in ONE launch: 1 (default here: one launch per
 *                     (parity, mu), "eight steps"), 2, 4 or 8. Consecutive sub-steps read the same 4V
 *                     links; run together while those are in L2 they move 8/g + 1 instead of 9 links per update.
 *                     Blocks wait on per-(sub-step, cell) completion counters, so every update sees exactly the links
 *                     it sees in the one-launch-per-sub-step sweep: the results are bitwise identical (tested).
 *                     Ignored (plain launches) in slab mode and for kernels without a fused form; su_get_option
 *                     "fuse_effective" tells what su_sweep will do.
 *   "fuse_chunk_planes", "fuse_margin", "fuse_cell_planes"   shape of the fused schedule (csrc/fused_schedule.cu).
 *   "fuse_wait_ns"    wall-clock limit (ns, default 10 s) of one dependency wait inside a fused launch. A correct schedule
 *                     never comes near it; if a wait does exceed it, that block and every block that waits after it stop
 *                     WITHOUT storing anything further, and the next synchronising call (su_synchronize, su_plaquette,
 *                     su_get_counters, ...) returns SU_ECUDA. The links are then a mixture of old and new: the handle
 *                     drops its fused tables and graphs and counts as uninitialised (SU_ESTATE) until su_init_* /
 *                     su_import_links / su_load_config. 0 = give up at the first unsuccessful poll (test hook).
 *   "reunit_on_store" 1: su_sweep leaves reunitarised links. Every link is updated exactly once in the last pass of
 *                     a sweep; there the register kernels of Nc <= 4 project the link they have just updated back to
 *                     SU(Nc) before they store it (PAPER.md:143 arithmetic, saving the separate read-modify-write of
 *                     su_reunitarize); the other kernels run the reunitarisation kernel at the end of the sweep. This
 *                     one DOES change results at rounding level against su_sweep + su_reunitarize (later sub-steps of
 *                     the last pass already see projected neighbours); su_sweep without it never reunitarises. 0: off.
 *   "substep_reunit"  test hook, 1: su_substep runs the kernel instances of that last pass (the link is projected back to
 *                     SU(Nc) right before it is stored), so that they can be compared with the reference sub-step by
 *                     sub-step. Register kernels of Nc <= 4 only (else SU_EUNSUPPORTED). Does not affect su_sweep.
 *   "coop_sweep"      1: su_sweep runs all heatbath passes of a sweep in ONE cooperative launch and all overrelaxation
 *                     passes in another, with grid barriers where the launch boundaries were (register kernels of
 *                     Nc <= 4, lattices whose V/2 threads are resident at once, not slabs; otherwise plain launches;
 *                     su_get_option "coop_sweep_effective": bit 0 heatbath, bit 1 overrelaxation). Bitwise the plain
 *                     sweep (tested). With at most 16 blocks per sub-step (8^4) the grid is one thread-block cluster and the
 *                     barrier the hardware cluster barrier. Measured 0 - 13 % faster than the CUDA-graph replay of the 40
 *                     launches at 8^4, no faster at 16^4 (profiles/r02g).
 *   "block_tile_z", "block_tile_t"   the warps of a thread block of the Nc = 3, 4 register kernels work on the same x-y
 *                     segments of this many consecutive z-planes / time slices (1: a block is consecutive segments of
 *                     one plane), dropped silently where the lattice or the block does not divide evenly. Only in libraries built
 *                     with -DSUG_BLOCK_TILES=1 (su_get_option "block_tiles_supported"); otherwise values != 1: SU_EUNSUPPORTED.
 *   "prefetch_slices" k > 0: every warp of an update kernel asks L2 (cp.async.bulk.prefetch.L2) for the link tiles of
 *                     its sites' positions k time slices ahead of the traversal. A hint; 0 (default) = off.
 *   "blocks_per_sm"   n > 0: update launches request unused dynamic shared memory so that only n blocks fit an SM.
 *                     (measurement knob: it also shrinks L1, which the loads in flight need; profiles/r02g.)
 * Unknown names: SU_EINVAL. */
su_status su_set_option(su_lattice*, const char* name, long long value);
su_status su_get_option(su_lattice*, const char* name, long long* value);

/* The micro-benchmarks behind bench.py's roofline denominators (su_measure_fma_peak, su_measure_l2_peak) and the test
 * hooks (su_debug_kp_math, su_fused_schedule_debug, su_fused_dep_debug) are declared in su_gauge_test.h: they are
 * exported by the same library but are not part of the product interface. */

/* ---- a measurement that allocates nothing ----
 * su_plaquette_static: the mean plaquette (eq 4; the quantity su_plaquette returns) of a link buffer
 * the caller already holds, with no su_lattice handle and without a single cudaMalloc, cudaFree, cudaMallocHost or
 * other allocating call inside the library. It is meant for the callers that cannot allocate: a job whose lattices
 * (or whose host program's memory pool, e.g. PyTorch's caching allocator) already occupy the GPU's memory, so that a
 * library-side cudaMalloc would fail or bypass that pool; monitoring code inside a running generation loop, where
 * cudaMalloc / cudaFree may synchronise the device and stall the sweeps on other streams; and a process that only
 * maps another owner's link buffer (su_ipc_open, a tensor of the host framework) and has no handle to measure with.
 * (su_lattice_create allocates five small device buffers and one pinned host buffer; su_plaquette then uses them.)
 *   - The only scratch the reduction needs, one partial sum per thread block, lives in a fixed 1 MiB __device__ array
 *     inside the library image. Every GPU on which libsugauge is loaded holds that 1 MiB until the process exits.
 *     It bounds the lattice: at most SU_STATIC_MAX_SITES = 64^4 sites; a larger lattice returns SU_EUNSUPPORTED and
 *     launches nothing. Nc = 2, 3, 4 only (the register layouts; RECON12 for Nc = 3), else SU_EUNSUPPORTED.
 *   - device_links: DEVICE pointer (input, read only, 16-byte aligned) to links in the library's device layout, i.e.
 *     the buffer of su_options::buffer / su_slab_links of a whole (non-slab) lattice with the same Nc, extents,
 *     precision and storage; links_bytes >= su_lattice_bytes(...). device_out: DEVICE pointer (output) to one double.
 *     Both stay the caller's. device: CUDA ordinal, -1 = current. stream: cudaStream_t, NULL = legacy default stream.
 *   - Asynchronous: two kernels are enqueued on `stream`; *device_out is valid once they have run. Nothing is copied
 *     to the host and the call does not synchronise.
 *   - The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, which may load the
 *     library's device code there); make that first call during set-up, before any stream capture and outside
 *     time-critical code. Later calls on that device only launch.
 *   - All calls on a device share the one array, and it keeps what the last call left. Each call overwrites every
 *     slot it later reads, so nothing has to start at zero and nothing is cleared. Two calls whose kernels can overlap
 *     on the GPU (different streams, several host threads, several lattices) race on it and give garbage: order them.
 *   - Under the default traversal rule the value is bit for bit su_plaquette's of the same links.
 * Errors: SU_EINVAL (null / misaligned pointers, bad extents, precision, storage, links_bytes too small),
 * SU_EUNSUPPORTED (too many sites, Nc > 4, device ordinal >= 64), SU_ECUDA. su_static_last_error() returns the text of
 * the calling thread's last failure in su_plaquette_static ("" after a success); owned by the library. */
#define SU_STATIC_MAX_SITES 16777216LL
su_status su_plaquette_static(int Nc, int Lx, int Ly, int Lz, int Lt, su_precision p, su_storage s, int device,
                              void* stream, const void* device_links, size_t links_bytes, double* device_out);
const char* su_static_last_error(void);

/* Text of the last error on this handle ("" if none); static text if the handle is NULL.
 * Owned by the library, valid until the next call on the handle. */
const char* su_last_error(const su_lattice*);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif
