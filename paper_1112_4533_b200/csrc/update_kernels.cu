// update_kernels.cu — instantiation and launch of the staple + link-update kernel
// (update_kernel.cuh) for one (parity, mu) sub-step. Compiled once per colour count with
// -DSUG_NC=<Nc>. Block size / minimum blocks per SM per variant: DESIGN.md "Launch configuration".
#include <map>
#include <mutex>
#include <tuple>

#include "su_internal.h"
#include "update_rows_kernel.cuh"

#ifndef SUG_NC
#error "compile with -DSUG_NC=<Nc>"
#endif

namespace sug {

constexpr int NC_ = SUG_NC;
#define SUG_CAT_(a, b) a##b
#define SUG_CAT(a, b) SUG_CAT_(a, b)

// One launch configuration: threads per block, the __launch_bounds__ minimum blocks per SM (= the
// register cap), and the kernel-structure switches of k_update (FUSE3, KUNR).
template <int BLOCK_, int MINB_, int FUSE3_ = 0, bool KUNR_ = false> struct Cfg {
    static constexpr int BLOCK = BLOCK_, MINB = MINB_, FUSE3 = FUSE3_;       // FUSE3: 0 two-step, 1 three links up front, 2 software-pipelined
    static constexpr bool KUNR = KUNR_;
};

// a.dyn_smem (su_set_option "blocks_per_sm"): unused dynamic shared memory requested with the launch, which caps the
// resident blocks per SM below what the registers allow - fused launches re-use links through L2 only while the
// blocks in flight cover less lattice than L2 holds.
template <class K> static void launch_k(K kern, unsigned grid, int block, cudaStream_t st, const UpdateArgs& a) {
    if (a.dyn_smem > 48 * 1024) {                 // above the default limit a kernel has to be opted in once
        static std::mutex mu;
        static std::map<const void*, int> granted;
        std::lock_guard<std::mutex> lock(mu);
        int& have = granted[(const void*)kern];
        if (a.dyn_smem > have && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, a.dyn_smem) == cudaSuccess)
            have = a.dyn_smem;
    }
    kern<<<grid, block, a.dyn_smem, st>>>(a);
}

// cooperative whole-pass launch (k_update_coop): every block of a sub-step resident at once, grid barriers inside
template <class K> static cudaError_t launch_coop(K kern, unsigned grid, int block, cudaStream_t st, const UpdateArgs& a0) {
    UpdateArgs a = a0;
    if (grid <= 16) {
        // the whole sub-step is at most 16 blocks: one thread-block cluster, hardware cluster barriers between the sub-steps.
        // Whether that cluster can run is decided per (kernel, grid, block) by an occupancy query, not by trying the launch:
        // the first launch of a handle in graph mode happens inside a stream capture, which a failing launch would
        // invalidate. The query and the attribute call enqueue nothing, so they are legal during a capture. One mutex
        // covers the decision, so two host threads never probe the same kernel at once.
        static std::mutex mu;
        static std::map<std::tuple<const void*, unsigned, int>, int> state;      // 1: cluster launches work for this configuration, -1: not
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = grid; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int st_k;
        {
            std::lock_guard<std::mutex> lock(mu);
            int& known = state[std::make_tuple((const void*)kern, grid, block)];
            if (known == 0) {
                int n_clusters = 0;
                const bool ok = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess &&
                                cudaOccupancyMaxActiveClusters(&n_clusters, kern, &cfg) == cudaSuccess && n_clusters >= 1;
                cudaGetLastError();
                known = ok ? 1 : -1;
            }
            st_k = known;
        }
        if (st_k == 1) {
            a.coop_cluster = 1;
            const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, a);
            if (e == cudaSuccess) return e;
            cudaGetLastError();                           // against the query's answer: this configuration only falls back to the grid barrier
            std::lock_guard<std::mutex> lock(mu);
            state[std::make_tuple((const void*)kern, grid, block)] = -1;
        }
    }
    a.coop_cluster = 0;
    void* args[] = {(void*)&a};
    return cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(block), args, 0, st);
}
// sites of one parity that a cooperative launch of this kernel can hold (0: cannot be queried)
template <class K> static long long coop_capacity(K kern, int block) {
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, block, 0) != cudaSuccess) { cudaGetLastError(); return 0; }
    return (long long)per_sm * sms * block;
}

// a.fz.work != NULL: the fused launch of a.fz.fg.g consecutive sub-steps (fused_schedule.h), one block per ticket
template <int NC, class T, int STORE, bool UNR, class HB, class OR = HB>
static cudaError_t launch_update_t(int kind, const UpdateArgs& a, cudaStream_t st) {
    const bool fused = a.fz.work != nullptr;
    if (a.coop_passes > 0) {
        if (kind == KIND_HB) return launch_coop(k_update_coop<NC, T, STORE, KIND_HB, UNR, HB::BLOCK, HB::MINB, HB::FUSE3, HB::KUNR>, (a.g.Vh_int + HB::BLOCK - 1) / HB::BLOCK, HB::BLOCK, st, a);
        return launch_coop(k_update_coop<NC, T, STORE, KIND_OR, UNR, OR::BLOCK, OR::MINB, OR::FUSE3, OR::KUNR>, (a.g.Vh_int + OR::BLOCK - 1) / OR::BLOCK, OR::BLOCK, st, a);
    }
    if (kind == KIND_HB) {
        const unsigned grid = (a.g.Vh_int + HB::BLOCK - 1) / HB::BLOCK;
        if (fused) launch_k(k_update<NC, T, STORE, KIND_HB, UNR, HB::BLOCK, HB::MINB, HB::FUSE3, HB::KUNR, true>, a.fz.n_tickets, HB::BLOCK, st, a);
        else       launch_k(k_update<NC, T, STORE, KIND_HB, UNR, HB::BLOCK, HB::MINB, HB::FUSE3, HB::KUNR>, grid, HB::BLOCK, st, a);
    } else {
        const unsigned grid = (a.g.Vh_int + OR::BLOCK - 1) / OR::BLOCK;
        if (fused) launch_k(k_update<NC, T, STORE, KIND_OR, UNR, OR::BLOCK, OR::MINB, OR::FUSE3, OR::KUNR, true>, a.fz.n_tickets, OR::BLOCK, st, a);
        else       launch_k(k_update<NC, T, STORE, KIND_OR, UNR, OR::BLOCK, OR::MINB, OR::FUSE3, OR::KUNR>, grid, OR::BLOCK, st, a);
    }
    return cudaGetLastError();
}
template <class HB, class OR = HB> static int spb_t(int kind) { return kind == KIND_HB ? HB::BLOCK : OR::BLOCK; }
template <int NC, class T, int STORE, bool UNR, class HB, class OR = HB> static long long coop_sites_t(int kind) {
    if (kind == KIND_HB) return coop_capacity(k_update_coop<NC, T, STORE, KIND_HB, UNR, HB::BLOCK, HB::MINB, HB::FUSE3, HB::KUNR>, HB::BLOCK);
    return coop_capacity(k_update_coop<NC, T, STORE, KIND_OR, UNR, OR::BLOCK, OR::MINB, OR::FUSE3, OR::KUNR>, OR::BLOCK);
}

// Tuning overrides (-DSUG_CFG_...="Cfg<...>"), used only while sweeping on the GPU; the defaults below are
// the measured choices (profiles/).
#ifndef SUG_SU3_F64_BLOCK          // integer knobs: nvcc splits -D values at commas, so Cfg<...> cannot come from the command line
#define SUG_SU3_F64_BLOCK 128
#endif
#ifndef SUG_SU3_F64_MINB
#define SUG_SU3_F64_MINB 3
#endif
#ifndef SUG_SU3_F64_SMODE
#define SUG_SU3_F64_SMODE 1
#endif
// heatbath, fp64: 2 blocks of 192 threads (the same 12 warps per SM as 3 x 128) measured 2-3 % faster (profiles/r02g)
#ifndef SUG_SU3_F64_HB_MINB
#define SUG_SU3_F64_HB_MINB 2
#endif
#ifndef SUG_SU3_F64_HB_BLOCK
#define SUG_SU3_F64_HB_BLOCK 192
#endif
#ifndef SUG_CFG_SU3_F64_HB
#define SUG_CFG_SU3_F64_HB Cfg<SUG_SU3_F64_HB_BLOCK, SUG_SU3_F64_HB_MINB, SUG_SU3_F64_SMODE, true>
#endif
#ifndef SUG_CFG_SU3_F64_OR
#define SUG_CFG_SU3_F64_OR Cfg<SUG_SU3_F64_BLOCK, SUG_SU3_F64_MINB, SUG_SU3_F64_SMODE, true>
#endif
#ifndef SUG_SU3_F32_SMODE
#define SUG_SU3_F32_SMODE 1
#endif
#ifndef SUG_SU3_F32_OR_MINB
#define SUG_SU3_F32_OR_MINB 5
#endif
#ifndef SUG_SU3_F32_HB_MINB
#define SUG_SU3_F32_HB_MINB 5
#endif
#ifndef SUG_SU3_F32_BLOCK
#define SUG_SU3_F32_BLOCK 128
#endif
#ifndef SUG_CFG_SU3_F32_HB
#define SUG_CFG_SU3_F32_HB Cfg<SUG_SU3_F32_BLOCK, SUG_SU3_F32_HB_MINB, SUG_SU3_F32_SMODE, true>
#endif
#ifndef SUG_CFG_SU3_F32_OR
#define SUG_CFG_SU3_F32_OR Cfg<SUG_SU3_F32_BLOCK, SUG_SU3_F32_OR_MINB, SUG_SU3_F32_SMODE, true>
#endif
// two-row storage: staple form (1: every link completed on load, 3: lazy third rows, Su3Rows) and register caps
#ifndef SUG_SU3R_SMODE
#define SUG_SU3R_SMODE 3
#endif
#ifndef SUG_SU3R_F64_MINB
#define SUG_SU3R_F64_MINB 3
#endif
#ifndef SUG_SU3R_F32_MINB
#define SUG_SU3R_F32_MINB 3
#endif
#ifndef SUG_SU3R_F32_HB_MINB
#define SUG_SU3R_F32_HB_MINB SUG_SU3R_F32_MINB
#endif
#ifndef SUG_CFG_SU3R_F64_HB
#define SUG_CFG_SU3R_F64_HB Cfg<128, SUG_SU3R_F64_MINB, SUG_SU3R_SMODE, true>
#endif
#ifndef SUG_CFG_SU3R_F64_OR
#define SUG_CFG_SU3R_F64_OR Cfg<128, SUG_SU3R_F64_MINB, SUG_SU3R_SMODE, true>
#endif
#ifndef SUG_CFG_SU3R_F32_HB
#define SUG_CFG_SU3R_F32_HB Cfg<128, SUG_SU3R_F32_HB_MINB, SUG_SU3R_SMODE, true>
#endif
#ifndef SUG_CFG_SU3R_F32_OR
#define SUG_CFG_SU3R_F32_OR Cfg<128, SUG_SU3R_F32_MINB, SUG_SU3R_SMODE, true>
#endif
#ifndef SUG_SU4_F64_HB_BLOCK
#define SUG_SU4_F64_HB_BLOCK 128
#endif
#ifndef SUG_SU4_F64_HB_MINB
#define SUG_SU4_F64_HB_MINB 1
#endif
#ifndef SUG_SU4_F64_HB_SMODE
#define SUG_SU4_F64_HB_SMODE 0
#endif
#ifndef SUG_SU4_F64_HB_KUNR
#define SUG_SU4_F64_HB_KUNR false
#endif
#ifndef SUG_CFG_SU4_F64_HB
#define SUG_CFG_SU4_F64_HB Cfg<SUG_SU4_F64_HB_BLOCK, SUG_SU4_F64_HB_MINB, SUG_SU4_F64_HB_SMODE, SUG_SU4_F64_HB_KUNR>
#endif
#ifndef SUG_CFG_SU4_F64_OR
#define SUG_CFG_SU4_F64_OR Cfg<128, 2, true, true>
#endif
#ifndef SUG_CFG_SU4_F32_HB
#define SUG_CFG_SU4_F32_HB Cfg<128, 3, true, true>
#endif
#ifndef SUG_CFG_SU4_F32_OR
#define SUG_CFG_SU4_F32_OR Cfg<128, 3, true, true>
#endif
// Generic SU(Nc): the row-per-lane kernel (update_rows_kernel.cuh) for full Nc x Nc storage; the rolled-loop
// thread-per-link form (local-memory arrays, small blocks) only for the SU(2) quaternion / SU(3) two-row layouts.
typedef Cfg<64, 1> GenericCfg;

cudaError_t SUG_CAT(update_nc, SUG_NC)(const Variant& v, int kind, const UpdateArgs& a, cudaStream_t st, uint64_t* n_launch) {
    constexpr int NC = SUG_NC;
    ++*n_launch;
    const bool f64 = v.prec == SU_FP64;
#if SUG_NC == 2
    if (!v.generic) {
        constexpr int BLOCK = 128;
        const unsigned grid = (a.g.Vh_int + BLOCK - 1) / BLOCK;
        if (a.coop_passes > 0) {
            if (f64) return kind == KIND_HB ? launch_coop(k_update_su2_coop<double, KIND_HB, BLOCK, 4>, grid, BLOCK, st, a) : launch_coop(k_update_su2_coop<double, KIND_OR, BLOCK, 4>, grid, BLOCK, st, a);
            return kind == KIND_HB ? launch_coop(k_update_su2_coop<float, KIND_HB, BLOCK, 4>, grid, BLOCK, st, a) : launch_coop(k_update_su2_coop<float, KIND_OR, BLOCK, 4>, grid, BLOCK, st, a);
        }
        if (f64) { if (kind == KIND_HB) k_update_su2<double, KIND_HB, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<double, KIND_OR, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); }
        else     { if (kind == KIND_HB) k_update_su2<float,  KIND_HB, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<float,  KIND_OR, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); }
        return cudaGetLastError();
    }
    return f64 ? launch_update_t<NC, double, STORE_QUAT, false, GenericCfg>(kind, a, st)
               : launch_update_t<NC, float,  STORE_QUAT, false, GenericCfg>(kind, a, st);
#elif SUG_NC == 3
    if (!v.generic) {
        if (v.store == STORE_RECON12)
            return f64 ? launch_update_t<NC, double, STORE_RECON12, true, SUG_CFG_SU3R_F64_HB, SUG_CFG_SU3R_F64_OR>(kind, a, st)
                       : launch_update_t<NC, float,  STORE_RECON12, true, SUG_CFG_SU3R_F32_HB, SUG_CFG_SU3R_F32_OR>(kind, a, st);
        return f64 ? launch_update_t<NC, double, STORE_FULL, true, SUG_CFG_SU3_F64_HB, SUG_CFG_SU3_F64_OR>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_FULL, true, SUG_CFG_SU3_F32_HB, SUG_CFG_SU3_F32_OR>(kind, a, st);
    }
    if (v.store == STORE_RECON12)
        return f64 ? launch_update_t<NC, double, STORE_RECON12, false, GenericCfg>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_RECON12, false, GenericCfg>(kind, a, st);
    return f64 ? launch_update_rows<NC, double>(kind, a, st) : launch_update_rows<NC, float>(kind, a, st);
#elif SUG_NC == 4
    if (!v.generic)
        return f64 ? launch_update_t<NC, double, STORE_FULL, true, SUG_CFG_SU4_F64_HB, SUG_CFG_SU4_F64_OR>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_FULL, true, SUG_CFG_SU4_F32_HB, SUG_CFG_SU4_F32_OR>(kind, a, st);
    return f64 ? launch_update_rows<NC, double>(kind, a, st) : launch_update_rows<NC, float>(kind, a, st);
#else
    return f64 ? launch_update_rows<NC, double>(kind, a, st) : launch_update_rows<NC, float>(kind, a, st);
#endif
}

// Sites per block of the kernel update_nc would launch for this variant and kind = the tile size of the fused
// schedule; 0: this kernel has no fused form (the caller then runs the sub-steps one launch each).
int SUG_CAT(update_spb_nc, SUG_NC)(const Variant& v, int kind) {
    const bool f64 = v.prec == SU_FP64;
#if SUG_NC == 2
    if (!v.generic) return 0;
    return spb_t<GenericCfg>(kind);
#elif SUG_NC == 3
    if (!v.generic) {
        if (v.store == STORE_RECON12) return f64 ? spb_t<SUG_CFG_SU3R_F64_HB, SUG_CFG_SU3R_F64_OR>(kind) : spb_t<SUG_CFG_SU3R_F32_HB, SUG_CFG_SU3R_F32_OR>(kind);
        return f64 ? spb_t<SUG_CFG_SU3_F64_HB, SUG_CFG_SU3_F64_OR>(kind) : spb_t<SUG_CFG_SU3_F32_HB, SUG_CFG_SU3_F32_OR>(kind);
    }
    if (v.store == STORE_RECON12) return spb_t<GenericCfg>(kind);
    return 0;
#elif SUG_NC == 4
    if (!v.generic) return f64 ? spb_t<SUG_CFG_SU4_F64_HB, SUG_CFG_SU4_F64_OR>(kind) : spb_t<SUG_CFG_SU4_F32_HB, SUG_CFG_SU4_F32_OR>(kind);
    return 0;
#else
    (void)f64;
    return 0;
#endif
}

// Sites of one parity that fit ONE cooperative whole-pass launch of the kernel update_nc would use for this variant and
// kind (all blocks resident at once); 0: this kernel has no cooperative form.
long long SUG_CAT(update_coop_sites_nc, SUG_NC)(const Variant& v, int kind) {
    const bool f64 = v.prec == SU_FP64;
#if SUG_NC == 2
    if (v.generic) return 0;
    if (f64) return kind == KIND_HB ? coop_capacity(k_update_su2_coop<double, KIND_HB, 128, 4>, 128) : coop_capacity(k_update_su2_coop<double, KIND_OR, 128, 4>, 128);
    return kind == KIND_HB ? coop_capacity(k_update_su2_coop<float, KIND_HB, 128, 4>, 128) : coop_capacity(k_update_su2_coop<float, KIND_OR, 128, 4>, 128);
#elif SUG_NC == 3
    if (v.generic) return 0;
    if (v.store == STORE_RECON12)
        return f64 ? coop_sites_t<NC_, double, STORE_RECON12, true, SUG_CFG_SU3R_F64_HB, SUG_CFG_SU3R_F64_OR>(kind)
                   : coop_sites_t<NC_, float,  STORE_RECON12, true, SUG_CFG_SU3R_F32_HB, SUG_CFG_SU3R_F32_OR>(kind);
    return f64 ? coop_sites_t<NC_, double, STORE_FULL, true, SUG_CFG_SU3_F64_HB, SUG_CFG_SU3_F64_OR>(kind)
               : coop_sites_t<NC_, float,  STORE_FULL, true, SUG_CFG_SU3_F32_HB, SUG_CFG_SU3_F32_OR>(kind);
#elif SUG_NC == 4
    if (v.generic) return 0;
    return f64 ? coop_sites_t<NC_, double, STORE_FULL, true, SUG_CFG_SU4_F64_HB, SUG_CFG_SU4_F64_OR>(kind)
               : coop_sites_t<NC_, float,  STORE_FULL, true, SUG_CFG_SU4_F32_HB, SUG_CFG_SU4_F32_OR>(kind);
#else
    (void)f64; (void)kind; (void)v;
    return 0;
#endif
}

}  // namespace sug
