// update_kernels.cu — instantiation and launch of the staple + link-update kernel
// (update_kernel.cuh) for one (parity, mu) sub-step. Compiled once per colour count with
// -DSUG_NC=<Nc>. Block size / minimum blocks per SM per variant: DESIGN.md "Launch configuration".
#include "su_internal.h"

#ifndef SUG_NC
#error "compile with -DSUG_NC=<Nc>"
#endif

namespace sug {

#define SUG_CAT_(a, b) a##b
#define SUG_CAT(a, b) SUG_CAT_(a, b)

// (HB_BLOCK, HB_MINB) and (OR_BLOCK, OR_MINB): threads per block and the __launch_bounds__ minimum
// blocks per SM (= the register cap) of the heatbath and of the overrelaxation instantiation.
template <int NC, class T, int STORE, bool UNR, int HB_BLOCK, int HB_MINB, int OR_BLOCK = HB_BLOCK, int OR_MINB = HB_MINB>
static cudaError_t launch_update_t(int kind, const UpdateArgs& a, cudaStream_t st) {
    if (kind == KIND_HB) {
        const unsigned grid = (a.g.Vh + HB_BLOCK - 1) / HB_BLOCK;
        k_update<NC, T, STORE, KIND_HB, UNR, HB_BLOCK, HB_MINB><<<grid, HB_BLOCK, 0, st>>>(a);
    } else {
        const unsigned grid = (a.g.Vh + OR_BLOCK - 1) / OR_BLOCK;
        k_update<NC, T, STORE, KIND_OR, UNR, OR_BLOCK, OR_MINB><<<grid, OR_BLOCK, 0, st>>>(a);
    }
    return cudaGetLastError();
}

cudaError_t SUG_CAT(update_nc, SUG_NC)(const Variant& v, int kind, const UpdateArgs& a, cudaStream_t st, uint64_t* n_launch) {
    constexpr int NC = SUG_NC;
    ++*n_launch;
    const bool f64 = v.prec == SU_FP64;
#if SUG_NC == 2
    if (!v.generic) {
        constexpr int BLOCK = 128;
        const unsigned grid = (a.g.Vh + BLOCK - 1) / BLOCK;
        if (f64) { if (kind == KIND_HB) k_update_su2<double, KIND_HB, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<double, KIND_OR, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); }
        else     { if (kind == KIND_HB) k_update_su2<float,  KIND_HB, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<float,  KIND_OR, BLOCK, 4><<<grid, BLOCK, 0, st>>>(a); }
        return cudaGetLastError();
    }
    return f64 ? launch_update_t<NC, double, STORE_QUAT, false, 64, 1>(kind, a, st)
               : launch_update_t<NC, float,  STORE_QUAT, false, 64, 1>(kind, a, st);
#elif SUG_NC == 3
    if (!v.generic) {
        if (v.store == STORE_RECON12)
            return f64 ? launch_update_t<NC, double, STORE_RECON12, true, 128, 1>(kind, a, st)
                       : launch_update_t<NC, float,  STORE_RECON12, true, 128, 1>(kind, a, st);
        // measured on B200 at 48^4 (profiles/r01b_*): fp64 168 registers / 3 blocks beats both the
        // spill-free 240 / 2 and the 128 / 4 build; fp32 fits 80 registers / 6 blocks without spills
        return f64 ? launch_update_t<NC, double, STORE_FULL, true, 256, 2, 128, 3>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_FULL, true, 128, 4, 128, 6>(kind, a, st);
    }
    if (v.store == STORE_RECON12)
        return f64 ? launch_update_t<NC, double, STORE_RECON12, false, 64, 1>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_RECON12, false, 64, 1>(kind, a, st);
    return f64 ? launch_update_t<NC, double, STORE_FULL, false, 64, 1>(kind, a, st)
               : launch_update_t<NC, float,  STORE_FULL, false, 64, 1>(kind, a, st);
#elif SUG_NC == 4
    if (!v.generic)
        return f64 ? launch_update_t<NC, double, STORE_FULL, true, 128, 1>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_FULL, true, 128, 1>(kind, a, st);
    return f64 ? launch_update_t<NC, double, STORE_FULL, false, 64, 1>(kind, a, st)
               : launch_update_t<NC, float,  STORE_FULL, false, 64, 1>(kind, a, st);
#else
    return f64 ? launch_update_t<NC, double, STORE_FULL, false, 64, 1>(kind, a, st)
               : launch_update_t<NC, float,  STORE_FULL, false, 64, 1>(kind, a, st);
#endif
}

}  // namespace sug
