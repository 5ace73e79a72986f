// su_internal.h — host-side declarations shared by the translation units of libsugauge.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/su_gauge.h"
#include "../../include/su_gauge_test.h"
#include "su_device.cuh"
#include "update_kernel.cuh"

namespace sug {

struct Variant {
    int Nc;
    int prec;      // su_precision
    int store;     // STORE_FULL / STORE_RECON12 / STORE_QUAT
    bool generic;  // rolled-loop generic kernel instead of the register-resident one
};

struct AuxArgs {
    void* links;
    Geom g;
    double* partials;        // device scratch for reductions
    double* result;          // device, up to 2 doubles
    double* staging;         // device, canonical layout chunk
    unsigned site0, nsites;  // lexicographic site range for import/export
    uint32_t k0, k1;
};

// Each returns cudaGetLastError() after the launch; n_launch is incremented per kernel launched.
#define SUG_DECLARE_NC(N)                                                                                   \
    cudaError_t update_nc##N(const Variant&, int kind, const UpdateArgs&, cudaStream_t, uint64_t* n_launch); \
    int update_spb_nc##N(const Variant&, int kind);                                                          \
    long long update_coop_sites_nc##N(const Variant&, int kind);                                             \
    cudaError_t plaquette_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);           \
    cudaError_t polyakov_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);            \
    cudaError_t reunit_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);              \
    cudaError_t init_cold_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);           \
    cudaError_t init_hot_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);            \
    cudaError_t export_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);              \
    cudaError_t import_nc##N(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);

SUG_DECLARE_NC(2)
SUG_DECLARE_NC(3)
SUG_DECLARE_NC(4)
SUG_DECLARE_NC(5)
SUG_DECLARE_NC(6)
SUG_DECLARE_NC(7)
SUG_DECLARE_NC(8)

// fused_schedule.cu
FusedGeom fused_make_geom(int Lx, int Ly, int Lz, int Lt, int spb, int g, int sub0, int U_force);
bool fused_build_schedule(const FusedGeom& fg, int chunk_units, int margin, std::vector<uint32_t>& work, int& n_tickets);

// big_kernels.cu: the runtime-Nc warp-per-link path (9 <= Nc <= SU_MAX_NC)
cudaError_t update_nc_big(const Variant&, int kind, const UpdateArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t plaquette_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t polyakov_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t reunit_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t init_cold_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t init_hot_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t export_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
cudaError_t import_nc_big(const Variant&, const AuxArgs&, cudaStream_t, uint64_t* n_launch);
constexpr int SUG_MAX_TEMPLATE_NC = 8;    // kernels compiled per Nc up to here; the warp-per-link path above

constexpr int REDUCE_BLOCK = 256;
inline unsigned reduce_blocks(unsigned n) { return (n + REDUCE_BLOCK - 1) / REDUCE_BLOCK; }
constexpr int ROWS_MIN_LINKS_PER_BLOCK = 4;   // row-per-lane kernels: 1 warp x floor(32 / SU_MAX_NC) sites per block at least
constexpr int PLAQ_BLOCK = 128;          // plaquette kernel: blocks alternate parity over the same region
// register caps of the plaquette kernel, measured at SU(3) 48^4: fp64 254 registers (1.22 vs 1.44 ms at 168), fp32 128 (0.60 vs 0.68 ms)
#ifndef PLAQ_MINB_F64
#define PLAQ_MINB_F64 2
#endif
#ifndef PLAQ_MINB_F32
#define PLAQ_MINB_F32 4
#endif
inline unsigned plaquette_blocks(unsigned Vh) { return 2u * ((Vh + PLAQ_BLOCK - 1) / PLAQ_BLOCK); }

}  // namespace sug
