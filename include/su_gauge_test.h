/*
 * su_gauge_test.h — entry points of libsugauge that are NOT part of the product interface (include/su_gauge.h):
 * the two micro-benchmarks that give bench.py its measured roofline denominators, and three hooks that exist so that
 * tests can look inside (the fused schedule on the CPU, the elementary functions of the Kennedy-Pendleton draw).
 * Same conventions as su_gauge.h (su_status, host pointers unless said otherwise). A program that generates
 * configurations needs none of them.
 */
#ifndef SU_GAUGE_TEST_H
#define SU_GAUGE_TEST_H
#include "su_gauge.h"
#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)
#endif

/* Host-only views of the fused schedule, for the CPU test that proves it (tests/test_fused_schedule.py): the
 * ticket table work[n_tickets][n_fused] (tile id = cell * nT + tile, 0xffffffff = none; cell = t * nzu + z-unit)
 * with geom = {planes per cell, cells per time slice, tiles per cell, sites per cell, sites per plane}, and the
 * k-th dependency (completion-counter index stage * cells + cell, or -1) of a work item, exactly as the kernel
 * enumerates it. No device is touched. planes_per_cell / chunk_planes 0 = default. */
su_status su_fused_schedule_debug(int Lx, int Ly, int Lz, int Lt, int sites_per_block, int n_fused, int first_substep,
                                  int planes_per_cell, int chunk_planes, int margin, uint32_t* work, size_t work_capacity,
                                  int* n_tickets, int* geom);
int su_fused_dep_debug(int Lx, int Ly, int Lz, int Lt, int sites_per_block, int n_fused, int first_substep,
                       int planes_per_cell, int stage, int cell, int tile, int k);

/* Measured FMA rate of the device's FP32 / FP64 pipes in TFLOP/s (FMA = 2 flops): a short register-only
 * micro-benchmark (16 independent chains per thread, 8 blocks of 256 threads per SM, best of 5 launches of a few
 * ms each), the denominator of the "alu" roofline of the variants that are not HBM-bound.
 * device -1 = current. ms (may be NULL): duration of the best launch. Synchronises the device. */
su_status su_measure_fma_peak(int device, su_precision p, double* tflops, double* ms);

/* Measured L2 -> SM read throughput of the device in GB/s: every thread block streams one 24 MB L2-resident buffer
 * with 128-bit loads that bypass L1 (through_l1 = 0: ld.global.cg) or allocate in it (through_l1 = 1: ld.global.nc, each
 * block's 24 MB still far beyond L1) (4 blocks of 256 threads per SM, 8 loads per thread in flight, best of 5
 * launches). The staple + update kernel issues 19 link loads per update of which L1 serves < 10 %, so 2.1 x its HBM
 * bytes cross this path; bench.py reports the fraction of this rate it uses (0.5 - 0.6 for 18-real SU(3): not the
 * limiter, profiles/r02g). device -1 = current.
 * ms (may be NULL): duration of the best launch; bytes_per_clock (may be NULL): the same throughput per SM clock
 * cycle (clock64 span of one block), the figure that carries over to a run at another clock. Synchronises the device. */
su_status su_measure_l2_peak(int device, int through_l1, double* gbs, double* ms, double* bytes_per_clock);

/* Test hook: the elementary functions of the Kennedy-Pendleton draw exactly as the fp64 kernels evaluate them (branch-free
 * ln / sincos / sqrt / rsqrt of csrc/su_device.cuh). For each of the n host words w, u = (w + 1) / 2^32:
 * out[5 i + 0..4] = ln u, sin 2 pi u, cos 2 pi u, sqrt u, 1 / sqrt(100 u + 0.001). Host pointers; synchronises. */
su_status su_debug_kp_math(int device, const uint32_t* words, size_t n, double* out);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif
