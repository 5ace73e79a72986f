// fused_schedule.h — several consecutive sub-steps of a pass in ONE launch (SURVEY.md 8(f) NEXT-4 "fusions around
// the path"; "these kernels have to be called in eight steps").
//
// Why. A sub-step (parity, mu) reads every link of the lattice once (3V nu-links + V mu-links) and writes V/2:
// 9 link transfers per update. g consecutive sub-steps of the sweep schedule read
// the SAME 4V links, so run together, while the links are still in L2, they move 4V + g V/2 links for g V/2
// updates: 8/g + 1 transfers per update (g = 2: 5, g = 4: 3, g = 8: 2). The result is bitwise the result of the
// g launches in sequence: every update sees exactly the links it would have seen.
//
// How. The lattice (one parity) is cut into CELLS = U consecutive z-planes of one time slice, and every cell into
// TILES of one thread block's worth of sites. A block takes a ticket k (atomic counter, so ticket order = start
// order) and executes up to g work items one after the other: a tile of stage 0, then a tile of stage 1 that lies
// a little "behind" it, and so on (a software pipeline across sub-steps, skewed in space; table built on the host,
// fused_schedule.cu). Stage b at site x conflicts with an earlier stage a at site y when one reads a link the
// other writes (both directions: read-after-write and write-after-read); the conflicting y are x plus a few unit
// offsets (fused_dep_offsets below). Before a work item starts, warp 0 of the block waits until the per-(stage,
// cell) completion counters of every cell it conflicts with are full; after its stores, the block bumps its own
// cell's counter (release / acquire at gpu scope). The table gives a work item only cells that were handed out to
// LOWER tickets, so a block only ever waits for blocks that have already started: no deadlock whatever the
// hardware's block order, and because the block itself spends its earlier phases working, the wait is normally
// already over when it gets there.
#pragma once
#include <stdint.h>

#ifndef __CUDACC__
#define __host__
#define __device__
#endif

namespace sug {

constexpr uint32_t FUSED_NONE = 0xffffffffu;
constexpr int FUSED_MAX_G = 8;            // a pass has 8 sub-steps
constexpr int FUSED_DEPS_PER_STAGE = 10;  // <= 5 (dz, dt) offsets per earlier stage x 2 ends of the tile's z-range

struct FusedGeom {
    int Lz, Lt;        // extents in z and t (stored = global: fused launches are not used in slab mode)
    int U;             // z-planes per cell (divides Lz)
    int nzu;           // cells per time slice = Lz / U
    int plane_sites;   // sites of one parity in one z-plane of one time slice = (Lx / 2) Ly
    int cell_sites;    // plane_sites * U
    int spb;           // sites per block (tile size)
    int nT;            // tiles per cell = ceil(cell_sites / spb)
    int g;             // sub-steps in the launch
    int sub0;          // first sub-step of the group: sub-step index = 4 parity + mu (reading R6: parity outer)
};

struct FusedCtrl {     // device: one per table
    unsigned ticket;   // next ticket of the running launch
    unsigned exited;   // blocks of the running launch that have finished
    unsigned epoch;    // finished launches on this table; the counters are cumulative: full = (epoch + 1) nT
    unsigned error;    // a dependency wait gave up (never in a correct schedule; the host then reports SU_ECUDA)
};

__host__ __device__ inline int fused_parity(const FusedGeom& fg, int s) { return ((fg.sub0 + s) >> 2) & 1; }
__host__ __device__ inline int fused_mu(const FusedGeom& fg, int s) { return (fg.sub0 + s) & 3; }

// (dz, dt) offsets, relative to a site x of stage b, of the sites y whose stage-a update (a earlier than b in the
// schedule) conflicts with the stage-b update of x. Link footprint of the update of U_mu(x) (eq 9):
//   reads (x,nu) (x+nu,mu) (x+mu,nu) (x-nu,nu) (x-nu,mu) (x-nu+mu,nu) for nu != mu, and (x,mu); writes (x,mu).
// "a writes what b reads" <=> (y,mu_a) in reads(b,x): mu_a != mu_b: y - x in {0, +mu_b, -mu_a, -mu_a+mu_b};
// mu_a == mu_b: y - x in {+-nu}. "b writes what a reads" gives the same sets. The parities of x and y select the
// even (0, -mu_a+mu_b) or odd (+mu_b, -mu_a, +-nu) offsets. Offsets in x and y stay inside a cell. Returns the count.
__host__ __device__ inline int fused_dep_offsets(int pa, int mua, int pb, int mub, int dz[5], int dt[5]) {
    int n = 0;
    auto add = [&](int sign_b, int sign_a) {        // offset = sign_b e_{mub} + sign_a e_{mua}
        int z = 0, t = 0;
        if (mub == 2) z += sign_b; if (mub == 3) t += sign_b;
        if (mua == 2) z += sign_a; if (mua == 3) t += sign_a;
        dz[n] = z; dt[n] = t; ++n;
    };
    if (mua != mub) {
        if (pa == pb) { add(0, 0); add(+1, -1); }
        else          { add(+1, 0); add(0, -1); }
    } else {                                         // same direction: the other parity, x +- nu
        dz[n] = 0; dt[n] = 0; ++n;                   // nu = x or y (at least one of them is != mu)
        if (mua != 2) { dz[n] = 1; dt[n] = 0; ++n; dz[n] = -1; dt[n] = 0; ++n; }
        if (mua != 3) { dz[n] = 0; dt[n] = 1; ++n; dz[n] = 0; dt[n] = -1; ++n; }
    }
    return n;
}

// k-th dependency of the work item (stage s, cell, tile), k in [0, s * FUSED_DEPS_PER_STAGE): the index of the
// completion counter to wait for (stage a, cell'), or -1 when that slot is empty.
__host__ __device__ inline int fused_dep(const FusedGeom& fg, int s, int cell, int tile, int k) {
    const int a = k / FUSED_DEPS_PER_STAGE, o = (k % FUSED_DEPS_PER_STAGE) >> 1, end = k & 1;
    int dz[5], dt[5];
    const int n = fused_dep_offsets(fused_parity(fg, a), fused_mu(fg, a), fused_parity(fg, s), fused_mu(fg, s), dz, dt);
    if (a >= s || o >= n) return -1;
    const int t = cell / fg.nzu, zu = cell - t * fg.nzu;
    const int r0 = tile * fg.spb;
    int r1 = r0 + fg.spb; if (r1 > fg.cell_sites) r1 = fg.cell_sites;
    const int zlo = zu * fg.U + r0 / fg.plane_sites, zhi = zu * fg.U + (r1 - 1) / fg.plane_sites;
    if (end == 1 && zhi == zlo) return -1;           // both ends in the same plane: one lookup
    int z = (end ? zhi : zlo) + dz[o];
    z = z < 0 ? z + fg.Lz : (z >= fg.Lz ? z - fg.Lz : z);
    int tt = t + dt[o];
    tt = tt < 0 ? tt + fg.Lt : (tt >= fg.Lt ? tt - fg.Lt : tt);
    return a * (fg.Lt * fg.nzu) + tt * fg.nzu + z / fg.U;
}

}  // namespace sug
