// update_kernel.cuh — the staple + link-update kernel (heatbath / overrelaxation) for one
// (parity, mu) sub-step of the sweep ("eight steps" per pass).
//
// One thread owns one link U_mu(x), x of the given parity. It gathers the 18 staple
// links (eq 9) from the tiled SoA planes with coalesced 64/128-bit loads, forms
// W = U S^dagger (step 2), runs the SU(2) subgroup loop (steps 3-5) and stores the link.
//   UNR = true : matrices fully unrolled into registers (specialised SU(3)/SU(4))
//   UNR = false: rolled loops over local arrays (generic SU(Nc))
//
// Thread -> site mapping: the thread index walks the lattice as
// (z-chunk, t, z within chunk, y, x/2), so that the data first touched at t+1 is touched again
// (at t and t-1) before 2 * Zc/Lz time slices of all planes have streamed through L2.
#pragma once
#include <cooperative_groups.h>

#include "su_device.cuh"
#include "fused_schedule.h"

namespace sug {

// three-links-up-front staple: request the own link before the last accumulation (see update_link)
#ifndef SUG_EARLY_SELF
#define SUG_EARLY_SELF 0
#endif
#ifndef SUG_TMINUS_STREAM
#define SUG_TMINUS_STREAM 1
#endif
// heatbath: what the register kernels evaluate ahead of the staple and park in shared memory (one private column
// per thread): 0 nothing, 1 the directions of the draws, 2 also attempt 0 of every draw (kp_attempt0).
// Measured at SU(3) 48^4 (profiles/r02b_heatbath.md): fp32 1 is best (-2.7 % against 0); fp64: 0 1.015 ms,
// 1 1.006 ms, 2 1.118 ms per sub-step - evaluating the fp64 log / cospi chains early lengthens the time to the
// first loads more than it shortens the tail, so fp64 keeps everything in the subgroup loop.
#ifndef SUG_KP_PRE_F32
#define SUG_KP_PRE_F32 1
#endif
#ifndef SUG_KP_PRE_F64
#define SUG_KP_PRE_F64 0
#endif

// fused launches: how neighbour links are loaded (3 = LD_COHERENT, ld.relaxed.gpu, always served by L2; 0 = LD_PLAIN,
// ordinary loads, correct because every work item starts behind an acquire at gpu scope, which also invalidates
// L1) and whether the updated link is stored / the own link loaded with the streaming (evict-first) hint of the
// plain kernel (there the link is not touched again in the launch; in a fused launch the next stages re-read it)
#ifndef SUG_FUSED_LD
#define SUG_FUSED_LD 0
#endif
#ifndef SUG_FUSED_STREAM
#define SUG_FUSED_STREAM 0
#endif

// how the plain (one sub-step per launch) register kernels load neighbour links: LD_RO (ld.global.nc), LD_CG, LD_NA, LD_STREAM
#ifndef SUG_NEIGHBOUR_LD
#define SUG_NEIGHBOUR_LD LD_RO
#endif

struct UpdateArgs {
    void* links;
    Geom g;
    int parity, mu;
    double beta;
    uint32_t k0, k1, sweep, pass;
    const uint32_t* sweep_ptr;         // device; when non-NULL the sweep counter is read from here (graph replay)
    int reunit;                        // != 0: project the updated link back to SU(Nc) right before the store (Nc <= 4 register kernels)
    int pf_slices;                     // > 0: every warp asks L2 for the link tiles of its sites' positions this many time slices ahead
    int dyn_smem;                      // host side only: unused dynamic shared memory per block (caps the resident blocks per SM)
    int coop_passes;                   // > 0: cooperative launch that runs this many whole passes (8 sub-steps each) with grid barriers
    int coop_cluster;                  // set by the launcher: the whole grid is ONE thread-block cluster (<= 16 blocks): cluster barriers
    uint8_t* attempts;                 // device, [n_sub][Vh] or NULL
    unsigned long long* counters;      // device, {kp_attempts_total, kp_exhausted}
    // slab mode: link buffers of the slabs below / above in t (peer memory over NVLink, or this device). The
    // kernel that updates a link of the first / last owned slice also stores it into that neighbour's halo.
    void* peer_lo;
    void* peer_hi;
    // fused launch of several consecutive sub-steps (fused_schedule.h); work == NULL: the plain one-sub-step launch
    struct Fused {
        const uint32_t* work;          // device, [n_tickets][g]: tile id (cell * nT + tile) of every stage, or FUSED_NONE
        unsigned* done;                // device, [g][cells]: cumulative count of finished tiles
        FusedCtrl* ctrl;               // device
        FusedGeom fg;
        unsigned n_tickets;            // = grid size
        unsigned long long wait_ns;    // a dependency wait longer than this gives up and aborts the launch (su_set_option "fuse_wait_ns")
    } fz;
};

// checkerboard index, in the neighbour's buffer, of the halo copy of an edge site (all slabs have Lt_int slices)
__device__ __forceinline__ unsigned halo_cb_lo(const Geom& g, unsigned cb) { SUG_ASSERT(cb + (unsigned)g.Lt_int * g.Vsh < g.Vh); return cb + (unsigned)g.Lt_int * g.Vsh; }   // -> their upper halo
__device__ __forceinline__ unsigned halo_cb_hi(const Geom& g, unsigned cb) { SUG_ASSERT(cb >= (unsigned)g.Lt_int * g.Vsh); return cb - (unsigned)g.Lt_int * g.Vsh; }   // -> their lower halo

// The site a thread works on and the checkerboard-index offsets of its 8 neighbours.
struct SiteNbr {
    unsigned cb;        // checkerboard index of x in the stored lattice
    uint32_t lex;       // lexicographic index of x in the global lattice (RNG counter word c0)
    int dp[4], dm[4];   // cb(x + e_d) - cb(x), cb(x - e_d) - cb(x)   (periodic)
};

__device__ __forceinline__ int sel4(int i, int v0, int v1, int v2, int v3) {
    return i == 0 ? v0 : (i == 1 ? v1 : (i == 2 ? v2 : v3));
}

// (x/2, y, z, stored t) of a site of the given parity -> checkerboard index, RNG site index, neighbour offsets
__device__ __forceinline__ void site_from_coords(const Geom& g, unsigned xh, unsigned y, unsigned z, unsigned t, int parity, SiteNbr& s) {
    const unsigned row = (unsigned)g.Lxh, pl = row * (unsigned)g.L[1];
    const int sy = (int)row, sz = (int)pl, st = (int)(pl * (unsigned)g.L[2]);
    const int q = (int)((y + z + t + (unsigned)g.t0g + (unsigned)parity) & 1u);          // x = 2 xh + q
    s.cb = xh + row * (y + (unsigned)g.L[1] * (z + (unsigned)g.L[2] * t));
    s.lex = 2u * (xh + row * (y + (unsigned)g.L[1] * (z + (unsigned)g.L[2] * (unsigned)global_t(g, (int)t)))) + (unsigned)q;
    s.dp[0] = q ? ((int)xh + 1 == g.Lxh ? 1 - g.Lxh : 1) : 0;
    s.dm[0] = q ? 0 : (xh == 0 ? g.Lxh - 1 : -1);
    s.dp[1] = ((int)y + 1 == g.L[1]) ? -(g.L[1] - 1) * sy : sy;
    s.dm[1] = (y == 0) ? (g.L[1] - 1) * sy : -sy;
    s.dp[2] = ((int)z + 1 == g.L[2]) ? -(g.L[2] - 1) * sz : sz;
    s.dm[2] = (z == 0) ? (g.L[2] - 1) * sz : -sz;
    if (g.t_halo) {             // the neighbours in t are the halo slices: no wrap inside the buffer
        s.dp[3] = st; s.dm[3] = -st;
    } else {
        s.dp[3] = ((int)t + 1 == g.L[3]) ? -(g.L[3] - 1) * st : st;
        s.dm[3] = (t == 0) ? (g.L[3] - 1) * st : -st;
    }
#if defined(SUG_CHECK) && SUG_CHECK
    SUG_ASSERT(s.cb < g.Vh);
    for (int d = 0; d < 4; ++d) {
        SUG_ASSERT(s.cb + (unsigned)s.dp[d] < g.Vh && s.cb + (unsigned)s.dm[d] < g.Vh);
        for (int e = 0; e < 4; ++e) SUG_ASSERT(e == d || s.cb + (unsigned)(s.dm[d] + s.dp[e]) < g.Vh);      // x - d + e
    }
#endif
}

// Block tiles (Geom::Bz, Bt; su_set_option "block_tile_z" / "block_tile_t") are compiled in only with -DSUG_BLOCK_TILES=1:
// the second decode path alone made ptxas keep 544 bytes of the SU(4) fp64 kernel's matrices in local memory (OR sub-step
// 0.093 -> 0.162 ms at 24^4), and the tiles bought nothing (profiles/r02g section 7).
#ifndef SUG_BLOCK_TILES
#define SUG_BLOCK_TILES 0
#endif
// traversal index (over the OWNED sites of one parity) -> (x/2, y, z, interior t); all indices stay in registers
__device__ __forceinline__ void traversal_coords(const Geom& g, unsigned tix, unsigned& xh, unsigned& y, unsigned& z, unsigned& ti) {
    const unsigned row = (unsigned)g.Lxh, pl = row * (unsigned)g.L[1];
#if SUG_BLOCK_TILES
    if (g.Bz * g.Bt > 1) {
        // block tiles: (z-chunk, t-block, z-block, x-y segment group | warp: segment, t in block, z in block | lane)
        const unsigned wb = (unsigned)g.Wb, bz = (unsigned)g.Bz, bt = (unsigned)g.Bt, sw = wb / (bz * bt);
        const unsigned W = tix >> 5, lane = tix & 31u, blk = W / wb, w = W - blk * wb;
        const unsigned dz = w % bz, dt = (w / bz) % bt, sl = w / (bz * bt);
        const unsigned sgroups = (pl >> 5) / sw, nzb = (unsigned)g.Zc / bz, ntb = (unsigned)g.Lt_int / bt;
        unsigned q = blk;
        const unsigned sb = q % sgroups; q /= sgroups;
        const unsigned zb = q % nzb;     q /= nzb;
        const unsigned tb = q % ntb;
        const unsigned zc = q / ntb;
        const unsigned r = ((sb * sw + sl) << 5) + lane;
        y = r / row; xh = r - y * row;
        z = zc * (unsigned)g.Zc + zb * bz + dz;
        ti = tb * bt + dt;
        return;
    }
#endif
    const unsigned grp = pl * (unsigned)g.Zc, span = grp * (unsigned)g.Lt_int;
    const unsigned zc = tix / span;  unsigned r = tix - zc * span;
    ti = r / grp;                    r -= ti * grp;
    const unsigned zi = r / pl;      r -= zi * pl;
    y = r / row;
    xh = r - y * row;
    z = zc * (unsigned)g.Zc + zi;
}
__device__ __forceinline__ void site_of_thread(const Geom& g, unsigned tix, int parity, SiteNbr& s) {
    unsigned xh, y, z, ti;
    traversal_coords(g, tix, xh, y, z, ti);
    site_from_coords(g, xh, y, z, ti + (unsigned)g.t_halo, parity, s);          // stored time slice
}

// slab mode: 1 = the thread's site lies in the first owned time slice, 2 = in the last one, 0 otherwise.
// Recomputed from the traversal index at store time so that nothing stays live across the kernel body.
__device__ __forceinline__ int slab_edge(const Geom& g, unsigned tix) {
    if (!g.t_halo) return 0;
    unsigned xh, y, z, ti;
    traversal_coords(g, tix, xh, y, z, ti);
    return (ti == 0 ? 1 : 0) | ((int)ti + 1 == g.Lt_int ? 2 : 0);
}

// L2 prefetch ahead of the traversal (su_set_option "prefetch_slices"). The traversal walks up in t inside a z-chunk,
// and the links of the slice above are the only ones a sub-step touches for the first time (DESIGN.md "Traversal
// order"); with few warps per SM (fused launches) nothing hides their DRAM latency. So every warp, before it starts on
// its 32 sites, asks L2 for the eight link tiles (4 mu x 2 parities, E * 512 B each, contiguous in the tiled layout)
// that hold the same sites k time slices further up: one cp.async.bulk.prefetch.L2 per (mu, parity), issued by lanes
// 0..7. A hint only: it moves no data into the SM, orders nothing and cannot change a result.
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
template <int E, class T2>
__device__ __forceinline__ void prefetch_slices_ahead(const void* links, const Geom& g, unsigned cb0, int k) {
    constexpr unsigned BYTES = E * LINK_TILE * sizeof(T2);
    if (BYTES % 16 != 0) return;
    const unsigned lane = threadIdx.x & 31u;
    if (lane < 8) {
        const unsigned cbT = (unsigned)(((unsigned long long)cb0 + (unsigned long long)k * g.Vsh) % g.Vh);
        const T2* p = (const T2*)links + (size_t)lane * E * g.Vhp + (size_t)(cbT / LINK_TILE) * (E * LINK_TILE);
        l2_prefetch_bulk(p, BYTES);
    }
}

// FUSE3: each staple term S += A B C (three links) is evaluated row by row with all three operands
// loaded up front (Mat::acc_nnd / acc_dnn): half as many load-wait phases per thread as the
// two-step form (P = A B; S += P C), for the same registers. KUNR: unroll the loop over nu.
// LDN: how neighbour links are loaded (LD_RO in a plain launch, LD_COHERENT in a fused one).
//
// update_link: staple, W = U S^dagger, subgroup loop and store for ONE link U_mu(x), x = s (rows a1-a6).
template <int NC, class T, int STORE, int KIND, bool UNR, int BLOCK, int FUSE3, bool KUNR, int LDN, int PRE, bool FUSED>
__device__ __forceinline__ void update_link(const UpdateArgs& a, const int p, const int mu, const SiteNbr& s, const unsigned tix,
                                            const unsigned warp_mask, const uint32_t sweep_ctr, T* dir_col,
                                            unsigned& att_total, unsigned& exhausted, cx<T>* s_col = nullptr) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    typedef Mat<NC, T, UNR> M;
    typedef cx<T> C;
    constexpr int NSUB = NC * (NC - 1) / 2;
    constexpr int LDT = (!FUSED && SUG_TMINUS_STREAM) ? LD_STREAM : LDN;     // links of the time slice below
    const unsigned cb = s.cb;
    const int dpmu = sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
    // heatbath, register kernels: the directions of all subgroup draws are link-independent; evaluate them
    // now, in the shadow of the first loads, and park them in shared memory (one private column per thread)
    // PRE == 4: the same quantities, but draw q is evaluated in the shadow of the loads of staple term 6 q / NSUB
    // (between issuing a term's three links and multiplying them), where the warp would otherwise only wait
    auto pre_draw = [&](int q) {
        T n[3], Q, R;
        kp_direction<T>(a.k0, a.k1, s.lex, sweep_ctr, pack_c2((int)a.pass, p, mu, q), n);
        kp_attempt0<T>(a.k0, a.k1, s.lex, sweep_ctr, pack_c2((int)a.pass, p, mu, q), Q, R);
        dir_col[(3 * q) * BLOCK] = n[0]; dir_col[(3 * q + 1) * BLOCK] = n[1]; dir_col[(3 * q + 2) * BLOCK] = n[2];
        dir_col[(3 * NSUB + 2 * q) * BLOCK] = Q; dir_col[(3 * NSUB + 2 * q + 1) * BLOCK] = R;
    };
    auto pre_slot = [&](int slot) {
        if (PRE == 4) {
#pragma unroll
            for (int q = 0; q < NSUB; ++q) if ((q * 6) / NSUB == slot) pre_draw(q);
        }
    };
    if (PRE >= 1 && PRE != 4) {
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            T n[3];
            kp_direction<T>(a.k0, a.k1, s.lex, sweep_ctr, pack_c2((int)a.pass, p, mu, q), n);
            dir_col[(3 * q) * BLOCK] = n[0]; dir_col[(3 * q + 1) * BLOCK] = n[1]; dir_col[(3 * q + 2) * BLOCK] = n[2];
        }
    }
    if (PRE >= 2 && PRE != 4) {
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            T Q, R;
            kp_attempt0<T>(a.k0, a.k1, s.lex, sweep_ctr, pack_c2((int)a.pass, p, mu, q), Q, R);
            dir_col[(3 * NSUB + 2 * q) * BLOCK] = Q; dir_col[(3 * NSUB + 2 * q + 1) * BLOCK] = R;
        }
    }

    C S[NC * NC], A[NC * NC], B[NC * NC], P[NC * NC];
    M::zero(S);
    bool self_loaded = false;
    const typename IO::T2* pl_mu_o = IO::plane((const void*)a.links, a.g, mu, 1 - p);
    typename IO::T2* pl_self = IO::plane(a.links, a.g, mu, p);
    constexpr bool STREAM_SELF = !FUSED || SUG_FUSED_STREAM;
    if constexpr (FUSE3 == 4) {
        // The staple sum lives in shared memory (one private column per thread, s_col[e * BLOCK]) while the six terms are
        // formed: 36 (fp64) registers fewer during the phase that holds three loaded links, so that a 128-register budget -
        // 16 instead of 12 warps per SM, a third more loads in flight - does not spill. Terms as in FUSE3 == 1 (three
        // links up front, row by row); the same sums in the same order.
        auto term = [&](bool upper, bool first) {
#pragma unroll
            for (int i = 0; i < NC; ++i) {
                C r[NC];
#pragma unroll
                for (int j = 0; j < NC; ++j) {
                    C acc = mk<T>(0, 0);
#pragma unroll
                    for (int k = 0; k < NC; ++k) { if (upper) mad(acc, A[i * NC + k], B[k * NC + j]); else mad_ca(acc, A[k * NC + i], B[k * NC + j]); }
                    r[j] = acc;
                }
#pragma unroll
                for (int j = 0; j < NC; ++j) {
                    C acc = first ? mk<T>(0, 0) : s_col[(i * NC + j) * BLOCK];
#pragma unroll
                    for (int k = 0; k < NC; ++k) { if (upper) mad_cb(acc, r[k], P[j * NC + k]); else mad(acc, r[k], P[k * NC + j]); }
                    s_col[(i * NC + j) * BLOCK] = acc;
                }
            }
        };
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int nu = k + (k >= mu ? 1 : 0);
            const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
            const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
            const typename IO::T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
            const typename IO::T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
            IO::template load<LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
            IO::template load<LDN>(pl_nu_o, cb + (unsigned)dpmu, P);
            IO::template load<LDN>(pl_nu_s, cb, A);
            term(true, k == 0);
            if (LDT != LDN && nu == 3) {
                IO::template load<LDT>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load<LDT>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load<LDT>(pl_nu_o, cb + (unsigned)dmnu, A);
            } else {
                IO::template load<LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load<LDN>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load<LDN>(pl_nu_o, cb + (unsigned)dmnu, A);
            }
            term(false, false);
        }
#pragma unroll
        for (int e = 0; e < NC * NC; ++e) S[e] = s_col[e * BLOCK];
    } else if constexpr (FUSE3 == 3) {
        // two-row storage with lazy third rows (Su3Rows): three links up front per term, as FUSE3 == 1
        static_assert(STORE == STORE_RECON12 && NC == 3 && UNR, "FUSE3 == 3 is the SU(3) two-row form");
#pragma unroll(KUNR ? 3 : 1)
        for (int k = 0; k < 3; ++k) {
            const int nu = k + (k >= mu ? 1 : 0);
            const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
            const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
            const typename IO::T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
            const typename IO::T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
            IO::template load_stored<LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
            IO::template load_stored<LDN>(pl_nu_o, cb + (unsigned)dpmu, P);
            IO::template load_stored<LDN>(pl_nu_s, cb, A);
            pre_slot(2 * k);
            Su3Rows<T>::acc_upper(S, A, B, P);
            if (LDT != LDN && nu == 3) {
                IO::template load_stored<LDT>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load_stored<LDT>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load_stored<LDT>(pl_nu_o, cb + (unsigned)dmnu, A);
            } else {
                IO::template load_stored<LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load_stored<LDN>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load_stored<LDN>(pl_nu_o, cb + (unsigned)dmnu, A);
            }
            pre_slot(2 * k + 1);
            Su3Rows<T>::acc_lower(S, A, B, P);
        }
    } else if constexpr (FUSE3 == 2) {
        // Software pipeline over the six staple terms (few warps per SM: nothing else hides the load latency). A term is
        // P = A B (or A^dagger B), then S += P C^dagger (or P C). While P is formed the term's third link C is in
        // flight; while S is accumulated the first two links of the NEXT term are (the own link after the last
        // term). Same sums in the same order as mul_nn + acc_nd / mul_dn + acc_nn, i.e. as the FUSE3 == 1 form.
        C Cm[NC * NC];
        auto nu_of = [&](int k) { return k + (k >= mu ? 1 : 0); };
        auto load_ab = [&](int t) {       // first two links of term t (t = 2 k: upper, 2 k + 1: lower)
            const int nu = nu_of(t >> 1);
            const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]), dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
            if (!(t & 1)) {               // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
                IO::template load<LDN>(IO::plane((const void*)a.links, a.g, nu, p), cb, A);
                IO::template load<LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
            } else if (LDT != LDN && nu == 3) {   // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu); slice below: evict-first
                IO::template load<LDT>(IO::plane((const void*)a.links, a.g, nu, 1 - p), cb + (unsigned)dmnu, A);
                IO::template load<LDT>(pl_mu_o, cb + (unsigned)dmnu, B);
            } else {
                IO::template load<LDN>(IO::plane((const void*)a.links, a.g, nu, 1 - p), cb + (unsigned)dmnu, A);
                IO::template load<LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
            }
        };
        auto load_c = [&](int t) {
            const int nu = nu_of(t >> 1);
            const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
            if (!(t & 1))                        IO::template load<LDN>(IO::plane((const void*)a.links, a.g, nu, 1 - p), cb + (unsigned)dpmu, Cm);
            else if (LDT != LDN && nu == 3)      IO::template load<LDT>(IO::plane((const void*)a.links, a.g, nu, p), cb + (unsigned)(dmnu + dpmu), Cm);
            else                                 IO::template load<LDN>(IO::plane((const void*)a.links, a.g, nu, p), cb + (unsigned)(dmnu + dpmu), Cm);
        };
        load_ab(0);
#pragma unroll
        for (int t = 0; t < 6; ++t) {
            load_c(t);
            if (!(t & 1)) M::mul_nn(A, B, P); else M::mul_dn(A, B, P);
            if (t < 5) load_ab(t + 1);
            else IO::template load<STREAM_SELF ? LD_STREAM : LDN>(pl_self, cb, A);       // the own link U
            pre_slot(t);
            if (!(t & 1)) M::acc_nd(S, P, Cm); else M::acc_nn(S, P, Cm);
        }
    } else {
#pragma unroll(KUNR ? 3 : 1)
    for (int k = 0; k < 3; ++k) {
        const int nu = k + (k >= mu ? 1 : 0);
        const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
        const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
        const typename IO::T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
        const typename IO::T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
        if (FUSE3) {
            // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
            IO::template load<LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
            IO::template load<LDN>(pl_nu_o, cb + (unsigned)dpmu, P);
            IO::template load<LDN>(pl_nu_s, cb, A);
            pre_slot(2 * k);
            M::acc_nnd(S, A, B, P);
            // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
            if (LDT != LDN && k == 2 && nu == 3) {
                // links of the time slice below: with the traversal walking up in t this is their last
                // use in the sub-step, so they are fetched evict-first and leave L2 to the slices ahead
                IO::template load<LDT>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load<LDT>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load<LDT>(pl_nu_o, cb + (unsigned)dmnu, A);
            } else {
                IO::template load<LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
                IO::template load<LDN>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                IO::template load<LDN>(pl_nu_o, cb + (unsigned)dmnu, A);
            }
            pre_slot(2 * k + 1);
            if (SUG_EARLY_SELF && UNR && k == 2) {
                // last term in two steps, B <- A^dagger B in place: A is free before the accumulation, so the own link (the
                // eighth and last load wait of the site) is requested now and arrives while S += B P runs. Same sums.
                M::mul_dn_inplace(A, B);
                IO::template load<STREAM_SELF ? LD_STREAM : LDN>(pl_self, cb, A);
                M::acc_nn(S, B, P);
                self_loaded = true;
            } else {
                M::acc_dnn(S, A, B, P);
            }
        } else {
            // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
            IO::template load<LDN>(pl_nu_s, cb, A);
            IO::template load<LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
            M::mul_nn(A, B, P);
            IO::template load<LDN>(pl_nu_o, cb + (unsigned)dpmu, A);
            M::acc_nd(S, P, A);
            // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
            IO::template load<LDN>(pl_nu_o, cb + (unsigned)dmnu, A);
            IO::template load<LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
            M::mul_dn(A, B, P);
            IO::template load<LDN>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), A);
            M::acc_nn(S, P, A);
        }
    }
    }
    C* U = A;
    C* W = B;
    if (FUSE3 != 2 && !self_loaded) IO::template load<STREAM_SELF ? LD_STREAM : LDN>(pl_self, cb, U);
    M::mul_nd(U, S, W);                                   // W = U S^dagger
    update_subgroups<NC, T, KIND, UNR>(U, W, (T)a.beta, a.k0, a.k1, s.lex, sweep_ctr,
                                       pack_c2((int)a.pass, p, mu, 0),
                                       a.attempts ? a.attempts + cb : nullptr, (size_t)a.g.Vh,
                                       att_total, exhausted, warp_mask,
                                       PRE >= 1 ? dir_col : nullptr, PRE >= 1 ? BLOCK : 0,
                                       PRE >= 2 ? dir_col + 3 * NSUB * BLOCK : nullptr);
    if (UNR && NC <= 4) {
        if (a.reunit) reunitarize_small<NC <= 4 ? NC : 2, T>(U);       // su_set_option "reunit_on_store": last pass of a sweep
    }
    IO::template store<STREAM_SELF>(pl_self, cb, U);
    if (!FUSED) {                             // plain launch: halo push fused into the store (slab mode only);
        if (const int edge = slab_edge(a.g, tix)) {       // recomputed here so that nothing stays live across the body
            if (edge & 1) IO::template store<true>(IO::plane(a.peer_lo, a.g, mu, p), halo_cb_lo(a.g, cb), U);
            if (edge & 2) IO::template store<true>(IO::plane(a.peer_hi, a.g, mu, p), halo_cb_hi(a.g, cb), U);
        }
    }
}

// ---- fused launches: waiting for and signalling the completion of (stage, cell) (fused_schedule.h) ----
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// warp 0 of the block, non-blocking: true iff every dependency of the work item is already complete
__device__ __forceinline__ bool fused_probe(const UpdateArgs::Fused& fz, int s, int cell, int tile, unsigned epoch) {
    const unsigned target = (epoch + 1u) * (unsigned)fz.fg.nT;
    bool ok = true;
    for (int k = (int)threadIdx.x; k < s * FUSED_DEPS_PER_STAGE; k += 32) {
        const int idx = fused_dep(fz.fg, s, cell, tile, k);
        if (idx >= 0 && (int)(ld_acquire_u32(fz.done + idx) - target) < 0) ok = false;
    }
    return __all_sync(0xffffffffu, ok);
}
// warp 0 of the block: every lane polls some of the work item's dependencies. Returns (to every lane) whether they are
// all complete. false = this wait, or one in another block, lasted longer than fz.wait_ns of WALL-CLOCK time
// (%globaltimer, so a slow instrumented or debug build does not trip it) and FusedCtrl::error is set: the caller must
// not run the work item, so that no link computed from incomplete neighbours is ever stored. A correct schedule never
// gets there; the host reports SU_ECUDA at its next synchronising call and rebuilds the tables (check_fused_error).
__device__ __forceinline__ bool fused_wait(const UpdateArgs::Fused& fz, int s, int cell, int tile, unsigned epoch) {
    const unsigned target = (epoch + 1u) * (unsigned)fz.fg.nT;
    bool ok = true;
    unsigned long long t0 = 0;
    for (int k = (int)threadIdx.x; ok && k < s * FUSED_DEPS_PER_STAGE; k += 32) {
        const int idx = fused_dep(fz.fg, s, cell, tile, k);
        if (idx < 0) continue;
        unsigned spins = 0;
        while ((int)(ld_acquire_u32(fz.done + idx) - target) < 0) {
            __nanosleep(64);
            if ((spins++ & 63u) == 0) {      // on the first unsuccessful poll, then every 64th
                if (*(volatile unsigned*)&fz.ctrl->error) { ok = false; break; }      // another block gave up: follow at once
                const unsigned long long now = global_ns();
                if (t0 == 0) t0 = now;
                if (now - t0 >= fz.wait_ns) { atomicExch(&fz.ctrl->error, 1u); ok = false; break; }
            }
        }
    }
    return __all_sync(0xffffffffu, ok);
}

template <int NC, class T, int STORE, int KIND, bool UNR, int BLOCK, int MINB, int FUSE3 = 0, bool KUNR = false, bool FUSED = false>
__global__ void __launch_bounds__(BLOCK, MINB) k_update(const UpdateArgs a) {
    constexpr int NSUB = NC * (NC - 1) / 2;
    constexpr int PRE_ASKED = ((KIND == KIND_HB) && UNR) ? (sizeof(T) == 4 ? SUG_KP_PRE_F32 : SUG_KP_PRE_F64) : 0;
    constexpr int PRE = (PRE_ASKED == 4 && !FUSE3) ? (sizeof(T) == 4 ? 1 : 0) : PRE_ASKED;     // 4 needs the three-link staple terms
    __shared__ T dir_sm[PRE >= 2 ? 5 * NSUB : (PRE == 1 ? 3 * NSUB : 1)][PRE ? BLOCK : 1];
    __shared__ cx<T> s_sm[FUSE3 == 4 ? NC * NC : 1][FUSE3 == 4 ? BLOCK : 1];      // FUSE3 == 4: the staple sums
    const uint32_t sweep_ctr = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
    unsigned att_total = 0, exhausted = 0;
    if (!FUSED) {
        const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
        const bool active = tix < a.g.Vh_int;
        const unsigned warp_mask = __ballot_sync(0xffffffffu, active);      // lanes that run the body (ragged last warp)
        if (active) {
            SiteNbr s;
            site_of_thread(a.g, tix, a.parity, s);
            if (a.pf_slices > 0)
                prefetch_slices_ahead<LinkIO<NC, T, STORE, UNR>::E, typename V2<T>::type>(a.links, a.g, __shfl_sync(warp_mask, s.cb, 0), a.pf_slices);
            update_link<NC, T, STORE, KIND, UNR, BLOCK, FUSE3, KUNR, SUG_NEIGHBOUR_LD, PRE, false>(
                a, a.parity, a.mu, s, tix, warp_mask, sweep_ctr, &dir_sm[0][PRE ? threadIdx.x : 0], att_total, exhausted,
                &s_sm[0][FUSE3 == 4 ? threadIdx.x : 0]);
        }
    } else {
        __shared__ unsigned sh_ticket, sh_epoch, sh_ready[2], sh_abort;     // sh_ready alternates per phase: no reuse race
        if (threadIdx.x == 0) {
            sh_abort = 0u;
            sh_epoch = *(volatile unsigned*)&a.fz.ctrl->epoch;
            sh_ticket = atomicAdd(&a.fz.ctrl->ticket, 1u);
        }
        __syncthreads();
        const unsigned ticket = sh_ticket, epoch = sh_epoch;
        const int ncells = a.fz.fg.Lt * a.fz.fg.nzu, g = a.fz.fg.g;
        const uint32_t* work = a.fz.work + (size_t)ticket * g;
        // Phase boundary = normally ONE block barrier. Warp 0 PROBES the dependencies of the next work item as soon as
        // it has issued its own stores of the current one (the other warps are still computing); after the barrier
        // the last warp publishes the finished item (fence + counter) while everybody already loads for the next
        // one. Only if the probe failed does warp 0 spin, after the publication (publishing must never wait on other
        // blocks: that would chain the blocks' signals one behind the other), followed by a second barrier.
        int st = 0, flip = 0;
        while (st < g && __ldg(work + st) == FUSED_NONE) ++st;
        if (st > 0 && st < g) {                                // a block whose first item is not of stage 0 (pipeline drain)
            const uint32_t id = __ldg(work + st);
            const int cell = (int)(id / (unsigned)a.fz.fg.nT);
            if (threadIdx.x < 32) {
                const bool ok = fused_wait(a.fz, st, cell, (int)(id - (unsigned)cell * (unsigned)a.fz.fg.nT), epoch);
                if (threadIdx.x == 0 && !ok) sh_abort = 1u;
            }
            __syncthreads();
            if (sh_abort) st = g;                              // gave up: run nothing, store nothing
        }
#pragma unroll 1
        while (st < g) {
            const uint32_t id = __ldg(work + st);              // uniform over the block
            const int cell = (int)(id / (unsigned)a.fz.fg.nT), tile = (int)(id - (unsigned)cell * (unsigned)a.fz.fg.nT);
            const unsigned r = (unsigned)tile * BLOCK + threadIdx.x;
            const bool active = r < (unsigned)a.fz.fg.cell_sites;
            const unsigned warp_mask = __ballot_sync(0xffffffffu, active);
            if (active) {
                const unsigned t = (unsigned)cell / (unsigned)a.fz.fg.nzu, zu = (unsigned)cell - t * (unsigned)a.fz.fg.nzu;
                const unsigned zi = r / (unsigned)a.fz.fg.plane_sites, rem = r - zi * (unsigned)a.fz.fg.plane_sites;
                const unsigned y = rem / (unsigned)a.g.Lxh, xh = rem - y * (unsigned)a.g.Lxh;
                const int p = fused_parity(a.fz.fg, st), mu = fused_mu(a.fz.fg, st);
                SiteNbr s;
                site_from_coords(a.g, xh, y, zu * (unsigned)a.fz.fg.U + zi, t, p, s);
                if (a.pf_slices > 0 && st == 0)             // the first stage is the one that touches links for the first time
                    prefetch_slices_ahead<LinkIO<NC, T, STORE, UNR>::E, typename V2<T>::type>(a.links, a.g, __shfl_sync(warp_mask, s.cb, 0), a.pf_slices);
                update_link<NC, T, STORE, KIND, UNR, BLOCK, FUSE3, KUNR, SUG_FUSED_LD, PRE, true>(
                    a, p, mu, s, 0u, warp_mask, sweep_ctr, &dir_sm[0][PRE ? threadIdx.x : 0], att_total, exhausted,
                    &s_sm[0][FUSE3 == 4 ? threadIdx.x : 0]);
            }
            int nx = st + 1;
            while (nx < g && __ldg(work + nx) == FUSED_NONE) ++nx;
            uint32_t idn = 0;
            int celln = 0, tilen = 0;
            if (nx < g) {
                idn = __ldg(work + nx);
                celln = (int)(idn / (unsigned)a.fz.fg.nT); tilen = (int)(idn - (unsigned)celln * (unsigned)a.fz.fg.nT);
                if (threadIdx.x < 32) {
                    const bool ok = fused_probe(a.fz, nx, celln, tilen, epoch);
                    if (threadIdx.x == 0) sh_ready[flip] = ok ? 1u : 0u;
                }
            }
            if (st + 1 < g) {                                  // nobody waits for the last stage
                __syncthreads();
                if (threadIdx.x == BLOCK - 32) { __threadfence(); atomicAdd(a.fz.done + (size_t)st * ncells + cell, 1u); }
                if (nx < g && !sh_ready[flip]) {               // uniform: written before the barrier
                    if (threadIdx.x < 32) {
                        const bool ok = fused_wait(a.fz, nx, celln, tilen, epoch);
                        if (threadIdx.x == 0 && !ok) sh_abort = 1u;
                    }
                    __syncthreads();
                    if (sh_abort) break;                       // gave up: the remaining work items are not run
                }
            }
            st = nx; flip ^= 1;
        }
        if (threadIdx.x == 0) {                                // the last block out re-arms the table for the next launch
            if (atomicAdd(&a.fz.ctrl->exited, 1u) == a.fz.n_tickets - 1u) {
                a.fz.ctrl->ticket = 0; a.fz.ctrl->exited = 0;
                __threadfence();
                a.fz.ctrl->epoch = epoch + 1u;
            }
        }
    }
    if (KIND == KIND_HB) {
        for (int o = 16; o > 0; o >>= 1) {
            att_total += __shfl_down_sync(0xffffffffu, att_total, o);
            exhausted += __shfl_down_sync(0xffffffffu, exhausted, o);
        }
        if ((threadIdx.x & 31) == 0) {
            if (att_total) atomicAdd(a.counters, (unsigned long long)att_total);
            if (exhausted) atomicAdd(a.counters + 1, (unsigned long long)exhausted);
        }
    }
}

// ------------------------------------------------------------------------------------------
// SU(2) in the 4-real parameterisation U = a0 + i a.sigma (eqs 6-8): links,
// staple and update are quaternion arithmetic. Same algebra as the matrix path:
// W = U S^bar, k = |W|, u~ = W/k, a = v u~^bar (heatbath, eq 14) or (u~^bar)^2 (eq 17), U' = a U.
// ------------------------------------------------------------------------------------------
template <class T> __device__ __forceinline__ size_t qsite(unsigned cb) {      // tiled layout, 2 pairs per link
    return (size_t)(cb / LINK_TILE) * (2 * LINK_TILE) + (cb % LINK_TILE);
}
template <class T, int LD> __device__ __forceinline__ void qload(const typename V2<T>::type* __restrict__ pl, unsigned cb, T q[4]) {
    pl += qsite<T>(cb);
    typename V2<T>::type v0 = ldg2<T, LD>(pl);
    typename V2<T>::type v1 = ldg2<T, LD>(pl + LINK_TILE);
    q[0] = v0.x; q[1] = v0.y; q[2] = v1.x; q[3] = v1.y;
}
template <class T> __device__ __forceinline__ void qconj(const T a[4], T o[4]) { o[0] = a[0]; o[1] = -a[1]; o[2] = -a[2]; o[3] = -a[3]; }

// one SU(2) link U_mu(x), x = s of parity p. LDN: how neighbour links are loaded; PLAIN: one sub-step per launch (streaming
// own link, halo push in slab mode) - false inside the cooperative whole-pass kernel
template <class T, int KIND, int LDN, bool PLAIN>
__device__ __forceinline__ void update_link_su2(const UpdateArgs& a, const int p, const int mu, const SiteNbr& s, const unsigned tix,
                                                const unsigned warp_mask, const uint32_t sweep_ctr, unsigned& att_total, unsigned& exhausted) {
    typedef typename V2<T>::type T2;
    const unsigned cb = s.cb;
    const int dpmu = sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
    const T2* base = (const T2*)a.links;
    auto plane = [&](int d, int par) { return base + (size_t)(d * 2 + par) * 2 * a.g.Vhp; };
    T S[4] = {0, 0, 0, 0}, A[4], B[4], Cq[4], P[4], Q[4];
    const T2* pl_mu_o = plane(mu, 1 - p);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int nu = k + (k >= mu ? 1 : 0);
        const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
        const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
        const T2* pl_nu_s = plane(nu, p);
        const T2* pl_nu_o = plane(nu, 1 - p);
        qload<T, LDN>(pl_nu_s, cb, A);
        qload<T, LDN>(pl_mu_o, cb + (unsigned)dpnu, B);
        qload<T, LDN>(pl_nu_o, cb + (unsigned)dpmu, Cq);
        quat_mul(A, B, P); qconj(Cq, A); quat_mul(P, A, Q);
        S[0] += Q[0]; S[1] += Q[1]; S[2] += Q[2]; S[3] += Q[3];
        qload<T, LDN>(pl_nu_o, cb + (unsigned)dmnu, A);
        qload<T, LDN>(pl_mu_o, cb + (unsigned)dmnu, B);
        qload<T, LDN>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), Cq);
        qconj(A, P); quat_mul(P, B, Q); quat_mul(Q, Cq, P);
        S[0] += P[0]; S[1] += P[1]; S[2] += P[2]; S[3] += P[3];
    }
    T2* pl_self = (T2*)a.links + (size_t)(mu * 2 + p) * 2 * a.g.Vhp;
    T U[4], W[4], a4[4] = {1, 0, 0, 0};
    qload<T, PLAIN ? LD_STREAM : LDN>(pl_self, cb, U);
    qconj(S, A);
    quat_mul(U, A, W);
    const T n2 = norm2_4(W[0], W[1], W[2], W[3]);      // k^2
    bool ok = (n2 >= Fn<T>::min_norm2()) && Fn<T>::finite(n2);      // as in update_subgroups
    int used = 0;
    const unsigned draw_mask = (KIND == KIND_HB) ? __ballot_sync(warp_mask, ok) : 0u;
    if (ok) {
        if (KIND == KIND_HB) {
            const T ik = Fn<T>::rsqrt_pos(n2), k = n2 * ik;
            T ud[4] = {W[0] * ik, -W[1] * ik, -W[2] * ik, -W[3] * ik};
            T v[4];
            used = kp_draw<T>(draw_mask, (T)a.beta * k, (T)-0.5 / (T)a.beta * ik, a.k0, a.k1, s.lex, sweep_ctr,
                              pack_c2((int)a.pass, p, mu, 0), v);
            if (used) quat_mul(v, ud, a4); else ok = false;
        } else {
            // a = conj(W)^2 / k^2 (eq 17)
            const T in2 = Fn<T>::rcp_pos(n2), m2w0 = (T)-2 * W[0] * in2;
            a4[0] = fma_x(W[0], W[0], -fma_x(W[3], W[3], fma_x(W[2], W[2], mul_x(W[1], W[1])))) * in2;
            a4[1] = m2w0 * W[1]; a4[2] = m2w0 * W[2]; a4[3] = m2w0 * W[3];
        }
    }
    if (KIND == KIND_HB) {
        att_total += (unsigned)used;
        exhausted += ok ? 0u : 1u;
        if (a.attempts) a.attempts[cb] = (uint8_t)(used > 255 ? 255 : used);
    }
    if (ok) {
        quat_mul(a4, U, P);
        if (a.reunit) {
            const T inv = (T)1 / Fn<T>::sqrt(norm2_4(P[0], P[1], P[2], P[3]));
            P[0] *= inv; P[1] *= inv; P[2] *= inv; P[3] *= inv;
        }
        T2* q = pl_self + qsite<T>(cb);
        stg2<T, PLAIN>(q, V2<T>::make(P[0], P[1]));
        stg2<T, PLAIN>(q + LINK_TILE, V2<T>::make(P[2], P[3]));
        if (PLAIN) {
            if (const int edge = slab_edge(a.g, tix)) {      // fused halo push (slab mode only)
                const size_t plane_off = (size_t)(mu * 2 + p) * 2 * a.g.Vhp;
                if (edge & 1) {
                    T2* h = (T2*)a.peer_lo + plane_off + qsite<T>(halo_cb_lo(a.g, cb));
                    stg2<T, true>(h, V2<T>::make(P[0], P[1])); stg2<T, true>(h + LINK_TILE, V2<T>::make(P[2], P[3]));
                }
                if (edge & 2) {
                    T2* h = (T2*)a.peer_hi + plane_off + qsite<T>(halo_cb_hi(a.g, cb));
                    stg2<T, true>(h, V2<T>::make(P[0], P[1])); stg2<T, true>(h + LINK_TILE, V2<T>::make(P[2], P[3]));
                }
            }
        }
    }
}

__device__ __forceinline__ void flush_kp_counters(const UpdateArgs& a, unsigned att_total, unsigned exhausted) {
    for (int o = 16; o > 0; o >>= 1) {
        att_total += __shfl_down_sync(0xffffffffu, att_total, o);
        exhausted += __shfl_down_sync(0xffffffffu, exhausted, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (att_total) atomicAdd(a.counters, (unsigned long long)att_total);
        if (exhausted) atomicAdd(a.counters + 1, (unsigned long long)exhausted);
    }
}

template <class T, int KIND, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) k_update_su2(const UpdateArgs a) {
    const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = tix < a.g.Vh_int;
    const unsigned warp_mask = __ballot_sync(0xffffffffu, active);
    unsigned att_total = 0, exhausted = 0;
    if (active) {
        SiteNbr s;
        site_of_thread(a.g, tix, a.parity, s);
        update_link_su2<T, KIND, LD_RO, true>(a, a.parity, a.mu, s, tix, warp_mask, a.sweep_ptr ? *a.sweep_ptr : a.sweep, att_total, exhausted);
    }
    if (KIND == KIND_HB) flush_kp_counters(a, att_total, exhausted);
}

// ------------------------------------------------------------------------------------------
// Cooperative whole-pass kernels (su_set_option "coop_sweep"; SURVEY.md 7 "small lattices are launch-bound"): when all
// the blocks of a sub-step fit the device at once, ONE cooperative launch runs a.coop_passes whole passes - 8 sub-steps
// each, in the order of reading R6 - with a grid barrier in place of every launch boundary. Same threads, same sites,
// same arithmetic as the plain launches (bitwise equal); neighbour links are read with ld.global.cg (L2 only), which
// needs no L1 invalidation to see what other blocks stored before the barrier. a.pass = number of the first pass;
// a.reunit applies to the last pass of the launch. Not for slab handles (no halo push in here).
// When the sub-step has at most 16 blocks (SU(2) / SU(3) 8^4: 2048 sites of one parity = 16 x 128 threads) the launcher makes
// the whole grid one thread-block cluster and the barrier is the hardware cluster barrier (barrier.cluster, release /
// acquire at cluster scope, ~0.2 us) instead of the cooperative-groups grid barrier (atomics through L2, ~2 us).
__device__ __forceinline__ void coop_barrier(const UpdateArgs& a) {
    namespace cg = cooperative_groups;
    if (a.coop_cluster) cg::this_cluster().sync();
    else cg::this_grid().sync();
}
// ------------------------------------------------------------------------------------------
template <int NC, class T, int STORE, int KIND, bool UNR, int BLOCK, int MINB, int FUSE3 = 0, bool KUNR = false>
__global__ void __launch_bounds__(BLOCK, MINB) k_update_coop(const UpdateArgs a) {
    constexpr int NSUB = NC * (NC - 1) / 2;
    constexpr int PRE_ASKED = ((KIND == KIND_HB) && UNR) ? (sizeof(T) == 4 ? SUG_KP_PRE_F32 : SUG_KP_PRE_F64) : 0;
    constexpr int PRE = (PRE_ASKED == 4 && !FUSE3) ? (sizeof(T) == 4 ? 1 : 0) : PRE_ASKED;
    __shared__ T dir_sm[PRE >= 2 ? 5 * NSUB : (PRE == 1 ? 3 * NSUB : 1)][PRE ? BLOCK : 1];
    __shared__ cx<T> s_sm[FUSE3 == 4 ? NC * NC : 1][FUSE3 == 4 ? BLOCK : 1];
    const uint32_t sweep_ctr = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
    const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = tix < a.g.Vh_int;
    const unsigned warp_mask = __ballot_sync(0xffffffffu, active);
    unsigned att_total = 0, exhausted = 0;
    UpdateArgs b = a;
#pragma unroll 1
    for (int ps = 0; ps < a.coop_passes; ++ps) {
        b.pass = a.pass + (uint32_t)ps;
        b.reunit = (a.reunit && ps == a.coop_passes - 1) ? 1 : 0;
#pragma unroll 1
        for (int sub = 0; sub < 8; ++sub) {
            if (active) {
                SiteNbr s;
                site_of_thread(a.g, tix, sub >> 2, s);
                update_link<NC, T, STORE, KIND, UNR, BLOCK, FUSE3, KUNR, LD_CG, PRE, true>(
                    b, sub >> 2, sub & 3, s, 0u, warp_mask, sweep_ctr, &dir_sm[0][PRE ? threadIdx.x : 0], att_total, exhausted,
                    &s_sm[0][FUSE3 == 4 ? threadIdx.x : 0]);
            }
            coop_barrier(a);
        }
    }
    if (KIND == KIND_HB) flush_kp_counters(a, att_total, exhausted);
}

template <class T, int KIND, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) k_update_su2_coop(const UpdateArgs a) {
    const uint32_t sweep_ctr = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
    const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = tix < a.g.Vh_int;
    const unsigned warp_mask = __ballot_sync(0xffffffffu, active);
    unsigned att_total = 0, exhausted = 0;
    UpdateArgs b = a;
#pragma unroll 1
    for (int ps = 0; ps < a.coop_passes; ++ps) {
        b.pass = a.pass + (uint32_t)ps;
        b.reunit = (a.reunit && ps == a.coop_passes - 1) ? 1 : 0;
#pragma unroll 1
        for (int sub = 0; sub < 8; ++sub) {
            if (active) {
                SiteNbr s;
                site_of_thread(a.g, tix, sub >> 2, s);
                update_link_su2<T, KIND, LD_CG, false>(b, sub >> 2, sub & 3, s, tix, warp_mask, sweep_ctr, att_total, exhausted);
            }
            coop_barrier(a);
        }
    }
    if (KIND == KIND_HB) flush_kp_counters(a, att_total, exhausted);
}

}  // namespace sug
