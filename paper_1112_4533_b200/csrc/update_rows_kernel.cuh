// update_rows_kernel.cuh — the GENERIC SU(Nc) staple + link-update kernel:
// any Nc, nothing specialised per group, full Nc x Nc storage.
//
// The paper's generic kernel gives one thread a whole link and keeps its Nc x Nc matrices in local
// memory; its cost explodes with Nc ("SU(6) ~ 10x optimised SU(3)"). Here a link is
// updated by a group of Nc lanes of one warp, lane r owning ROW r of every matrix in registers:
//   staple term  S_r += (A_r . B) . C^dagger         A_r in registers, B and C staged in shared memory
//                S_r += (A^dagger B)_r . C           A, B, C staged in shared memory
//   W_r = U_r . S^dagger                             S staged in shared memory
//   subgroup (i,j): lanes i and j exchange the four entries of the 2x2 block and their rows by warp
//                   shuffle, both evaluate the projection and the Kennedy-Pendleton draw (same counter
//                   -> same numbers) and rotate their own row (eq 15); subgroups on disjoint row pairs
//                   commute exactly, so the lexicographic sequence runs as a wavefront of 2 Nc - 3 slots.
// A warp holds floor(32 / Nc) links; left-over lanes shadow the last group and never store.
// The order of operations inside every sum is the one of update_kernel.cuh (products left to right).
#pragma once
#include "update_kernel.cuh"

namespace sug {

#ifndef SUG_ROWS_MINB
#define SUG_ROWS_MINB 4
#endif
#ifndef SUG_ROWS_MAXW
#define SUG_ROWS_MAXW 4
#endif

template <int NC> struct RowsCfg {
    static constexpr int LPW = 32 / NC;                       // links per warp
    // Row pitch of a staged matrix in complex elements. With pitch 8 (128 B in fp64) all rows of a matrix start in the same
    // bank and the Nc lanes of a link, which store / read one element of Nc different rows per instruction, serialise: pitch 9
    // (SU(8) 16^4 fp64 iteration 8.71 -> 7.70 ms). For the other Nc an odd pitch was measured too and lost (SU(6): the larger
    // matrices leave 2 instead of 3 warps per block, OR 0.160 -> 0.169 ms; SU(4): 0.216 -> 0.223 ms): profiles/r02g section 13.
    static constexpr int PITCH = NC + (NC % 8 == 0 ? 1 : 0);
    static constexpr int STRIDE = NC * PITCH + 1;             // complex elements per staged matrix (+1: bank spread between links)
    static constexpr int NBUF = 5;                            // upper term: B, C; lower term: A, B, C
    static constexpr size_t bytes(int w, size_t real, int nbuf) { return (size_t)w * LPW * nbuf * STRIDE * 2 * real; }
};
// warps per block: as many (<= 4) as keep NB staged matrices per link within 48 KB of static shared memory
template <int NC, class T, int NB = RowsCfg<NC>::NBUF> struct RowsWarps {
    static constexpr size_t LIM = 48 * 1024, R = sizeof(T);
    static constexpr int fit = RowsCfg<NC>::bytes(4, R, NB) <= LIM ? 4 : (RowsCfg<NC>::bytes(3, R, NB) <= LIM ? 3 : (RowsCfg<NC>::bytes(2, R, NB) <= LIM ? 2 : 1));
    static constexpr int value = fit < SUG_ROWS_MAXW ? fit : SUG_ROWS_MAXW;
};

template <class T> __device__ __forceinline__ cx<T> shfl_cx(cx<T> v, int src) {
    return mk<T>(__shfl_sync(0xffffffffu, v.re, src), __shfl_sync(0xffffffffu, v.im, src));
}
// element `idx` of a register-resident row without dynamic indexing
template <int NC, class T> __device__ __forceinline__ cx<T> row_pick(const cx<T>* row, int idx) {
    cx<T> v = row[0];
#pragma unroll
    for (int c = 1; c < NC; ++c) if (idx == c) v = row[c];
    return v;
}

// resident blocks per SM asked of the compiler: 16 warps with 4-warp blocks, else 12 warps (as many as the registers of a
// 168-register kernel allow), whatever the number of warps the staging buffers leave per block
template <int NC, class T> struct RowsMinBlocks {
    static constexpr int W = RowsWarps<NC, T>::value;
    static constexpr int value = W == 4 ? SUG_ROWS_MINB : (W == 3 ? 4 : (W == 2 ? 6 : 8));
};

template <int NC, class T, int KIND>
__global__ void __launch_bounds__(32 * RowsWarps<NC, T>::value, RowsMinBlocks<NC, T>::value) k_update_rows(const UpdateArgs a) {
    typedef RowsCfg<NC> Cfg;
    typedef LinkIO<NC, T, STORE_FULL, true> IO;
    typedef typename IO::T2 T2;
    typedef cx<T> C;
    constexpr int WARPS = RowsWarps<NC, T>::value;
    constexpr int LPW = Cfg::LPW, STRIDE = Cfg::STRIDE, PT = Cfg::PITCH;
    __shared__ C stage[WARPS * LPW][Cfg::NBUF][STRIDE];

    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    const bool shadow = lane >= LPW * NC;                     // left-over lanes repeat the last group's work
    const int g = shadow ? LPW - 1 : lane / NC;               // link slot in the warp
    const int r = shadow ? lane - LPW * NC : lane - g * NC;   // row owned by this lane
    const int gbase = g * NC;                                 // first lane of the group
    unsigned tix = (blockIdx.x * WARPS + (unsigned)warp) * LPW + (unsigned)g;
    const bool owner = !shadow && tix < a.g.Vh_int;           // lanes past the end redo the last link, never store
    if (tix >= a.g.Vh_int) tix = a.g.Vh_int - 1;
    C(*M)[STRIDE] = stage[warp * LPW + g];

    const int p = a.parity, mu = a.mu;
    SiteNbr s;
    site_of_thread(a.g, tix, p, s);
    const unsigned cb = s.cb;
    const int dpmu = sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);

    // row r of a link straight from the tiled SoA plane
    auto load_row = [&](const T2* pl, unsigned site, C* row) {
        const T2* q = IO::site(pl, site) + (size_t)r * NC * LINK_TILE;
#pragma unroll
        for (int c = 0; c < NC; ++c) { T2 v = __ldg(q + c * LINK_TILE); row[c] = mk<T>(v.x, v.y); }
    };
    auto stage_row = [&](int buf, const C* row) {
#pragma unroll
        for (int c = 0; c < NC; ++c) M[buf][r * PT + c] = row[c];
    };

    C S[NC], A[NC], B[NC], D[NC], P[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) S[c] = mk<T>(0, 0);
    const T2* pl_mu_o = IO::plane((const void*)a.links, a.g, mu, 1 - p);
#pragma unroll 1
    for (int k = 0; k < 3; ++k) {
        const int nu = k + (k >= mu ? 1 : 0);
        const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
        const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
        const T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
        const T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
        // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
        load_row(pl_nu_s, cb, A);
        load_row(pl_mu_o, cb + (unsigned)dpnu, B);
        load_row(pl_nu_o, cb + (unsigned)dpmu, D);
        stage_row(0, B);
        stage_row(1, D);
        __syncwarp();
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            C acc = mk<T>(0, 0);
#pragma unroll
            for (int q = 0; q < NC; ++q) mad(acc, A[q], M[0][q * PT + j]);
            P[j] = acc;
        }
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            C acc = S[j];
#pragma unroll
            for (int q = 0; q < NC; ++q) mad_cb(acc, P[q], M[1][j * PT + q]);
            S[j] = acc;
        }
        // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
        load_row(pl_nu_o, cb + (unsigned)dmnu, A);
        load_row(pl_mu_o, cb + (unsigned)dmnu, B);
        load_row(pl_nu_s, cb + (unsigned)(dmnu + dpmu), D);
        stage_row(2, A);
        stage_row(3, B);
        stage_row(4, D);
        __syncwarp();           // also orders the upper term's reads of buffers 0, 1 before their next writes
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            C acc = mk<T>(0, 0);
#pragma unroll
            for (int q = 0; q < NC; ++q) mad_ca(acc, M[2][q * PT + r], M[3][q * PT + j]);
            P[j] = acc;
        }
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            C acc = S[j];
#pragma unroll
            for (int q = 0; q < NC; ++q) mad(acc, P[q], M[4][q * PT + j]);
            S[j] = acc;
        }
    }
    // W = U S^dagger (step 2)
    T2* pl_self = IO::plane(a.links, a.g, mu, p);
    C U[NC], W[NC];
    {
        const T2* q = IO::site((const T2*)pl_self, cb) + (size_t)r * NC * LINK_TILE;
#pragma unroll
        for (int c = 0; c < NC; ++c) { T2 v = __ldcs(q + c * LINK_TILE); U[c] = mk<T>(v.x, v.y); }
    }
    stage_row(0, S);            // buffer 0 was last read before the previous barrier
    __syncwarp();
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        C acc = mk<T>(0, 0);
#pragma unroll
        for (int q = 0; q < NC; ++q) mad_cb(acc, U[q], M[0][j * PT + q]);
        W[j] = acc;
    }

    // steps 3-5: every SU(2) subgroup (i<j), lexicographic (reading R5)
    const T beta = (T)a.beta;
    const T two_beta_over_nc = (T)2 * beta / (T)NC;
    const T m_nc_over_4beta = (T)-0.25 * (T)NC / beta;
    const uint32_t c1 = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
    const uint32_t c2_base = pack_c2((int)a.pass, p, mu, 0);
    unsigned att_total = 0, exhausted = 0;
    // Wavefront over the lexicographic subgroup order: step (i,j) only depends on earlier steps that touched
    // row i or row j, and steps on disjoint row pairs commute exactly (A_ij is built from rows i,j of W and
    // rotates rows i,j only). All pairs with i + j = t + 1 are disjoint and have all their predecessors in
    // earlier slots, so slot t runs them at once: 2 Nc - 3 slots instead of Nc (Nc - 1) / 2 steps, every lane
    // busy in most of them, with the result of the sequential order (the reordered steps commute exactly).
#pragma unroll 1
    for (int t = 0; t <= 2 * NC - 4; ++t) {
        const int sidx = t + 1 - r;
        const bool paired = sidx >= 0 && sidx < NC && sidx != r;
        const int pr = paired ? sidx : r;                       // partner row (self when idle in this slot)
        const bool is_i = r < pr;
        const int i = is_i ? r : pr, j = is_i ? pr : r;
        const int sub = i * NC - (i * (i + 1)) / 2 + (j - i - 1);   // lexicographic index of (i,j)
        const C wd = row_pick<NC, T>(W, r), wo = row_pick<NC, T>(W, pr);       // W_rr, W_r,pr
        const C pd = shfl_cx(wd, gbase + pr), po = shfl_cx(wo, gbase + pr);     // W_pr,pr, W_pr,r
        const C wii = is_i ? wd : pd, wij = is_i ? wo : po, wji = is_i ? po : wo, wjj = is_i ? pd : wd;
        T r0 = (T)0.5 * (wii.re + wjj.re), r1 = (T)0.5 * (wij.im + wji.im);
        T r2 = (T)0.5 * (wij.re - wji.re), r3 = (T)0.5 * (wii.im - wjj.im);
        const T n2 = r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3;
        bool ok = paired && (n2 >= Fn<T>::min_norm2()) && Fn<T>::finite(n2);      // as in update_subgroups
        T q4[4] = {(T)1, (T)0, (T)0, (T)0};
        int used = 0;
        const unsigned draw_mask = (KIND == KIND_HB) ? __ballot_sync(0xffffffffu, ok) : 0u;   // all 32 lanes are here
        if (ok) {
            if (KIND == KIND_HB) {
                const T ik = Fn<T>::rsqrt_pos(n2), kk = n2 * ik;
                T ud[4] = {r0 * ik, -r1 * ik, -r2 * ik, -r3 * ik};
                T v[4];
                used = kp_draw<T>(draw_mask, two_beta_over_nc * kk, m_nc_over_4beta * ik, a.k0, a.k1, s.lex, c1,
                                  c2_base | (uint32_t)sub, v);
                if (used) quat_mul(v, ud, q4); else ok = false;
            } else {
                const T in2 = Fn<T>::rcp_pos(n2), m2r0 = (T)-2 * r0 * in2;
                q4[0] = (r0 * r0 - (r1 * r1 + r2 * r2 + r3 * r3)) * in2;
                q4[1] = m2r0 * r1; q4[2] = m2r0 * r2; q4[3] = m2r0 * r3;
            }
        }
        if (KIND == KIND_HB && owner && paired && is_i) {        // lane i of the pair keeps the books
            att_total += (unsigned)used;
            if (!ok) exhausted += 1u;
            if (a.attempts) a.attempts[(size_t)sub * a.g.Vh + cb] = (uint8_t)(used > 255 ? 255 : used);
        }
        // rows i and j <- a . rows (eq 15): lane i: a00 own + a01 other ; lane j: a10 other + a11 own
        const C c_own = is_i ? mk<T>(q4[0], q4[3]) : mk<T>(q4[0], -q4[3]);
        const C c_oth = is_i ? mk<T>(q4[2], q4[1]) : mk<T>(-q4[2], q4[1]);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const C ou = shfl_cx(U[c], gbase + pr), ow = shfl_cx(W[c], gbase + pr);
            if (ok) {
                U[c] = is_i ? (c_own * U[c] + c_oth * ou) : (c_oth * ou + c_own * U[c]);
                W[c] = is_i ? (c_own * W[c] + c_oth * ow) : (c_oth * ow + c_own * W[c]);
            }
        }
    }
    if (owner) {
        T2* q = IO::site(pl_self, cb) + (size_t)r * NC * LINK_TILE;
#pragma unroll
        for (int c = 0; c < NC; ++c) __stcs(q + c * LINK_TILE, V2<T>::make(U[c].re, U[c].im));
        if (const int edge = slab_edge(a.g, tix)) {          // fused halo push (slab mode only)
            if (edge & 1) {
                T2* h = IO::site(IO::plane(a.peer_lo, a.g, mu, p), halo_cb_lo(a.g, cb)) + (size_t)r * NC * LINK_TILE;
#pragma unroll
                for (int c = 0; c < NC; ++c) __stcs(h + c * LINK_TILE, V2<T>::make(U[c].re, U[c].im));
            }
            if (edge & 2) {
                T2* h = IO::site(IO::plane(a.peer_hi, a.g, mu, p), halo_cb_hi(a.g, cb)) + (size_t)r * NC * LINK_TILE;
#pragma unroll
                for (int c = 0; c < NC; ++c) __stcs(h + c * LINK_TILE, V2<T>::make(U[c].re, U[c].im));
            }
        }
    }
    if (KIND == KIND_HB) {
        for (int o = 16; o > 0; o >>= 1) {
            att_total += __shfl_down_sync(0xffffffffu, att_total, o);
            exhausted += __shfl_down_sync(0xffffffffu, exhausted, o);
        }
        if (lane == 0) {
            if (att_total) atomicAdd(a.counters, (unsigned long long)att_total);
            if (exhausted) atomicAdd(a.counters + 1, (unsigned long long)exhausted);
        }
    }
}

template <int NC, class T>
static cudaError_t launch_update_rows(int kind, const UpdateArgs& a, cudaStream_t st) {
    constexpr int WARPS = RowsWarps<NC, T>::value;
    const unsigned per_block = (unsigned)(WARPS * RowsCfg<NC>::LPW);
    const unsigned grid = (a.g.Vh_int + per_block - 1) / per_block;
    if (kind == KIND_HB) k_update_rows<NC, T, KIND_HB><<<grid, 32 * WARPS, 0, st>>>(a);
    else                 k_update_rows<NC, T, KIND_OR><<<grid, 32 * WARPS, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace sug
