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
#include "su_device.cuh"

namespace sug {

#ifndef SUG_TMINUS_STREAM
#define SUG_TMINUS_STREAM 1
#endif
#ifndef SUG_KP_PREDIR
#define SUG_KP_PREDIR 1
#endif

struct UpdateArgs {
    void* links;
    Geom g;
    int parity, mu;
    double beta;
    uint32_t k0, k1, sweep, pass;
    const uint32_t* sweep_ptr;         // device; when non-NULL the sweep counter is read from here (graph replay)
    uint8_t* attempts;                 // device, [n_sub][Vh] or NULL
    unsigned long long* counters;      // device, {kp_attempts_total, kp_exhausted}
    // slab mode: link buffers of the slabs below / above in t (peer memory over NVLink, or this device). The
    // kernel that updates a link of the first / last owned slice also stores it into that neighbour's halo.
    void* peer_lo;
    void* peer_hi;
};

// checkerboard index, in the neighbour's buffer, of the halo copy of an edge site (all slabs have Lt_int slices)
__device__ __forceinline__ unsigned halo_cb_lo(const Geom& g, unsigned cb) { return cb + (unsigned)g.Lt_int * g.Vsh; }   // -> their upper halo
__device__ __forceinline__ unsigned halo_cb_hi(const Geom& g, unsigned cb) { return cb - (unsigned)g.Lt_int * g.Vsh; }   // -> their lower halo

// The site a thread works on and the checkerboard-index offsets of its 8 neighbours.
struct SiteNbr {
    unsigned cb;        // checkerboard index of x in the stored lattice
    uint32_t lex;       // lexicographic index of x in the global lattice (RNG counter word c0)
    int dp[4], dm[4];   // cb(x + e_d) - cb(x), cb(x - e_d) - cb(x)   (periodic)
};

__device__ __forceinline__ int sel4(int i, int v0, int v1, int v2, int v3) {
    return i == 0 ? v0 : (i == 1 ? v1 : (i == 2 ? v2 : v3));
}

// traversal index (over the OWNED sites of one parity) -> site; all indices stay in registers
__device__ __forceinline__ void site_of_thread(const Geom& g, unsigned tix, int parity, SiteNbr& s) {
    const unsigned row = (unsigned)g.Lxh, pl = row * (unsigned)g.L[1];
    const unsigned grp = pl * (unsigned)g.Zc, span = grp * (unsigned)g.Lt_int;
    const unsigned zc = tix / span;  unsigned r = tix - zc * span;
    const unsigned ti = r / grp;     r -= ti * grp;
    const unsigned zi = r / pl;      r -= zi * pl;
    const unsigned y = r / row;
    const unsigned xh = r - y * row;
    const unsigned z = zc * (unsigned)g.Zc + zi;
    const unsigned t = ti + (unsigned)g.t_halo;                          // stored time slice
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
}

// slab mode: 1 = the thread's site lies in the first owned time slice, 2 = in the last one, 0 otherwise.
// Recomputed from the traversal index at store time so that nothing stays live across the kernel body.
__device__ __forceinline__ int slab_edge(const Geom& g, unsigned tix) {
    if (!g.t_halo) return 0;
    const unsigned grp = (unsigned)g.Lxh * (unsigned)g.L[1] * (unsigned)g.Zc, span = grp * (unsigned)g.Lt_int;
    const unsigned ti = (tix % span) / grp;
    return (ti == 0 ? 1 : 0) | ((int)ti + 1 == g.Lt_int ? 2 : 0);
}

// FUSE3: each staple term S += A B C (three links) is evaluated row by row with all three operands
// loaded up front (Mat::acc_nnd / acc_dnn): half as many load-wait phases per thread as the
// two-step form (P = A B; S += P C), for the same registers. KUNR: unroll the loop over nu.
template <int NC, class T, int STORE, int KIND, bool UNR, int BLOCK, int MINB, bool FUSE3 = false, bool KUNR = false>
__global__ void __launch_bounds__(BLOCK, MINB) k_update(const UpdateArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    typedef Mat<NC, T, UNR> M;
    typedef cx<T> C;
    const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = tix < a.g.Vh_int;
    const unsigned warp_mask = __ballot_sync(0xffffffffu, active);      // lanes that run the body (ragged last warp)
    unsigned att_total = 0, exhausted = 0;
    if (active) {
        const int p = a.parity, mu = a.mu;
        SiteNbr s;
        site_of_thread(a.g, tix, p, s);
        const unsigned cb = s.cb;
        const int dpmu = sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);

        // heatbath, register kernels: the directions of all subgroup draws are link-independent; evaluate them
        // now, in the shadow of the first loads, and park them in shared memory (one private column per thread)
        constexpr int NSUB = NC * (NC - 1) / 2;
        constexpr bool PREDIR = (KIND == KIND_HB) && UNR && SUG_KP_PREDIR && sizeof(T) == 4;   // fp32 only: measured -2.7 % (fp64: +5 %)
        __shared__ T dir_sm[PREDIR ? 3 * NSUB : 1][PREDIR ? BLOCK : 1];
        const uint32_t sweep_ctr = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
        if (PREDIR) {
#pragma unroll
            for (int q = 0; q < NSUB; ++q) {
                T n[3];
                kp_direction<T>(a.k0, a.k1, s.lex, sweep_ctr, pack_c2((int)a.pass, p, mu, q), n);
                dir_sm[3 * q][threadIdx.x] = n[0]; dir_sm[3 * q + 1][threadIdx.x] = n[1]; dir_sm[3 * q + 2][threadIdx.x] = n[2];
            }
        }

        C S[NC * NC], A[NC * NC], B[NC * NC], P[NC * NC];
        M::zero(S);
        const typename IO::T2* pl_mu_o = IO::plane((const void*)a.links, a.g, mu, 1 - p);
#pragma unroll(KUNR ? 3 : 1)
        for (int k = 0; k < 3; ++k) {
            const int nu = k + (k >= mu ? 1 : 0);
            const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
            const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
            const typename IO::T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
            const typename IO::T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
            if (FUSE3) {
                // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
                IO::template load<LD_RO>(pl_mu_o, cb + (unsigned)dpnu, B);
                IO::template load<LD_RO>(pl_nu_o, cb + (unsigned)dpmu, P);
                IO::template load<LD_RO>(pl_nu_s, cb, A);
                M::acc_nnd(S, A, B, P);
                // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
                if (SUG_TMINUS_STREAM && k == 2 && nu == 3) {
                    // links of the time slice below: with the traversal walking up in t this is their last
                    // use in the sub-step, so they are fetched evict-first and leave L2 to the slices ahead
                    IO::template load<LD_STREAM>(pl_mu_o, cb + (unsigned)dmnu, B);
                    IO::template load<LD_STREAM>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                    IO::template load<LD_STREAM>(pl_nu_o, cb + (unsigned)dmnu, A);
                } else {
                    IO::template load<LD_RO>(pl_mu_o, cb + (unsigned)dmnu, B);
                    IO::template load<LD_RO>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), P);
                    IO::template load<LD_RO>(pl_nu_o, cb + (unsigned)dmnu, A);
                }
                M::acc_dnn(S, A, B, P);
            } else {
                // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
                IO::template load<LD_RO>(pl_nu_s, cb, A);
                IO::template load<LD_RO>(pl_mu_o, cb + (unsigned)dpnu, B);
                M::mul_nn(A, B, P);
                IO::template load<LD_RO>(pl_nu_o, cb + (unsigned)dpmu, A);
                M::acc_nd(S, P, A);
                // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
                IO::template load<LD_RO>(pl_nu_o, cb + (unsigned)dmnu, A);
                IO::template load<LD_RO>(pl_mu_o, cb + (unsigned)dmnu, B);
                M::mul_dn(A, B, P);
                IO::template load<LD_RO>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), A);
                M::acc_nn(S, P, A);
            }
        }
        typename IO::T2* pl_self = IO::plane(a.links, a.g, mu, p);
        C* U = A;
        C* W = B;
        IO::template load<LD_STREAM>(pl_self, cb, U);
        M::mul_nd(U, S, W);                                   // W = U S^dagger
        update_subgroups<NC, T, KIND, UNR>(U, W, (T)a.beta, a.k0, a.k1, s.lex, sweep_ctr,
                                           pack_c2((int)a.pass, p, mu, 0),
                                           a.attempts ? a.attempts + cb : nullptr, (size_t)a.g.Vh,
                                           att_total, exhausted, warp_mask,
                                           PREDIR ? &dir_sm[0][threadIdx.x] : nullptr, PREDIR ? BLOCK : 0);
        IO::template store<true>(pl_self, cb, U);
        if (const int edge = slab_edge(a.g, tix)) {          // fused halo push (slab mode only)
            if (edge & 1) IO::template store<true>(IO::plane(a.peer_lo, a.g, mu, p), halo_cb_lo(a.g, cb), U);
            if (edge & 2) IO::template store<true>(IO::plane(a.peer_hi, a.g, mu, p), halo_cb_hi(a.g, cb), U);
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

template <class T, int KIND, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) k_update_su2(const UpdateArgs a) {
    typedef typename V2<T>::type T2;
    const unsigned tix = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = tix < a.g.Vh_int;
    const unsigned warp_mask = __ballot_sync(0xffffffffu, active);
    unsigned att_total = 0, exhausted = 0;
    if (active) {
        const int p = a.parity, mu = a.mu;
        SiteNbr s;
        site_of_thread(a.g, tix, p, s);
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
            qload<T, LD_RO>(pl_nu_s, cb, A);
            qload<T, LD_RO>(pl_mu_o, cb + (unsigned)dpnu, B);
            qload<T, LD_RO>(pl_nu_o, cb + (unsigned)dpmu, Cq);
            quat_mul(A, B, P); qconj(Cq, A); quat_mul(P, A, Q);
            S[0] += Q[0]; S[1] += Q[1]; S[2] += Q[2]; S[3] += Q[3];
            qload<T, LD_RO>(pl_nu_o, cb + (unsigned)dmnu, A);
            qload<T, LD_RO>(pl_mu_o, cb + (unsigned)dmnu, B);
            qload<T, LD_RO>(pl_nu_s, cb + (unsigned)(dmnu + dpmu), Cq);
            qconj(A, P); quat_mul(P, B, Q); quat_mul(Q, Cq, P);
            S[0] += P[0]; S[1] += P[1]; S[2] += P[2]; S[3] += P[3];
        }
        T2* pl_self = (T2*)a.links + (size_t)(mu * 2 + p) * 2 * a.g.Vhp;
        T U[4], W[4], a4[4] = {1, 0, 0, 0};
        qload<T, LD_STREAM>(pl_self, cb, U);
        qconj(S, A);
        quat_mul(U, A, W);
        const T n2 = W[0] * W[0] + W[1] * W[1] + W[2] * W[2] + W[3] * W[3];      // k^2
        bool ok = (n2 > (T)0) && Fn<T>::finite(n2);
        int used = 0;
        const unsigned draw_mask = (KIND == KIND_HB) ? __ballot_sync(warp_mask, ok) : 0u;
        if (ok) {
            if (KIND == KIND_HB) {
                const T ik = Fn<T>::rsqrt(n2), k = n2 * ik;
                T ud[4] = {W[0] * ik, -W[1] * ik, -W[2] * ik, -W[3] * ik};
                T v[4];
                used = kp_draw<T>(draw_mask, (T)a.beta * k, (T)-0.5 / (T)a.beta * ik, a.k0, a.k1, s.lex, a.sweep_ptr ? *a.sweep_ptr : a.sweep,
                                  pack_c2((int)a.pass, p, mu, 0), v);
                if (used) quat_mul(v, ud, a4); else ok = false;
            } else {
                // a = conj(W)^2 / k^2 (eq 17)
                const T in2 = (T)1 / n2, m2w0 = (T)-2 * W[0] * in2;
                a4[0] = (W[0] * W[0] - (W[1] * W[1] + W[2] * W[2] + W[3] * W[3])) * in2;
                a4[1] = m2w0 * W[1]; a4[2] = m2w0 * W[2]; a4[3] = m2w0 * W[3];
            }
        }
        if (KIND == KIND_HB) {
            att_total = (unsigned)used;
            exhausted = ok ? 0u : 1u;
            if (a.attempts) a.attempts[cb] = (uint8_t)(used > 255 ? 255 : used);
        }
        if (ok) {
            quat_mul(a4, U, P);
            T2* q = pl_self + qsite<T>(cb);
            stg2<T, true>(q, V2<T>::make(P[0], P[1]));
            stg2<T, true>(q + LINK_TILE, V2<T>::make(P[2], P[3]));
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

}  // namespace sug
