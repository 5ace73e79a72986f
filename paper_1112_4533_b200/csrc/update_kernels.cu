// update_kernels.cu — the staple + link-update kernel (heatbath / overrelaxation) for one
// (parity, mu) sub-step. Compiled once per colour count with -DSUG_NC=<Nc>.
//
// One thread owns one link U_mu(x), x of the given parity ("one thread per lattice
// site", :161 chessboard by direction and parity). It gathers the 18 staple links (eq 9,
// PAPER.md:83,189) from the SoA planes with coalesced 64/128-bit loads, forms W = U S^dagger
// (step 2), runs the SU(2) subgroup loop (steps 3-5) and stores the link.
//   UNR = true : matrices fully unrolled into registers (specialised SU(2)/SU(3)/SU(4))
//   UNR = false: rolled loops over local arrays (generic SU(Nc))
#include "su_internal.h"

#ifndef SUG_NC
#error "compile with -DSUG_NC=<Nc>"
#endif

namespace sug {

#define SUG_CAT_(a, b) a##b
#define SUG_CAT(a, b) SUG_CAT_(a, b)

template <int NC, class T, int STORE, int KIND, bool UNR, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) k_update(const UpdateArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    typedef Mat<NC, T, UNR> M;
    typedef cx<T> C;
    const unsigned cb = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = cb < a.g.Vh;
    unsigned att_total = 0, exhausted = 0;
    if (active) {
        const int p = a.parity, mu = a.mu;
        const unsigned Vh = a.g.Vh;
        int c[4];
        decode_cb(a.g, cb, p, c);
        const unsigned cb_pmu = cb_shift(a.g, c, mu, +1);

        C S[NC * NC], A[NC * NC], B[NC * NC], P[NC * NC];
        M::zero(S);
        const typename IO::T2* pl_mu_o = IO::plane((const void*)a.links, a.g, mu, 1 - p);
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {
            if (nu == mu) continue;
            const typename IO::T2* pl_nu_s = IO::plane((const void*)a.links, a.g, nu, p);
            const typename IO::T2* pl_nu_o = IO::plane((const void*)a.links, a.g, nu, 1 - p);
            // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
            IO::template load<true>(pl_nu_s, Vh, cb, A);
            IO::template load<true>(pl_mu_o, Vh, cb_shift(a.g, c, nu, +1), B);
            M::mul_nn(A, B, P);
            IO::template load<true>(pl_nu_o, Vh, cb_pmu, A);
            M::acc_nd(S, P, A);
            // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
            const unsigned cb_mnu = cb_shift(a.g, c, nu, -1);
            IO::template load<true>(pl_nu_o, Vh, cb_mnu, A);
            IO::template load<true>(pl_mu_o, Vh, cb_mnu, B);
            M::mul_dn(A, B, P);
            IO::template load<true>(pl_nu_s, Vh, cb_shift(a.g, c, nu, -1, mu, +1), A);
            M::acc_nn(S, P, A);
        }
        typename IO::T2* pl_self = IO::plane(a.links, a.g, mu, p);
        C* U = A;
        C* W = B;
        IO::template load<false>(pl_self, Vh, cb, U);
        M::mul_nd(U, S, W);                                   // W = U S^dagger
        update_subgroups<NC, T, KIND, UNR>(U, W, (T)a.beta, a.k0, a.k1, lex_of(a.g, c),
                                           a.sweep_ptr ? *a.sweep_ptr : a.sweep,
                                           pack_c2(0, (int)a.pass, p, mu, 0),
                                           a.attempts ? a.attempts + cb : nullptr, (size_t)Vh,
                                           att_total, exhausted);
        IO::store(pl_self, Vh, cb, U);
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

#if SUG_NC == 2
// ------------------------------------------------------------------------------------------
// SU(2) in the 4-real parameterisation U = a0 + i a.sigma (eqs 6-8): links,
// staple and update are quaternion arithmetic. Same algebra as the matrix path:
// W = U S^bar, k = |W|, u~ = W/k, a = v u~^bar (heatbath, eq 14) or (u~^bar)^2 (eq 17), U' = a U.
// ------------------------------------------------------------------------------------------
template <class T> __device__ __forceinline__ void qload(const typename V2<T>::type* __restrict__ pl, unsigned Vh, unsigned cb, T q[4], bool ro) {
    typename V2<T>::type v0 = ro ? __ldg(pl + cb) : pl[cb];
    typename V2<T>::type v1 = ro ? __ldg(pl + Vh + cb) : pl[Vh + cb];
    q[0] = v0.x; q[1] = v0.y; q[2] = v1.x; q[3] = v1.y;
}
template <class T> __device__ __forceinline__ void qconj(const T a[4], T o[4]) { o[0] = a[0]; o[1] = -a[1]; o[2] = -a[2]; o[3] = -a[3]; }

template <class T, int KIND, int BLOCK>
__global__ void __launch_bounds__(BLOCK) k_update_su2(const UpdateArgs a) {
    typedef typename V2<T>::type T2;
    const unsigned cb = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = cb < a.g.Vh;
    unsigned att_total = 0, exhausted = 0;
    if (active) {
        const int p = a.parity, mu = a.mu;
        const unsigned Vh = a.g.Vh;
        int c[4];
        decode_cb(a.g, cb, p, c);
        const unsigned cb_pmu = cb_shift(a.g, c, mu, +1);
        const T2* base = (const T2*)a.links;
        auto plane = [&](int d, int par) { return base + (size_t)(d * 2 + par) * 2 * Vh; };
        T S[4] = {0, 0, 0, 0}, A[4], B[4], Cq[4], P[4], Q[4];
        const T2* pl_mu_o = plane(mu, 1 - p);
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {
            if (nu == mu) continue;
            const T2* pl_nu_s = plane(nu, p);
            const T2* pl_nu_o = plane(nu, 1 - p);
            qload<T>(pl_nu_s, Vh, cb, A, true);
            qload<T>(pl_mu_o, Vh, cb_shift(a.g, c, nu, +1), B, true);
            qload<T>(pl_nu_o, Vh, cb_pmu, Cq, true);
            quat_mul(A, B, P); qconj(Cq, A); quat_mul(P, A, Q);
            S[0] += Q[0]; S[1] += Q[1]; S[2] += Q[2]; S[3] += Q[3];
            const unsigned cb_mnu = cb_shift(a.g, c, nu, -1);
            qload<T>(pl_nu_o, Vh, cb_mnu, A, true);
            qload<T>(pl_mu_o, Vh, cb_mnu, B, true);
            qload<T>(pl_nu_s, Vh, cb_shift(a.g, c, nu, -1, mu, +1), Cq, true);
            qconj(A, P); quat_mul(P, B, Q); quat_mul(Q, Cq, P);
            S[0] += P[0]; S[1] += P[1]; S[2] += P[2]; S[3] += P[3];
        }
        T2* pl_self = (T2*)a.links + (size_t)(mu * 2 + p) * 2 * Vh;
        T U[4], W[4], a4[4] = {1, 0, 0, 0};
        qload<T>(pl_self, Vh, cb, U, false);
        qconj(S, A);
        quat_mul(U, A, W);
        T k = Fn<T>::sqrt(W[0] * W[0] + W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
        bool ok = (k > (T)0) && Fn<T>::finite(k);
        int used = 0;
        if (ok) {
            T ud[4] = {W[0] / k, -W[1] / k, -W[2] / k, -W[3] / k};
            if (KIND == KIND_HB) {
                T v[4];
                used = kp_draw<T>((T)a.beta * k, a.k0, a.k1, lex_of(a.g, c), a.sweep_ptr ? *a.sweep_ptr : a.sweep,
                                  pack_c2(0, (int)a.pass, p, mu, 0), v);
                if (used) quat_mul(v, ud, a4); else ok = false;
            } else {
                quat_mul(ud, ud, a4);
            }
        }
        if (KIND == KIND_HB) {
            att_total = (unsigned)used;
            exhausted = ok ? 0u : 1u;
            if (a.attempts) a.attempts[cb] = (uint8_t)(used > 255 ? 255 : used);
        }
        if (ok) {
            quat_mul(a4, U, P);
            pl_self[cb] = V2<T>::make(P[0], P[1]);
            pl_self[Vh + cb] = V2<T>::make(P[2], P[3]);
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
#endif

template <int NC, class T, int STORE, bool UNR, int BLOCK, int MINB>
static cudaError_t launch_update_t(int kind, const UpdateArgs& a, cudaStream_t st) {
    const unsigned grid = (a.g.Vh + BLOCK - 1) / BLOCK;
    if (kind == KIND_HB) k_update<NC, T, STORE, KIND_HB, UNR, BLOCK, MINB><<<grid, BLOCK, 0, st>>>(a);
    else                 k_update<NC, T, STORE, KIND_OR, UNR, BLOCK, MINB><<<grid, BLOCK, 0, st>>>(a);
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
        if (f64) { if (kind == KIND_HB) k_update_su2<double, KIND_HB, BLOCK><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<double, KIND_OR, BLOCK><<<grid, BLOCK, 0, st>>>(a); }
        else     { if (kind == KIND_HB) k_update_su2<float,  KIND_HB, BLOCK><<<grid, BLOCK, 0, st>>>(a); else k_update_su2<float,  KIND_OR, BLOCK><<<grid, BLOCK, 0, st>>>(a); }
        return cudaGetLastError();
    }
    return f64 ? launch_update_t<NC, double, STORE_QUAT, false, 64, 1>(kind, a, st)
               : launch_update_t<NC, float,  STORE_QUAT, false, 64, 1>(kind, a, st);
#elif SUG_NC == 3
    if (!v.generic) {
        if (v.store == STORE_RECON12)
            return f64 ? launch_update_t<NC, double, STORE_RECON12, true, 128, 1>(kind, a, st)
                       : launch_update_t<NC, float,  STORE_RECON12, true, 128, 1>(kind, a, st);
        return f64 ? launch_update_t<NC, double, STORE_FULL, true, 128, 1>(kind, a, st)
                   : launch_update_t<NC, float,  STORE_FULL, true, 128, 1>(kind, a, st);
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
