// aux_kernels.cu — everything on the path except the link update: plaquette and Polyakov-loop
// reductions (fp64 accumulation, warp shuffle + block + final pass), reunitarisation, cold / hot
// start, and the tiled-SoA <-> canonical-layout conversion used by export / import.
// Compiled once per colour count with -DSUG_NC=<Nc>.
#include "su_internal.h"
#include "update_rows_kernel.cuh"

#ifndef SUG_NC
#error "compile with -DSUG_NC=<Nc>"
#endif

namespace sug {

#define SUG_CAT_(a, b) a##b
#define SUG_CAT(a, b) SUG_CAT_(a, b)

// ------------------------------------------------------------------------------------------
// Plaquette (eq 4): per site the six P_mu,nu; Re Tr P = Re Tr[(U_mu(x) U_nu(x+mu))
// (U_nu(x) U_mu(x+nu))^dagger]. Products in T, site sum and reduction in double.
// ------------------------------------------------------------------------------------------
#ifndef SUG_PLAQ_BOTH_PARITIES
#define SUG_PLAQ_BOTH_PARITIES 1
#endif
// Thread -> site: blocks alternate between the two parities of the same lattice region and walk it in the
// update kernel's z-chunked order (site_of_thread), so a link is fetched from DRAM once: it is read as
// "own" link by its site and as forward neighbour by three sites of the other parity in the same or the
// next chunk, all while it is still in L2.
template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(PLAQ_BLOCK, (sizeof(T) == 8 ? PLAQ_MINB_F64 : PLAQ_MINB_F32)) k_plaquette(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    typedef Mat<NC, T, UNR> M;
    typedef cx<T> C;
#if SUG_PLAQ_BOTH_PARITIES
    // one block = both parities of PLAQ_BLOCK / 2 consecutive sites: a site's forward neighbours in x and y are own
    // links of the other half of the block, so they are found in L1
    const int p = (int)(threadIdx.x / (PLAQ_BLOCK / 2));
    const unsigned tix = blockIdx.x * (PLAQ_BLOCK / 2) + (threadIdx.x % (PLAQ_BLOCK / 2));
#else
    const int p = (int)(blockIdx.x & 1u);
    const unsigned tix = (blockIdx.x >> 1) * PLAQ_BLOCK + threadIdx.x;
#endif
    double acc = 0.0;
    if (tix < a.g.Vh_int) {
        SiteNbr s;
        site_of_thread(a.g, tix, p, s);
        const unsigned cb = s.cb;
        if (UNR && NC <= 3) {
            // the site's four links stay in registers; each of the 6 plaquettes adds two neighbour loads
            C Uo[4][NC * NC], B[NC * NC], D[NC * NC], P[NC * NC], Q[NC * NC];
#pragma unroll
            for (int d = 0; d < 4; ++d) IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, d, p), cb, Uo[d]);
#pragma unroll
            for (int mu = 0; mu < 3; ++mu)
#pragma unroll
                for (int nu = mu + 1; nu < 4; ++nu) {
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, nu, 1 - p), cb + (unsigned)s.dp[mu], B);
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, mu, 1 - p), cb + (unsigned)s.dp[nu], D);
                    M::mul_nn(Uo[mu], B, P);
                    M::mul_nn(Uo[nu], D, Q);
                    acc += (double)M::retr_nd(P, Q);
                }
        } else {
            // Nc >= 4: four resident links would not fit the register file; two loads per product instead
            C A[NC * NC], B[NC * NC], P[NC * NC], Q[NC * NC];
#pragma unroll 1
            for (int mu = 0; mu < 3; ++mu)
#pragma unroll 1
                for (int nu = mu + 1; nu < 4; ++nu) {
                    const unsigned fmu = cb + (unsigned)sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
                    const unsigned fnu = cb + (unsigned)sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, mu, p), cb, A);
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, nu, 1 - p), fmu, B);
                    M::mul_nn(A, B, P);
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, nu, p), cb, A);
                    IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, mu, 1 - p), fnu, B);
                    M::mul_nn(A, B, Q);
                    acc += (double)M::retr_nd(P, Q);
                }
        }
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) a.partials[blockIdx.x] = acc;
}

// Polyakov loop (reading R9): per spatial site Tr prod_t U_3(x,t); complex, double accumulation.
template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(REDUCE_BLOCK) k_polyakov(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    typedef Mat<NC, T, UNR> M;
    typedef cx<T> C;
    const unsigned Vs = (unsigned)a.g.L[0] * a.g.L[1] * a.g.L[2];
    const unsigned xs = blockIdx.x * REDUCE_BLOCK + threadIdx.x;
    double re = 0.0, im = 0.0;
    if (xs < Vs) {
        const int x = (int)(xs % (unsigned)a.g.L[0]);
        const int y = (int)((xs / (unsigned)a.g.L[0]) % (unsigned)a.g.L[1]);
        const int z = (int)(xs / ((unsigned)a.g.L[0] * a.g.L[1]));
        C P[NC * NC], A[NC * NC], Q[NC * NC];
        IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, 3, site_parity(a.g, x, y, z, 0)), cb_of(a.g, x, y, z, 0), P);
#pragma unroll 1
        for (int t = 1; t < a.g.L[3]; ++t) {
            IO::template load<LD_RO>(IO::plane((const void*)a.links, a.g, 3, site_parity(a.g, x, y, z, t)), cb_of(a.g, x, y, z, t), A);
            M::mul_nn(P, A, Q);
#pragma unroll(UNR ? NC * NC : 1)
            for (int e = 0; e < NC * NC; ++e) P[e] = Q[e];
        }
#pragma unroll(UNR ? NC : 1)
        for (int d = 0; d < NC; ++d) { re += (double)P[d * NC + d].re; im += (double)P[d * NC + d].im; }
    }
    re = block_sum(re);
    im = block_sum(im);
    if (threadIdx.x == 0) { a.partials[blockIdx.x] = re; a.partials[gridDim.x + blockIdx.x] = im; }
}

// ------------------------------------------------------------------------------------------
// Row-per-lane forms of the two reductions for the generic SU(Nc) path (same decomposition as
// update_rows_kernel.cuh): Nc lanes per site, lane r owns row r, the right-hand operands are
// staged in shared memory (double-buffered: one __syncwarp per product pair).
// ------------------------------------------------------------------------------------------
template <int NC, class T>
__global__ void __launch_bounds__(32 * RowsWarps<NC, T, 4>::value) k_plaquette_rows(const AuxArgs a) {
    typedef RowsCfg<NC> Cfg;
    typedef LinkIO<NC, T, STORE_FULL, true> IO;
    typedef typename IO::T2 T2;
    typedef cx<T> C;
    constexpr int WARPS = RowsWarps<NC, T, 4>::value, LPW = Cfg::LPW, STRIDE = Cfg::STRIDE;
    __shared__ C stage[WARPS * LPW][4][STRIDE];
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    const bool shadow = lane >= LPW * NC;
    const int g = shadow ? LPW - 1 : lane / NC;
    const int r = shadow ? lane - LPW * NC : lane - g * NC;
    const int p = (int)(blockIdx.x & 1u);
    unsigned tix = ((blockIdx.x >> 1) * WARPS + (unsigned)warp) * LPW + (unsigned)g;
    const bool owner = !shadow && tix < a.g.Vh_int;
    if (tix >= a.g.Vh_int) tix = a.g.Vh_int - 1;
    C(*M)[STRIDE] = stage[warp * LPW + g];
    SiteNbr s;
    site_of_thread(a.g, tix, p, s);
    const unsigned cb = s.cb;
    auto load_row = [&](int d, int par, unsigned site, C* row) {
        const T2* q = IO::site(IO::plane((const void*)a.links, a.g, d, par), site) + (size_t)r * NC * LINK_TILE;
#pragma unroll
        for (int c = 0; c < NC; ++c) { T2 v = __ldg(q + c * LINK_TILE); row[c] = mk<T>(v.x, v.y); }
    };
    C Uo[4][NC];
#pragma unroll
    for (int d = 0; d < 4; ++d) load_row(d, p, cb, Uo[d]);
    double acc = 0.0;
    int pair = 0;
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
        for (int nu = mu + 1; nu < 4; ++nu, ++pair) {
            const int b0 = (pair & 1) * 2;
            C B[NC], D[NC];
            load_row(nu, 1 - p, cb + (unsigned)s.dp[mu], B);
            load_row(mu, 1 - p, cb + (unsigned)s.dp[nu], D);
#pragma unroll
            for (int c = 0; c < NC; ++c) { M[b0][r * NC + c] = B[c]; M[b0 + 1][r * NC + c] = D[c]; }
            __syncwarp();
            T t = 0;
#pragma unroll
            for (int j = 0; j < NC; ++j) {
                C pj = mk<T>(0, 0), qj = mk<T>(0, 0);
#pragma unroll
                for (int q = 0; q < NC; ++q) { mad(pj, Uo[mu][q], M[b0][q * NC + j]); mad(qj, Uo[nu][q], M[b0 + 1][q * NC + j]); }
                t += pj.re * qj.re + pj.im * qj.im;
            }
            if (owner) acc += (double)t;
        }
    acc = block_sum(acc);
    if (threadIdx.x == 0) a.partials[blockIdx.x] = acc;
}

template <int NC, class T>
__global__ void __launch_bounds__(32 * RowsWarps<NC, T, 2>::value) k_polyakov_rows(const AuxArgs a) {
    typedef RowsCfg<NC> Cfg;
    typedef LinkIO<NC, T, STORE_FULL, true> IO;
    typedef typename IO::T2 T2;
    typedef cx<T> C;
    constexpr int WARPS = RowsWarps<NC, T, 2>::value, LPW = Cfg::LPW, STRIDE = Cfg::STRIDE;
    __shared__ C stage[WARPS * LPW][2][STRIDE];
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    const bool shadow = lane >= LPW * NC;
    const int g = shadow ? LPW - 1 : lane / NC;
    const int r = shadow ? lane - LPW * NC : lane - g * NC;
    const unsigned Vs = (unsigned)a.g.L[0] * a.g.L[1] * a.g.L[2];
    unsigned xs = (blockIdx.x * WARPS + (unsigned)warp) * LPW + (unsigned)g;
    const bool owner = !shadow && xs < Vs;
    if (xs >= Vs) xs = Vs - 1;
    C(*M)[STRIDE] = stage[warp * LPW + g];
    const int x = (int)(xs % (unsigned)a.g.L[0]);
    const int y = (int)((xs / (unsigned)a.g.L[0]) % (unsigned)a.g.L[1]);
    const int z = (int)(xs / ((unsigned)a.g.L[0] * a.g.L[1]));
    auto load_row = [&](int t, C* row) {
        const T2* q = IO::site(IO::plane((const void*)a.links, a.g, 3, site_parity(a.g, x, y, z, t)), cb_of(a.g, x, y, z, t)) +
                      (size_t)r * NC * LINK_TILE;
#pragma unroll
        for (int c = 0; c < NC; ++c) { T2 v = __ldg(q + c * LINK_TILE); row[c] = mk<T>(v.x, v.y); }
    };
    C P[NC], A[NC], Q[NC];
    load_row(0, P);
#pragma unroll 1
    for (int t = 1; t < a.g.L[3]; ++t) {
        const int b = t & 1;
        load_row(t, A);
#pragma unroll
        for (int c = 0; c < NC; ++c) M[b][r * NC + c] = A[c];
        __syncwarp();
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            C acc = mk<T>(0, 0);
#pragma unroll
            for (int q = 0; q < NC; ++q) mad(acc, P[q], M[b][q * NC + j]);
            Q[j] = acc;
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) P[c] = Q[c];
    }
    const C d = row_pick<NC, T>(P, r);
    double re = owner ? (double)d.re : 0.0, im = owner ? (double)d.im : 0.0;
    re = block_sum(re);
    im = block_sum(im);
    if (threadIdx.x == 0) { a.partials[blockIdx.x] = re; a.partials[gridDim.x + blockIdx.x] = im; }
}

// Final pass: result[c] = scale * sum_b partials[c * nb + b], c < ncomp. One block; fixed order.
static __global__ void __launch_bounds__(REDUCE_BLOCK) k_reduce_final(const double* __restrict__ partials, unsigned nb,
                                                               int ncomp, double scale, double* __restrict__ result) {
    for (int c = 0; c < ncomp; ++c) {
        double s = 0.0;
        for (unsigned i = threadIdx.x; i < nb; i += REDUCE_BLOCK) s += partials[(size_t)c * nb + i];
        s = block_sum(s);
        if (threadIdx.x == 0) result[c] = s * scale;
        __syncthreads();
    }
}

template <int NC, class R>
__device__ cx<R> determinant(const cx<R>* A) {
    cx<R> Mx[NC * NC];
    for (int e = 0; e < NC * NC; ++e) Mx[e] = A[e];
    cx<R> det = mk<R>(1, 0);
#pragma unroll 1
    for (int c = 0; c < NC; ++c) {
        int p = c;
        R best = Mx[c * NC + c].re * Mx[c * NC + c].re + Mx[c * NC + c].im * Mx[c * NC + c].im;
        for (int r = c + 1; r < NC; ++r) {
            R m = Mx[r * NC + c].re * Mx[r * NC + c].re + Mx[r * NC + c].im * Mx[r * NC + c].im;
            if (m > best) { best = m; p = r; }
        }
        if (best == (R)0) return mk<R>(0, 0);
        if (p != c) {
            for (int k = 0; k < NC; ++k) { cx<R> t = Mx[p * NC + k]; Mx[p * NC + k] = Mx[c * NC + k]; Mx[c * NC + k] = t; }
            det = mk<R>(-det.re, -det.im);
        }
        det = det * Mx[c * NC + c];
        const cx<R> pinv = (1 / best) * conj(Mx[c * NC + c]);
        for (int r = c + 1; r < NC; ++r) {
            cx<R> f = Mx[r * NC + c] * pinv;
            for (int k = c; k < NC; ++k) Mx[r * NC + k] = Mx[r * NC + k] - f * Mx[c * NC + k];
        }
    }
    return det;
}

template <int NC, class R>
__device__ void fix_determinant_phase(cx<R>* U) {          // last row *= conj(det)/|det|
    cx<R> d = determinant<NC, R>(U);
    R inv = (R)1 / Fn<R>::sqrt(d.re * d.re + d.im * d.im);
    cx<R> ph = mk<R>(d.re * inv, -d.im * inv);
    for (int k = 0; k < NC; ++k) U[(NC - 1) * NC + k] = U[(NC - 1) * NC + k] * ph;
}

// one thread per link; idx = plane * Vh + cb so that stores coalesce
__device__ __forceinline__ bool link_of_thread(const Geom& g, unsigned idx, int& mu, int& p, unsigned& cb) {
    if (idx >= 8u * g.Vh) return false;
    unsigned plane = idx / g.Vh;
    cb = idx - plane * g.Vh;
    mu = (int)(plane >> 1);
    p = (int)(plane & 1u);
    return true;
}

// Reunitarisation, row-per-lane (generic path): modified Gram-Schmidt over the rows with the finished row
// broadcast by warp shuffle, then the determinant by Gaussian elimination with partial pivoting distributed
// over the lanes (the pivot row is the unused lane with the largest |M_rc|^2; no rows are swapped, the sign is
// the parity of the pivot order), last row *= conj(det)/|det| (reading R10). Same formulas as
// gram_schmidt_rows / determinant, which the thread-per-link kernel runs on local arrays.
template <int NC, class T>
__global__ void __launch_bounds__(128) k_reunit_rows(const AuxArgs a) {
    typedef RowsCfg<NC> Cfg;
    typedef LinkIO<NC, T, STORE_FULL, true> IO;
    typedef typename IO::T2 T2;
    typedef cx<T> C;
    constexpr int LPW = Cfg::LPW;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    const bool shadow = lane >= LPW * NC;
    const int g = shadow ? LPW - 1 : lane / NC;
    const int r = shadow ? lane - LPW * NC : lane - g * NC;
    const int gbase = g * NC;
    const unsigned nlinks = 8u * a.g.Vh;
    unsigned idx = (blockIdx.x * 4u + (unsigned)warp) * LPW + (unsigned)g;
    const bool owner = !shadow && idx < nlinks;
    if (idx >= nlinks) idx = nlinks - 1;
    int mu, p; unsigned cb;
    link_of_thread(a.g, idx, mu, p, cb);
    T2* q = IO::site(IO::plane(a.links, a.g, mu, p), cb) + (size_t)r * NC * LINK_TILE;
    C U[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) { T2 v = __ldcs(q + c * LINK_TILE); U[c] = mk<T>(v.x, v.y); }
    // modified Gram-Schmidt, rows top to bottom
#pragma unroll 1
    for (int pr = 0; pr < NC; ++pr) {
        T n2 = 0;
#pragma unroll
        for (int k = 0; k < NC; ++k) n2 += U[k].re * U[k].re + U[k].im * U[k].im;
        const T inv = (T)1 / Fn<T>::sqrt(n2);
        if (r == pr) {
#pragma unroll
            for (int k = 0; k < NC; ++k) U[k] = inv * U[k];
        }
        C dot = mk<T>(0, 0), row[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) { row[k] = shfl_cx(U[k], gbase + pr); mad_ca(dot, row[k], U[k]); }
        if (r > pr) {
#pragma unroll
            for (int k = 0; k < NC; ++k) U[k] = U[k] - dot * row[k];
        }
    }
    // determinant
    C M[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) M[k] = U[k];
    C det = mk<T>(1, 0);
    bool used = false, odd = false;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const T mag = used ? (T)-1 : M[c].re * M[c].re + M[c].im * M[c].im;
        T best = (T)-1;
        int pl = 0;
#pragma unroll
        for (int l = 0; l < NC; ++l) {
            const T ml = __shfl_sync(0xffffffffu, mag, gbase + l);
            if (ml > best) { best = ml; pl = l; }
        }
        const unsigned unused = (__ballot_sync(0xffffffffu, !used) >> gbase) & ((1u << NC) - 1u);
        if (__popc(unused & ((1u << pl) - 1u)) & 1) odd = !odd;      // unused rows above the pivot row = inversions
        C piv[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) piv[k] = shfl_cx(M[k], gbase + pl);
        det = det * piv[c];
        const C pinv = ((T)1 / best) * conj(piv[c]);
        if (r == pl) used = true;
        if (!used) {
            const C f = M[c] * pinv;
#pragma unroll
            for (int k = c; k < NC; ++k) M[k] = M[k] - f * piv[k];
        }
    }
    if (odd) det = mk<T>(-det.re, -det.im);
    const T dinv = (T)1 / Fn<T>::sqrt(det.re * det.re + det.im * det.im);
    const C ph = mk<T>(det.re * dinv, -det.im * dinv);
    if (r == NC - 1) {
#pragma unroll
        for (int k = 0; k < NC; ++k) U[k] = U[k] * ph;
    }
    if (owner) {
#pragma unroll
        for (int c = 0; c < NC; ++c) __stcs(q + c * LINK_TILE, V2<T>::make(U[c].re, U[c].im));
    }
}

// Reunitarisation (reading R10), arithmetic in T. Nc <= 4 runs in registers.
template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(128) k_reunit(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, (NC <= 4)> IO;
    int mu, p; unsigned cb;
    if (!link_of_thread(a.g, blockIdx.x * 128u + threadIdx.x, mu, p, cb)) return;
    typename IO::T2* pl = IO::plane(a.links, a.g, mu, p);
    cx<T> U[NC * NC];
    IO::template load<LD_STREAM>(pl, cb, U);
    if (NC <= 4) {
        reunitarize_small<(NC <= 4 ? NC : 2), T>(U);        // (the conditional only keeps the dead branch of Nc > 4 compilable)
    } else {
        gram_schmidt_rows<NC, T>(U, NC);
        fix_determinant_phase<NC, T>(U);
    }
    IO::template store<true>(pl, cb, U);
}

template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(128) k_init_cold(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    int mu, p; unsigned cb;
    if (!link_of_thread(a.g, blockIdx.x * 128u + threadIdx.x, mu, p, cb)) return;
    cx<T> U[NC * NC];
    for (int i = 0; i < NC; ++i)
        for (int j = 0; j < NC; ++j) U[i * NC + j] = mk<T>(i == j ? (T)1 : (T)0, (T)0);
    IO::store(IO::plane(a.links, a.g, mu, p), cb, U);
}

// Hot start (readings R12, R20): Haar SU(Nc) per link from Philox blocks
// (kind 2, c0 = site, c1 = 0, c3 = block): uniforms in fours -> Box-Muller pairs -> 2Nc^2 Gaussians
// row-major (re,im) -> modified Gram-Schmidt -> last row * conj(det)/|det|. Nc = 2: the first four
// Gaussians, normalised, are (a0..a3). Computed in double, rounded to T on store.
template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(128) k_init_hot(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    int mu, p; unsigned cb;
    if (!link_of_thread(a.g, blockIdx.x * 128u + threadIdx.x, mu, p, cb)) return;
    int c[4];
    decode_cb(a.g, cb, p, c);
    const uint32_t site = lex_of(a.g, c);
    constexpr int NG = (NC == 2) ? 4 : 2 * NC * NC;
    constexpr int NB = (NG + 3) / 4;
    const double TWO_PI = 6.283185307179586476925286766559;
    double g[NB * 4];
#pragma unroll 1
    for (int b = 0; b < NB; ++b) {
        uint32_t w[4];
        philox4x32_10(site, 0u, c2_kind(pack_c2(0, p, mu, 0), RNG_HOT), (uint32_t)b, a.k0, a.k1, w);
        for (int h = 0; h < 2; ++h) {
            double ua = uniform01<double>(w[2 * h]), ub = uniform01<double>(w[2 * h + 1]);
            double rad = ::sqrt(-2.0 * ::log(ua));
            double s, co;
            ::sincos(TWO_PI * ub, &s, &co);
            g[4 * b + 2 * h] = rad * co;
            g[4 * b + 2 * h + 1] = rad * s;
        }
    }
    cx<double> Md[NC * NC];
    if (NC == 2) {
        double n = ::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2] + g[3] * g[3]);
        double a0 = g[0] / n, a1 = g[1] / n, a2 = g[2] / n, a3 = g[3] / n;
        Md[0] = mk<double>(a0, a3); Md[1] = mk<double>(a2, a1);
        Md[NC * NC - 2] = mk<double>(-a2, a1); Md[NC * NC - 1] = mk<double>(a0, -a3);
    } else {
        for (int e = 0; e < NC * NC; ++e) Md[e] = mk<double>(g[2 * e], g[2 * e + 1]);
        gram_schmidt_rows<NC, double>(Md, NC);
        fix_determinant_phase<NC, double>(Md);
    }
    cx<T> U[NC * NC];
    for (int e = 0; e < NC * NC; ++e) U[e] = mk<T>((T)Md[e].re, (T)Md[e].im);
    IO::store(IO::plane(a.links, a.g, mu, p), cb, U);
}

// SoA -> canonical [site][mu][row][col][re,im] doubles for lexicographic sites [site0, site0+nsites)
template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(128) k_export(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    const unsigned l = blockIdx.x * 128u + threadIdx.x;      // local link index = (site - site0) * 4 + mu
    if (l >= a.nsites * 4u) return;
    const unsigned s = a.site0 + (l >> 2);
    const int mu = (int)(l & 3u);
    const int x = (int)(s % (unsigned)a.g.L[0]);
    unsigned r = s / (unsigned)a.g.L[0];
    const int y = (int)(r % (unsigned)a.g.L[1]); r /= (unsigned)a.g.L[1];
    const int z = (int)(r % (unsigned)a.g.L[2]);
    const int t = (int)(r / (unsigned)a.g.L[2]) + a.g.t_halo;                // stored slice of owned slice t
    const int p = site_parity(a.g, x, y, z, t);
    cx<T> U[NC * NC];
    IO::template load<LD_PLAIN>(IO::plane((const void*)a.links, a.g, mu, p), cb_of(a.g, x, y, z, t), U);
    double2* dst = (double2*)a.staging + (size_t)l * NC * NC;
    for (int e = 0; e < NC * NC; ++e) dst[e] = make_double2((double)U[e].re, (double)U[e].im);
}

template <int NC, class T, int STORE, bool UNR>
__global__ void __launch_bounds__(128) k_import(const AuxArgs a) {
    typedef LinkIO<NC, T, STORE, UNR> IO;
    const unsigned l = blockIdx.x * 128u + threadIdx.x;
    if (l >= a.nsites * 4u) return;
    const unsigned s = a.site0 + (l >> 2);
    const int mu = (int)(l & 3u);
    const int x = (int)(s % (unsigned)a.g.L[0]);
    unsigned r = s / (unsigned)a.g.L[0];
    const int y = (int)(r % (unsigned)a.g.L[1]); r /= (unsigned)a.g.L[1];
    const int z = (int)(r % (unsigned)a.g.L[2]);
    const int t = (int)(r / (unsigned)a.g.L[2]) + a.g.t_halo;
    const int p = site_parity(a.g, x, y, z, t);
    const double2* src = (const double2*)a.staging + (size_t)l * NC * NC;
    cx<T> U[NC * NC];
    for (int e = 0; e < NC * NC; ++e) { double2 v = src[e]; U[e] = mk<T>((T)v.x, (T)v.y); }
    IO::store(IO::plane(a.links, a.g, mu, p), cb_of(a.g, x, y, z, t), U);
}

// ---- dispatch -----------------------------------------------------------------------------
// Reunitarise / init / import / export use rolled loops over local arrays for every Nc
// (Gram-Schmidt and the pivoted determinant need dynamic row indices; none of them is hot).
#define SUG_AUX_DISPATCH(KERNEL, GRID, BLOCK)                                                              \
    do {                                                                                                   \
        constexpr int NC = SUG_NC;                                                                         \
        constexpr int ST0 = (NC == 2 ? STORE_QUAT : STORE_FULL);                                           \
        constexpr int ST1 = (NC == 3 ? STORE_RECON12 : ST0);                                               \
        const bool f64 = v.prec == SU_FP64;                                                                \
        if (NC == 3 && v.store == STORE_RECON12) {                                                         \
            if (f64) KERNEL<NC, double, ST1, false><<<GRID, BLOCK, 0, st>>>(a);                            \
            else     KERNEL<NC, float,  ST1, false><<<GRID, BLOCK, 0, st>>>(a);                            \
        } else {                                                                                           \
            if (f64) KERNEL<NC, double, ST0, false><<<GRID, BLOCK, 0, st>>>(a);                            \
            else     KERNEL<NC, float,  ST0, false><<<GRID, BLOCK, 0, st>>>(a);                            \
        }                                                                                                  \
        ++*n_launch;                                                                                       \
    } while (0)

// measurement kernels: unrolled for the specialised variants of Nc <= 4
#define SUG_MEAS_DISPATCH(KERNEL, GRID, BLOCK)                                                                  \
    do {                                                                                                        \
        constexpr int NC = SUG_NC;                                                                              \
        constexpr bool CAN_UNR = NC <= 4;                                                                       \
        constexpr int ST0 = (NC == 2 ? STORE_QUAT : STORE_FULL);                                                \
        constexpr int ST1 = (NC == 3 ? STORE_RECON12 : ST0);                                                    \
        const bool f64 = v.prec == SU_FP64;                                                                     \
        const bool unr = CAN_UNR && !v.generic;                                                                 \
        const bool r12 = (NC == 3 && v.store == STORE_RECON12);                                                 \
        if (unr) {                                                                                              \
            if (r12) { if (f64) KERNEL<NC, double, ST1, CAN_UNR><<<GRID, BLOCK, 0, st>>>(a); else KERNEL<NC, float, ST1, CAN_UNR><<<GRID, BLOCK, 0, st>>>(a); } \
            else     { if (f64) KERNEL<NC, double, ST0, CAN_UNR><<<GRID, BLOCK, 0, st>>>(a); else KERNEL<NC, float, ST0, CAN_UNR><<<GRID, BLOCK, 0, st>>>(a); } \
        } else {                                                                                                \
            if (r12) { if (f64) KERNEL<NC, double, ST1, false><<<GRID, BLOCK, 0, st>>>(a); else KERNEL<NC, float, ST1, false><<<GRID, BLOCK, 0, st>>>(a); }     \
            else     { if (f64) KERNEL<NC, double, ST0, false><<<GRID, BLOCK, 0, st>>>(a); else KERNEL<NC, float, ST0, false><<<GRID, BLOCK, 0, st>>>(a); }     \
        }                                                                                                       \
        ++*n_launch;                                                                                            \
    } while (0)

// the generic path (and every Nc >= 5) measures with the row-per-lane kernels, except in the SU(2) quaternion /
// SU(3) two-row layouts
static bool use_rows(const Variant& v) { return SUG_NC >= 3 && v.store == STORE_FULL && (v.generic || SUG_NC > 4); }

cudaError_t SUG_CAT(plaquette_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    unsigned nb = plaquette_blocks(a.g.Vh_int);
#if SUG_NC >= 3
    if (use_rows(v)) {
        constexpr int NC = SUG_NC;
        if (v.prec == SU_FP64) {
            constexpr unsigned PB = RowsWarps<NC, double, 4>::value * RowsCfg<NC>::LPW;
            nb = 2u * ((a.g.Vh_int + PB - 1) / PB);
            k_plaquette_rows<NC, double><<<nb, 32 * RowsWarps<NC, double, 4>::value, 0, st>>>(a);
        } else {
            constexpr unsigned PB = RowsWarps<NC, float, 4>::value * RowsCfg<NC>::LPW;
            nb = 2u * ((a.g.Vh_int + PB - 1) / PB);
            k_plaquette_rows<NC, float><<<nb, 32 * RowsWarps<NC, float, 4>::value, 0, st>>>(a);
        }
        ++*n_launch;
    } else
#endif
    SUG_MEAS_DISPATCH(k_plaquette, nb, PLAQ_BLOCK);
    // normalised by the GLOBAL volume: in slab mode the result is this slab's share of the plaquette
    const double scale = 1.0 / (6.0 * 2.0 * (double)a.g.Vsh * (double)a.g.Lt_glob * (double)SUG_NC);
    k_reduce_final<<<1, REDUCE_BLOCK, 0, st>>>(a.partials, nb, 1, scale, a.result);
    ++*n_launch;
    return cudaGetLastError();
}

cudaError_t SUG_CAT(polyakov_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned Vs = (unsigned)a.g.L[0] * a.g.L[1] * a.g.L[2];
    unsigned nb = reduce_blocks(Vs);
#if SUG_NC >= 3
    if (use_rows(v)) {
        constexpr int NC = SUG_NC;
        if (v.prec == SU_FP64) {
            constexpr unsigned PB = RowsWarps<NC, double, 2>::value * RowsCfg<NC>::LPW;
            nb = (Vs + PB - 1) / PB;
            k_polyakov_rows<NC, double><<<nb, 32 * RowsWarps<NC, double, 2>::value, 0, st>>>(a);
        } else {
            constexpr unsigned PB = RowsWarps<NC, float, 2>::value * RowsCfg<NC>::LPW;
            nb = (Vs + PB - 1) / PB;
            k_polyakov_rows<NC, float><<<nb, 32 * RowsWarps<NC, float, 2>::value, 0, st>>>(a);
        }
        ++*n_launch;
    } else
#endif
    SUG_MEAS_DISPATCH(k_polyakov, nb, REDUCE_BLOCK);
    k_reduce_final<<<1, REDUCE_BLOCK, 0, st>>>(a.partials, nb, 2, 1.0 / ((double)Vs * (double)SUG_NC), a.result);
    ++*n_launch;
    return cudaGetLastError();
}

cudaError_t SUG_CAT(reunit_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
#if SUG_NC >= 5
    if (use_rows(v)) {          // Nc <= 4 already reunitarise in registers, one thread per link
        constexpr int NC = SUG_NC;
        const unsigned per_block = 4u * RowsCfg<NC>::LPW;
        const unsigned grid_r = (8u * a.g.Vh + per_block - 1) / per_block;
        if (v.prec == SU_FP64) k_reunit_rows<NC, double><<<grid_r, 128, 0, st>>>(a);
        else                   k_reunit_rows<NC, float><<<grid_r, 128, 0, st>>>(a);
        ++*n_launch;
        return cudaGetLastError();
    }
#endif
    const unsigned grid = (8u * a.g.Vh + 127u) / 128u;
    SUG_AUX_DISPATCH(k_reunit, grid, 128);
    return cudaGetLastError();
}
cudaError_t SUG_CAT(init_cold_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned grid = (8u * a.g.Vh + 127u) / 128u;
    SUG_AUX_DISPATCH(k_init_cold, grid, 128);
    return cudaGetLastError();
}
cudaError_t SUG_CAT(init_hot_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned grid = (8u * a.g.Vh + 127u) / 128u;
    SUG_AUX_DISPATCH(k_init_hot, grid, 128);
    return cudaGetLastError();
}
cudaError_t SUG_CAT(export_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned grid = (a.nsites * 4u + 127u) / 128u;
    SUG_AUX_DISPATCH(k_export, grid, 128);
    return cudaGetLastError();
}
cudaError_t SUG_CAT(import_nc, SUG_NC)(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned grid = (a.nsites * 4u + 127u) / 128u;
    SUG_AUX_DISPATCH(k_import, grid, 128);
    return cudaGetLastError();
}

}  // namespace sug
