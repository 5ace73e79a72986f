// big_kernels.cu — the runtime-Nc path of libsugauge for 9 <= Nc <= SU_MAX_NC = 32 (the
// generic SU(Nc) code, measured up to Nc = 16 in double and 32 in single precision).
//
// Nc <= 8 have kernels compiled per Nc (register-resident matrices, update_kernel.cuh; one row per lane,
// update_rows_kernel.cuh). Beyond that a row of a matrix no longer fits a lane's registers, and one kernel per Nc
// would be 24 more template instances of everything. Here Nc is a kernel ARGUMENT and ONE WARP owns a link:
//   * the link's matrices live in shared memory (5 buffers of Nc x Nc complex per warp, dynamic shared memory);
//   * products are spread over the lanes as (row, block of 8 columns): one operand row element is reused for 8
//     columns, sums run over k ascending (the order of the plain definition);
//   * the subgroup loop runs the lexicographic sequence as a wavefront of 2 Nc - 3 slots (pairs with i + j = t + 1
//     are disjoint and commute exactly, as in update_rows_kernel.cuh); a pair is handled by 32 / (Nc / 2) lanes, all
//     of which evaluate the projection and the Kennedy-Pendleton draw (same counter -> same numbers) and share the
//     columns of rows i, j of U and W (eq 15);
//   * the same warp-per-link toolkit carries the plaquette, the Polyakov loop, reunitarisation (modified
//     Gram-Schmidt + phase of the determinant by pivoted elimination), the hot start (in double, reading R20),
//     the cold start and the layout conversion of export / import.
// Storage is the same tiled SoA as everywhere (element e of a link at + e * LINK_TILE); a warp reads a link as Nc^2
// 16-byte (fp64) words 512 bytes apart - half-used sectors, accepted: above Nc ~ 8 the update is bound by the
// Nc^3 products, not by memory (time per update ~ Nc^3).
#include "su_internal.h"

namespace sug {

namespace {

constexpr int BIG_CW = 8;                 // at most this many columns per lane and product chunk (accumulators in registers)

template <class T> struct BigLink {
    typedef typename V2<T>::type T2;
    static __device__ __forceinline__ size_t plane_off(const Geom& g, int nc, int mu, int par) { return (size_t)(mu * 2 + par) * (size_t)(nc * nc) * g.Vhp; }
    static __device__ __forceinline__ size_t site_off(int nc, unsigned cb) { return (size_t)(cb / LINK_TILE) * ((size_t)(nc * nc) * LINK_TILE) + (cb % LINK_TILE); }
    // whole link -> shared memory (row-major), all lanes
    static __device__ __forceinline__ void load(const void* links, const Geom& g, int nc, int mu, int par, unsigned cb, cx<T>* dst, int lane) {
        const T2* p = (const T2*)links + plane_off(g, nc, mu, par) + site_off(nc, cb);
        for (int e = lane; e < nc * nc; e += 32) { const T2 v = p[(size_t)e * LINK_TILE]; dst[e] = mk<T>(v.x, v.y); }
    }
    static __device__ __forceinline__ void store(void* links, const Geom& g, int nc, int mu, int par, unsigned cb, const cx<T>* src, int lane) {
        T2* p = (T2*)links + plane_off(g, nc, mu, par) + site_off(nc, cb);
        for (int e = lane; e < nc * nc; e += 32) p[(size_t)e * LINK_TILE] = V2<T>::make(src[e].re, src[e].im);
    }
};

// D (+)= X' Y', X' = X or X^dagger, Y' = Y or Y^dagger; all n x n row-major in shared memory, D distinct from X, Y.
// Lane -> (row = lane % n, group = lane / n); the 8-column chunks are dealt round-robin to the 32 / n groups.
template <class T, bool XD, bool YD, bool ACC>
__device__ __forceinline__ void wmm(int n, const cx<T>* X, const cx<T>* Y, cx<T>* D, int lane) {
    const int ngroups = 32 / n > 0 ? 32 / n : 1;
    const int row = lane % n, grp = lane / n;
    // (dealing ceil(n / groups) columns to every group instead of chunks of 8 balances the lanes on paper but measured
    //  slower at Nc = 9, 10 and equal elsewhere: the short chunks lose the reuse of the row element; profiles/r02f)
    const int cw = BIG_CW;
    if (grp < ngroups && lane < 32) {
        int chunk = 0;
        for (int c0 = 0; c0 < n; c0 += cw, ++chunk) {
            if (chunk % ngroups != grp) continue;
            const int cend = c0 + cw < n ? c0 + cw : n;
            cx<T> acc[BIG_CW];
#pragma unroll
            for (int jj = 0; jj < BIG_CW; ++jj) acc[jj] = mk<T>(0, 0);
            for (int k = 0; k < n; ++k) {
                const cx<T> x = XD ? conj(X[k * n + row]) : X[row * n + k];
#pragma unroll
                for (int jj = 0; jj < BIG_CW; ++jj) {
                    const int col = c0 + jj;
                    if (col < cend) {
                        const cx<T> y = YD ? conj(Y[col * n + k]) : Y[k * n + col];
                        mad(acc[jj], x, y);
                    }
                }
            }
#pragma unroll
            for (int jj = 0; jj < BIG_CW; ++jj) {
                const int col = c0 + jj;
                if (col < cend) D[row * n + col] = ACC ? D[row * n + col] + acc[jj] : acc[jj];
            }
        }
    }
    __syncwarp();
}

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Modified Gram-Schmidt over the rows (top to bottom, positive normalisation), then last row *= conj(det)/|det|
// (readings R10, R12). M: n x n in shared memory, Wk: n x n scratch. R = arithmetic type.
template <class R>
__device__ void warp_reunitarize(int n, cx<R>* M, cx<R>* Wk, int lane) {
    for (int r = 0; r < n; ++r) {
        for (int p = 0; p < r; ++p) {
            double dre = 0, dim = 0;                       // dot = sum_k conj(M[p][k]) M[r][k]
            for (int k = lane; k < n; k += 32) {
                const cx<R> a = M[p * n + k], b = M[r * n + k];
                dre += (double)(a.re * b.re + a.im * b.im); dim += (double)(a.re * b.im - a.im * b.re);
            }
            const cx<R> dot = mk<R>((R)warp_sum(dre), (R)warp_sum(dim));
            for (int k = lane; k < n; k += 32) M[r * n + k] = M[r * n + k] - dot * M[p * n + k];
            __syncwarp();
        }
        double n2 = 0;
        for (int k = lane; k < n; k += 32) n2 += (double)(M[r * n + k].re * M[r * n + k].re + M[r * n + k].im * M[r * n + k].im);
        const R inv = (R)1 / Fn<R>::sqrt((R)warp_sum(n2));
        for (int k = lane; k < n; k += 32) M[r * n + k] = inv * M[r * n + k];
        __syncwarp();
    }
    // determinant by elimination with partial pivoting on a copy (row swaps flip the sign)
    for (int e = lane; e < n * n; e += 32) Wk[e] = M[e];
    __syncwarp();
    cx<R> det = mk<R>(1, 0);
    for (int c = 0; c < n; ++c) {
        int piv = c;
        R best = Wk[c * n + c].re * Wk[c * n + c].re + Wk[c * n + c].im * Wk[c * n + c].im;
        for (int r = c + 1; r < n; ++r) {                  // every lane scans (n <= 32: cheap, and uniform)
            const R m = Wk[r * n + c].re * Wk[r * n + c].re + Wk[r * n + c].im * Wk[r * n + c].im;
            if (m > best) { best = m; piv = r; }
        }
        if (piv != c) {
            for (int k = lane; k < n; k += 32) { const cx<R> t = Wk[piv * n + k]; Wk[piv * n + k] = Wk[c * n + k]; Wk[c * n + k] = t; }
            det = mk<R>(-det.re, -det.im);
            __syncwarp();
        }
        const cx<R> pc = Wk[c * n + c];
        det = det * pc;
        const cx<R> pinv = ((R)1 / best) * conj(pc);
        __syncwarp();
        for (int r = c + 1 + lane / 8; r < n; r += 4) {    // 4 rows at a time, 8 lanes per row
            const cx<R> f = Wk[r * n + c] * pinv;
            for (int k = c + 1 + (lane & 7); k < n; k += 8) Wk[r * n + k] = Wk[r * n + k] - f * Wk[c * n + k];
        }
        __syncwarp();
    }
    const R dinv = (R)1 / Fn<R>::sqrt(det.re * det.re + det.im * det.im);
    const cx<R> ph = mk<R>(det.re * dinv, -det.im * dinv);
    for (int k = lane; k < n; k += 32) M[(n - 1) * n + k] = M[(n - 1) * n + k] * ph;
    __syncwarp();
}

struct BigCommon {
    int nc;
    int wpb;                 // warps per block
};

// ------------------------------------------------------------------------------------------
// staple + update of one link per warp (rows a1-a6 of SURVEY.md 8(a))
// ------------------------------------------------------------------------------------------
template <class T, int KIND>
__global__ void k_update_big(const UpdateArgs a, const BigCommon bc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    cx<T>* S = (cx<T>*)smem_raw + (size_t)warp * 5 * nn;
    cx<T>* X0 = S + nn; cx<T>* X1 = X0 + nn; cx<T>* X2 = X1 + nn; cx<T>* X3 = X2 + nn;
    const unsigned tix = blockIdx.x * (unsigned)bc.wpb + (unsigned)warp;
    if (tix >= a.g.Vh_int) return;                          // whole warps leave together
    const int p = a.parity, mu = a.mu;
    SiteNbr s;
    site_of_thread(a.g, tix, p, s);
    const unsigned cb = s.cb;
    const int dpmu = sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
    for (int e = lane; e < nn; e += 32) S[e] = mk<T>(0, 0);
    for (int k = 0; k < 3; ++k) {
        const int nu = k + (k >= mu ? 1 : 0);
        const int dpnu = sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
        const int dmnu = sel4(nu, s.dm[0], s.dm[1], s.dm[2], s.dm[3]);
        // upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
        BigLink<T>::load(a.links, a.g, n, nu, p, cb, X0, lane);
        BigLink<T>::load(a.links, a.g, n, mu, 1 - p, cb + (unsigned)dpnu, X1, lane);
        BigLink<T>::load(a.links, a.g, n, nu, 1 - p, cb + (unsigned)dpmu, X2, lane);
        __syncwarp();
        wmm<T, false, false, false>(n, X0, X1, X3, lane);
        wmm<T, false, true, true>(n, X3, X2, S, lane);
        // lower: U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
        BigLink<T>::load(a.links, a.g, n, nu, 1 - p, cb + (unsigned)dmnu, X0, lane);
        BigLink<T>::load(a.links, a.g, n, mu, 1 - p, cb + (unsigned)dmnu, X1, lane);
        BigLink<T>::load(a.links, a.g, n, nu, p, cb + (unsigned)(dmnu + dpmu), X2, lane);
        __syncwarp();
        wmm<T, true, false, false>(n, X0, X1, X3, lane);
        wmm<T, false, false, true>(n, X3, X2, S, lane);
    }
    cx<T>* U = X0; cx<T>* W = X1;
    BigLink<T>::load(a.links, a.g, n, mu, p, cb, U, lane);
    __syncwarp();
    wmm<T, false, true, false>(n, U, S, W, lane);          // W = U S^dagger (step 2)

    // steps 3-5: the lexicographic subgroup sequence as a wavefront (disjoint pairs of a slot commute exactly)
    const T beta = (T)a.beta;
    const T two_beta_over_nc = (T)2 * beta / (T)n, m_nc_over_4beta = (T)-0.25 * (T)n / beta;
    const uint32_t c1 = a.sweep_ptr ? *a.sweep_ptr : a.sweep;
    const uint32_t c2_base = pack_c2((int)a.pass, p, mu, 0);
    const int lpp = 32 / (n / 2);                          // lanes per pair, >= 2 for n <= 32
    const int my_pair = lane / lpp, sub_lane = lane % lpp;
    unsigned att_total = 0, exhausted = 0;
    for (int t = 0; t <= 2 * n - 4; ++t) {
        const int i_min = t + 1 - (n - 1) > 0 ? t + 1 - (n - 1) : 0, i_max = t / 2;          // pairs (i, t+1-i), i < j
        const int npairs = i_max - i_min + 1;
        const bool have = my_pair < npairs;
        const int i = i_min + (have ? my_pair : 0), j = t + 1 - i;
        const int sub = i * n - (i * (i + 1)) / 2 + (j - i - 1);                             // lexicographic index of (i,j)
        const cx<T> wii = W[i * n + i], wij = W[i * n + j], wji = W[j * n + i], wjj = W[j * n + j];
        T r0 = (T)0.5 * (wii.re + wjj.re), r1 = (T)0.5 * (wij.im + wji.im);
        T r2 = (T)0.5 * (wij.re - wji.re), r3 = (T)0.5 * (wii.im - wjj.im);
        const T n2 = r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3;
        bool ok = have && (n2 >= Fn<T>::min_norm2()) && Fn<T>::finite(n2);      // as in update_subgroups
        T q4[4] = {(T)1, (T)0, (T)0, (T)0};
        int used = 0;
        const unsigned draw_mask = (KIND == KIND_HB) ? __ballot_sync(0xffffffffu, ok) : 0u;
        if (ok) {
            if (KIND == KIND_HB) {
                const T ik = Fn<T>::rsqrt_pos(n2), kk = n2 * ik;
                T ud[4] = {r0 * ik, -r1 * ik, -r2 * ik, -r3 * ik};
                T v[4];
                used = kp_draw<T>(draw_mask, two_beta_over_nc * kk, m_nc_over_4beta * ik, a.k0, a.k1, s.lex, c1, c2_base | (uint32_t)sub, v);
                if (used) quat_mul(v, ud, q4); else ok = false;
            } else {
                const T in2 = Fn<T>::rcp_pos(n2), m2r0 = (T)-2 * r0 * in2;
                q4[0] = (r0 * r0 - (r1 * r1 + r2 * r2 + r3 * r3)) * in2;
                q4[1] = m2r0 * r1; q4[2] = m2r0 * r2; q4[3] = m2r0 * r3;
            }
        }
        if (KIND == KIND_HB && have && sub_lane == 0) {
            att_total += (unsigned)used;
            if (!ok) exhausted += 1u;
            if (a.attempts) a.attempts[(size_t)sub * a.g.Vh + cb] = (uint8_t)(used > 255 ? 255 : used);
        }
        __syncwarp();                                      // every lane has read its 2x2 block before rows change
        if (ok) {
            const cx<T> a00 = mk<T>(q4[0], q4[3]), a01 = mk<T>(q4[2], q4[1]), a10 = mk<T>(-q4[2], q4[1]), a11 = mk<T>(q4[0], -q4[3]);
            for (int c = sub_lane; c < 2 * n; c += lpp) {  // columns of U, then of W
                cx<T>* Mx = c < n ? U : W;
                const int col = c < n ? c : c - n;
                const cx<T> ui = Mx[i * n + col], uj = Mx[j * n + col];
                Mx[i * n + col] = a00 * ui + a01 * uj;
                Mx[j * n + col] = a10 * ui + a11 * uj;
            }
        }
        __syncwarp();
    }
    BigLink<T>::store(a.links, a.g, n, mu, p, cb, U, lane);
    if (const int edge = slab_edge(a.g, tix)) {            // fused halo push (slab mode only)
        if (edge & 1) BigLink<T>::store(a.peer_lo, a.g, n, mu, p, halo_cb_lo(a.g, cb), U, lane);
        if (edge & 2) BigLink<T>::store(a.peer_hi, a.g, n, mu, p, halo_cb_hi(a.g, cb), U, lane);
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

// ------------------------------------------------------------------------------------------
// reductions: per-warp partial sums (one site per warp), then k_reduce_big
// ------------------------------------------------------------------------------------------
template <class T>
__global__ void k_plaquette_big(const AuxArgs a, const BigCommon bc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    cx<T>* A = (cx<T>*)smem_raw + (size_t)warp * 4 * nn;
    cx<T>* B = A + nn; cx<T>* P = B + nn; cx<T>* Q = P + nn;
    const unsigned w = blockIdx.x * (unsigned)bc.wpb + (unsigned)warp;        // site index over both parities
    if (w >= 2u * a.g.Vh_int) return;
    const int p = (int)(w & 1u);
    SiteNbr s;
    site_of_thread(a.g, w >> 1, p, s);
    double acc = 0.0;
    for (int mu = 0; mu < 3; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu) {
            const unsigned fmu = s.cb + (unsigned)sel4(mu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
            const unsigned fnu = s.cb + (unsigned)sel4(nu, s.dp[0], s.dp[1], s.dp[2], s.dp[3]);
            BigLink<T>::load(a.links, a.g, n, mu, p, s.cb, A, lane);
            BigLink<T>::load(a.links, a.g, n, nu, 1 - p, fmu, B, lane);
            __syncwarp();
            wmm<T, false, false, false>(n, A, B, P, lane);
            BigLink<T>::load(a.links, a.g, n, nu, p, s.cb, A, lane);
            BigLink<T>::load(a.links, a.g, n, mu, 1 - p, fnu, B, lane);
            __syncwarp();
            wmm<T, false, false, false>(n, A, B, Q, lane);
            T t = 0;
            for (int e = lane; e < nn; e += 32) t += P[e].re * Q[e].re + P[e].im * Q[e].im;
            acc += (double)t;
            __syncwarp();
        }
    acc = warp_sum(acc);
    if (lane == 0) a.partials[w] = acc;
}

template <class T>
__global__ void k_polyakov_big(const AuxArgs a, const BigCommon bc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    cx<T>* P = (cx<T>*)smem_raw + (size_t)warp * 3 * nn;
    cx<T>* A = P + nn; cx<T>* Q = A + nn;
    const unsigned Vs = (unsigned)a.g.L[0] * a.g.L[1] * a.g.L[2];
    const unsigned xs = blockIdx.x * (unsigned)bc.wpb + (unsigned)warp;
    if (xs >= Vs) return;
    const int x = (int)(xs % (unsigned)a.g.L[0]);
    const int y = (int)((xs / (unsigned)a.g.L[0]) % (unsigned)a.g.L[1]);
    const int z = (int)(xs / ((unsigned)a.g.L[0] * a.g.L[1]));
    BigLink<T>::load(a.links, a.g, n, 3, site_parity(a.g, x, y, z, 0), cb_of(a.g, x, y, z, 0), P, lane);
    for (int t = 1; t < a.g.L[3]; ++t) {
        BigLink<T>::load(a.links, a.g, n, 3, site_parity(a.g, x, y, z, t), cb_of(a.g, x, y, z, t), A, lane);
        __syncwarp();
        wmm<T, false, false, false>(n, P, A, Q, lane);
        cx<T>* tmp = P; P = Q; Q = tmp;
    }
    __syncwarp();
    double re = 0, im = 0;
    for (int d = lane; d < n; d += 32) { re += (double)P[d * n + d].re; im += (double)P[d * n + d].im; }
    re = warp_sum(re); im = warp_sum(im);
    if (lane == 0) { a.partials[xs] = re; a.partials[Vs + xs] = im; }
}

// result[c] = scale * sum_i partials[c * n + i]; one block, fixed order
__global__ void __launch_bounds__(REDUCE_BLOCK) k_reduce_big(const double* __restrict__ partials, unsigned n, int ncomp, double scale, double* __restrict__ result) {
    for (int c = 0; c < ncomp; ++c) {
        double s = 0.0;
        for (unsigned i = threadIdx.x; i < n; i += REDUCE_BLOCK) s += partials[(size_t)c * n + i];
        s = block_sum(s);
        if (threadIdx.x == 0) result[c] = s * scale;
        __syncthreads();
    }
}

__device__ __forceinline__ bool big_link_of_warp(const Geom& g, unsigned idx, int& mu, int& p, unsigned& cb) {
    if (idx >= 8u * g.Vh) return false;
    const unsigned plane = idx / g.Vh;
    cb = idx - plane * g.Vh; mu = (int)(plane >> 1); p = (int)(plane & 1u);
    return true;
}

template <class T>
__global__ void k_reunit_big(const AuxArgs a, const BigCommon bc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    cx<T>* M = (cx<T>*)smem_raw + (size_t)warp * 2 * nn;
    int mu, p; unsigned cb;
    if (!big_link_of_warp(a.g, blockIdx.x * (unsigned)bc.wpb + (unsigned)warp, mu, p, cb)) return;
    BigLink<T>::load(a.links, a.g, n, mu, p, cb, M, lane);
    __syncwarp();
    warp_reunitarize<T>(n, M, M + nn, lane);
    BigLink<T>::store(a.links, a.g, n, mu, p, cb, M, lane);
}

template <class T>
__global__ void k_init_cold_big(const AuxArgs a, const BigCommon bc) {
    const int n = bc.nc;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    int mu, p; unsigned cb;
    if (!big_link_of_warp(a.g, blockIdx.x * (unsigned)bc.wpb + (unsigned)warp, mu, p, cb)) return;
    typedef typename V2<T>::type T2;
    T2* q = (T2*)a.links + BigLink<T>::plane_off(a.g, n, mu, p) + BigLink<T>::site_off(n, cb);
    for (int e = lane; e < n * n; e += 32) q[(size_t)e * LINK_TILE] = V2<T>::make((e / n == e % n) ? (T)1 : (T)0, (T)0);
}

// Hot start (readings R12, R20): Philox kind-2 blocks b = 0.. give four uniforms each -> two Box-Muller
// pairs -> the 2 Nc^2 Gaussians of the matrix, row-major (re, im); Gram-Schmidt and determinant phase in double.
template <class T>
__global__ void k_init_hot_big(const AuxArgs a, const BigCommon bc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    cx<double>* M = (cx<double>*)smem_raw + (size_t)warp * 2 * nn;
    int mu, p; unsigned cb;
    if (!big_link_of_warp(a.g, blockIdx.x * (unsigned)bc.wpb + (unsigned)warp, mu, p, cb)) return;
    int c[4];
    decode_cb(a.g, cb, p, c);
    const uint32_t site = lex_of(a.g, c);
    const double TWO_PI = 6.283185307179586476925286766559;
    double* gflat = (double*)M;                            // 2 nn doubles = the matrix itself, (re, im) interleaved
    const int nblocks = (2 * nn + 3) / 4;
    for (int b = lane; b < nblocks; b += 32) {
        uint32_t w[4];
        philox4x32_10(site, 0u, c2_kind(pack_c2(0, p, mu, 0), RNG_HOT), (uint32_t)b, a.k0, a.k1, w);
        for (int h = 0; h < 2; ++h) {
            const double ua = uniform01<double>(w[2 * h]), ub = uniform01<double>(w[2 * h + 1]);
            const double rad = ::sqrt(-2.0 * ::log(ua));
            double sn, co;
            ::sincos(TWO_PI * ub, &sn, &co);
            const int i0 = 4 * b + 2 * h;
            if (i0 < 2 * nn) gflat[i0] = rad * co;
            if (i0 + 1 < 2 * nn) gflat[i0 + 1] = rad * sn;
        }
    }
    __syncwarp();
    warp_reunitarize<double>(n, M, M + nn, lane);
    typedef typename V2<T>::type T2;
    T2* q = (T2*)a.links + BigLink<T>::plane_off(a.g, n, mu, p) + BigLink<T>::site_off(n, cb);
    for (int e = lane; e < nn; e += 32) q[(size_t)e * LINK_TILE] = V2<T>::make((T)M[e].re, (T)M[e].im);
}

// tiled SoA <-> canonical [site][mu][row][col][re,im] doubles for lexicographic sites [site0, site0 + nsites)
template <class T, bool TO_HOST>
__global__ void k_convert_big(const AuxArgs a, const BigCommon bc) {
    const int n = bc.nc, nn = n * n;
    const int lane = (int)(threadIdx.x & 31u), warp = (int)(threadIdx.x >> 5);
    const unsigned l = blockIdx.x * (unsigned)bc.wpb + (unsigned)warp;         // local link index = (site - site0) * 4 + mu
    if (l >= a.nsites * 4u) return;
    const unsigned s = a.site0 + (l >> 2);
    const int mu = (int)(l & 3u);
    const int x = (int)(s % (unsigned)a.g.L[0]);
    unsigned r = s / (unsigned)a.g.L[0];
    const int y = (int)(r % (unsigned)a.g.L[1]); r /= (unsigned)a.g.L[1];
    const int z = (int)(r % (unsigned)a.g.L[2]);
    const int t = (int)(r / (unsigned)a.g.L[2]) + a.g.t_halo;
    const int p = site_parity(a.g, x, y, z, t);
    typedef typename V2<T>::type T2;
    T2* q = (T2*)a.links + BigLink<T>::plane_off(a.g, n, mu, p) + BigLink<T>::site_off(n, cb_of(a.g, x, y, z, t));
    double2* h = (double2*)a.staging + (size_t)l * nn;
    for (int e = lane; e < nn; e += 32) {
        if (TO_HOST) { const T2 v = q[(size_t)e * LINK_TILE]; h[e] = make_double2((double)v.x, (double)v.y); }
        else { const double2 v = h[e]; q[(size_t)e * LINK_TILE] = V2<T>::make((T)v.x, (T)v.y); }
    }
}

// warps per block for nbuf matrices of Nc x Nc complex<R> per warp within ~96 KB of dynamic shared memory
int big_wpb(int nc, size_t real, int nbuf, size_t* bytes) {
    const size_t per_warp = (size_t)nbuf * nc * nc * 2 * real;
    if (per_warp == 0) { *bytes = 0; return 4; }
    int w = (int)((96 * 1024) / per_warp);
    if (w < 1) w = 1;
    if (w > 4) w = 4;
    *bytes = per_warp * w;
    return w;
}

template <class K> cudaError_t big_attr(K kernel, size_t bytes) {
    return bytes > 48 * 1024 ? cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) : cudaSuccess;
}

#define BIG_LAUNCH(KERNEL, ARGS, NWARPS, REAL, NBUF)                                              \
    do {                                                                                          \
        size_t bytes__ = 0;                                                                       \
        BigCommon bc__{v.Nc, big_wpb(v.Nc, REAL, NBUF, &bytes__)};                                \
        cudaError_t e__ = big_attr(KERNEL, bytes__);                                              \
        if (e__ != cudaSuccess) return e__;                                                       \
        const unsigned grid__ = (unsigned)(((size_t)(NWARPS) + bc__.wpb - 1) / bc__.wpb);         \
        KERNEL<<<grid__, 32 * bc__.wpb, bytes__, st>>>(ARGS, bc__);                               \
        ++*n_launch;                                                                              \
    } while (0)

}  // namespace

cudaError_t update_nc_big(const Variant& v, int kind, const UpdateArgs& a, cudaStream_t st, uint64_t* n_launch) {
    if (v.prec == SU_FP64) {
        if (kind == KIND_HB) BIG_LAUNCH((k_update_big<double, KIND_HB>), a, a.g.Vh_int, 8, 5);
        else                 BIG_LAUNCH((k_update_big<double, KIND_OR>), a, a.g.Vh_int, 8, 5);
    } else {
        if (kind == KIND_HB) BIG_LAUNCH((k_update_big<float, KIND_HB>), a, a.g.Vh_int, 4, 5);
        else                 BIG_LAUNCH((k_update_big<float, KIND_OR>), a, a.g.Vh_int, 4, 5);
    }
    return cudaGetLastError();
}

cudaError_t plaquette_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned nw = 2u * a.g.Vh_int;
    if (v.prec == SU_FP64) BIG_LAUNCH(k_plaquette_big<double>, a, nw, 8, 4);
    else                   BIG_LAUNCH(k_plaquette_big<float>, a, nw, 4, 4);
    const double scale = 1.0 / (6.0 * 2.0 * (double)a.g.Vsh * (double)a.g.Lt_glob * (double)v.Nc);
    k_reduce_big<<<1, REDUCE_BLOCK, 0, st>>>(a.partials, nw, 1, scale, a.result);
    ++*n_launch;
    return cudaGetLastError();
}

cudaError_t polyakov_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const unsigned Vs = (unsigned)a.g.L[0] * a.g.L[1] * a.g.L[2];
    if (v.prec == SU_FP64) BIG_LAUNCH(k_polyakov_big<double>, a, Vs, 8, 3);
    else                   BIG_LAUNCH(k_polyakov_big<float>, a, Vs, 4, 3);
    k_reduce_big<<<1, REDUCE_BLOCK, 0, st>>>(a.partials, Vs, 2, 1.0 / ((double)Vs * (double)v.Nc), a.result);
    ++*n_launch;
    return cudaGetLastError();
}

cudaError_t reunit_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const size_t nw = 8 * (size_t)a.g.Vh;
    if (v.prec == SU_FP64) BIG_LAUNCH(k_reunit_big<double>, a, nw, 8, 2);
    else                   BIG_LAUNCH(k_reunit_big<float>, a, nw, 4, 2);
    return cudaGetLastError();
}

cudaError_t init_cold_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const size_t nw = 8 * (size_t)a.g.Vh;
    if (v.prec == SU_FP64) BIG_LAUNCH(k_init_cold_big<double>, a, nw, 8, 0);
    else                   BIG_LAUNCH(k_init_cold_big<float>, a, nw, 4, 0);
    return cudaGetLastError();
}

cudaError_t init_hot_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const size_t nw = 8 * (size_t)a.g.Vh;
    if (v.prec == SU_FP64) BIG_LAUNCH(k_init_hot_big<double>, a, nw, 8, 2);
    else                   BIG_LAUNCH(k_init_hot_big<float>, a, nw, 8, 2);     // the hot start is always computed in double
    return cudaGetLastError();
}

cudaError_t export_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const size_t nw = (size_t)a.nsites * 4;
    if (v.prec == SU_FP64) BIG_LAUNCH((k_convert_big<double, true>), a, nw, 8, 0);
    else                   BIG_LAUNCH((k_convert_big<float, true>), a, nw, 4, 0);
    return cudaGetLastError();
}

cudaError_t import_nc_big(const Variant& v, const AuxArgs& a, cudaStream_t st, uint64_t* n_launch) {
    const size_t nw = (size_t)a.nsites * 4;
    if (v.prec == SU_FP64) BIG_LAUNCH((k_convert_big<double, false>), a, nw, 8, 0);
    else                   BIG_LAUNCH((k_convert_big<float, false>), a, nw, 4, 0);
    return cudaGetLastError();
}

}  // namespace sug
