// su_oracle.cpp — CPU ORACLE (test infrastructure, not the product; see su_oracle.h).
//
// Plain restatement of Cardoso & Bicudo, arXiv:1112.4533, section 2:
// Wilson action, staple (eq 9), SU(2) heatbath (eqs 10-14) with a Kennedy-Pendleton a0 draw,
// Cabibbo-Marinari subgroup sweep (steps 1-5, eq 15), overrelaxation (eq 17), reunitarisation,
// plaquette (eq 4) and a Polyakov loop. Slow on purpose: runtime Nc, std::complex, no blocking,
// no fusion. OpenMP only distributes the independent links of one (parity, mu) sub-step; the
// counter-based RNG makes the result bitwise independent of the thread count.
//
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).
#include "su_oracle.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <limits>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11).
// Counter (c0..c3), key (k0,k1). One round:
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// key bumped by (W0,W1) between rounds, 10 rounds.
// ------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Uniform in (0,1], exact in T: fp64 (w+1)/2^32, fp32 ((w>>8)+1)/2^24.
template <class T> T uniform01(uint32_t w);
template <> double uniform01<double>(uint32_t w) { return ((double)w + 1.0) * (1.0 / 4294967296.0); }
template <> float  uniform01<float >(uint32_t w) { return ((float)(w >> 8) + 1.0f) * (1.0f / 16777216.0f); }

// RNG counter word c2 = kind<<28 | pass<<20 | parity<<19 | mu<<17 | subgroup.
enum { KIND_KP = 0, KIND_DIR = 1, KIND_HOT = 2 };
inline uint32_t pack_c2(int kind, int pass, int parity, int mu, int subgroup) {
    return ((uint32_t)kind << 28) | ((uint32_t)(pass & 0xff) << 20) | ((uint32_t)parity << 19) |
           ((uint32_t)mu << 17) | (uint32_t)subgroup;
}

const int KP_MAX_ATTEMPTS = 1024;   // DESIGN.md reading R15

// ------------------------------------------------------------------------------------------
// Kennedy-Pendleton draw of v = (a0, a) with P(a0) ~ sqrt(1-a0^2) exp(alpha a0) (eq 13,
// PAPER.md:100) and a uniform on the sphere of radius sqrt(1-a0^2).
// c2_base carries pass/parity/mu/subgroup with kind bits zero. Returns attempts used (>=1) or 0
// if the attempt cap was hit / alpha unusable (then v is untouched).
// ------------------------------------------------------------------------------------------
template <class T>
int kp_draw(T alpha, const uint32_t key[2], uint32_t c0, uint32_t c1, uint32_t c2_base, T v[4]) {
    const T TWO_PI = (T)6.283185307179586476925286766559;
    if (!(alpha > (T)0) || !std::isfinite(alpha)) return 0;
    T a0 = 0;
    int used = 0;
    for (int n = 0; n < KP_MAX_ATTEMPTS; ++n) {
        uint32_t ctr[4] = {c0, c1, c2_base | ((uint32_t)KIND_KP << 28), (uint32_t)n}, w[4];
        philox4x32_10(ctr, key, w);
        T r1 = uniform01<T>(w[0]), r2 = uniform01<T>(w[1]), r3 = uniform01<T>(w[2]), r4 = uniform01<T>(w[3]);
        T c = std::cos(TWO_PI * r2);
        T lambda2 = -(std::log(r1) + c * c * std::log(r3)) / ((T)2 * alpha);
        if (r4 * r4 <= (T)1 - lambda2) {          // reading R14: accept on equality
            a0 = (T)1 - (T)2 * lambda2;
            used = n + 1;
            break;
        }
    }
    if (!used) return 0;
    uint32_t ctr[4] = {c0, c1, c2_base | ((uint32_t)KIND_DIR << 28), 0u}, w[4];
    philox4x32_10(ctr, key, w);
    T u1 = uniform01<T>(w[0]), u2 = uniform01<T>(w[1]);
    T cos_t = (T)1 - (T)2 * u1;
    T sin_t = std::sqrt(std::max((T)0, (T)1 - cos_t * cos_t));
    T phi = TWO_PI * u2;
    T rho = std::sqrt(std::max((T)0, (T)1 - a0 * a0));
    v[0] = a0;
    v[1] = rho * sin_t * std::cos(phi);
    v[2] = rho * sin_t * std::sin(phi);
    v[3] = rho * cos_t;
    return used;
}

// Quaternion product in the parameterisation U = a0 + i a.sigma (eq 6):
// (ab)_0 = a0 b0 - a.b ; (ab)_vec = a0 b + b0 a - a x b.
template <class T> void quat_mul(const T a[4], const T b[4], T out[4]) {
    out[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    out[1] = a[0] * b[1] + b[0] * a[1] - (a[2] * b[3] - a[3] * b[2]);
    out[2] = a[0] * b[2] + b[0] * a[2] - (a[3] * b[1] - a[1] * b[3]);
    out[3] = a[0] * b[3] + b[0] * a[3] - (a[1] * b[2] - a[2] * b[1]);
}

// ---- plain Nc x Nc complex matrix helpers (row-major) ----
template <class T> using cx = std::complex<T>;

template <class T> void mat_mul(int N, const cx<T>* A, const cx<T>* B, cx<T>* C) {          // C = A B
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
            cx<T> s(0, 0);
            for (int k = 0; k < N; ++k) s += A[i * N + k] * B[k * N + j];
            C[i * N + j] = s;
        }
}
template <class T> void mat_dagger(int N, const cx<T>* A, cx<T>* C) {                       // C = A^dagger
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) C[i * N + j] = std::conj(A[j * N + i]);
}
template <class T> void mat_add(int N, cx<T>* S, const cx<T>* A) {
    for (int i = 0; i < N * N; ++i) S[i] += A[i];
}

// Third row of an SU(3) matrix from the first two: row2 = conj(row0 x row1).
template <class T> void su3_third_row(cx<T>* U) {
    U[6] = std::conj(U[1] * U[5] - U[2] * U[4]);
    U[7] = std::conj(U[2] * U[3] - U[0] * U[5]);
    U[8] = std::conj(U[0] * U[4] - U[1] * U[3]);
}

// Determinant by Gaussian elimination with partial pivoting.
template <class T> cx<T> mat_det(int N, const cx<T>* A) {
    std::vector<cx<T>> M(A, A + N * N);
    cx<T> det(1, 0);
    for (int c = 0; c < N; ++c) {
        int p = c;
        for (int r = c + 1; r < N; ++r)
            if (std::abs(M[r * N + c]) > std::abs(M[p * N + c])) p = r;
        if (std::abs(M[p * N + c]) == (T)0) return cx<T>(0, 0);
        if (p != c) {
            for (int k = 0; k < N; ++k) std::swap(M[p * N + k], M[c * N + k]);
            det = -det;
        }
        det *= M[c * N + c];
        for (int r = c + 1; r < N; ++r) {
            cx<T> f = M[r * N + c] / M[c * N + c];
            for (int k = c; k < N; ++k) M[r * N + k] -= f * M[c * N + k];
        }
    }
    return det;
}

// Modified Gram-Schmidt over rows, top to bottom, positive normalisation.
template <class T> void gram_schmidt_rows(int N, cx<T>* U, int nrows) {
    for (int r = 0; r < nrows; ++r) {
        for (int p = 0; p < r; ++p) {
            cx<T> dot(0, 0);                                   // <row_p, row_r> = sum conj(p) r
            for (int k = 0; k < N; ++k) dot += std::conj(U[p * N + k]) * U[r * N + k];
            for (int k = 0; k < N; ++k) U[r * N + k] -= dot * U[p * N + k];
        }
        T n2 = 0;
        for (int k = 0; k < N; ++k) n2 += std::norm(U[r * N + k]);
        T inv = (T)1 / std::sqrt(n2);
        for (int k = 0; k < N; ++k) U[r * N + k] *= inv;
    }
}

// Reunitarisation of one link (reading R10).
template <class T> void reunitarize_link(int N, cx<T>* U) {
    if (N == 2) {                       // normalise the first row, rebuild the second
        T n = std::sqrt(std::norm(U[0]) + std::norm(U[1]));
        U[0] /= n; U[1] /= n;
        U[2] = -std::conj(U[1]);
        U[3] = std::conj(U[0]);
    } else if (N == 3) {                // Gram-Schmidt on rows 0,1; row 2 by the cross product
        gram_schmidt_rows(N, U, 2);
        su3_third_row(U);
    } else {                            // Gram-Schmidt, then a phase on the last row: det = 1
        gram_schmidt_rows(N, U, N);
        cx<T> d = mat_det(N, U);
        cx<T> ph = std::conj(d) / std::abs(d);
        for (int k = 0; k < N; ++k) U[(N - 1) * N + k] *= ph;
    }
}

// ------------------------------------------------------------------------------------------
// Steps 3-5 of the Cabibbo-Marinari procedure on one link: for every
// subgroup (i<j) in lexicographic order, project the 2x2 block of W = U S^dagger (eq 11), get
// the SU(2) element a by heatbath (kind 0) or overrelaxation (kind 1), and left-multiply rows
// i,j of U and of W by a embedded (eqs 15,16). Returns number of exhausted/unchanged HB draws.
// ------------------------------------------------------------------------------------------
template <class T>
int update_subgroups(int N, T beta, int kind, const uint32_t key[2], uint32_t c0, uint32_t c1,
                     uint32_t c2_base, cx<T>* U, cx<T>* W, uint8_t* attempts, uint64_t* attempts_total) {
    int exhausted = 0, q = 0;
    for (int i = 0; i < N - 1; ++i)
        for (int j = i + 1; j < N; ++j, ++q) {
            if (attempts) attempts[q] = 0;
            const cx<T> wii = W[i * N + i], wij = W[i * N + j], wji = W[j * N + i], wjj = W[j * N + j];
            T r[4] = {(T)0.5 * (wii.real() + wjj.real()), (T)0.5 * (wij.imag() + wji.imag()),
                      (T)0.5 * (wij.real() - wji.real()), (T)0.5 * (wii.imag() - wjj.imag())};
            T k = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
            if (!(k > (T)0) || !std::isfinite(k)) { if (kind == 0) ++exhausted; continue; }
            // u~ = r/k; its inverse (dagger) as a quaternion: (u0, -u1, -u2, -u3)
            T ud[4] = {r[0] / k, -r[1] / k, -r[2] / k, -r[3] / k};
            T a[4];
            if (kind == 0) {
                T alpha = (T)2 * beta * k / (T)N;          // reading R3: weight exp(alpha * a0)
                T v[4];
                int used = kp_draw<T>(alpha, key, c0, c1, c2_base | (uint32_t)q, v);
                if (!used) { ++exhausted; continue; }
                if (attempts) attempts[q] = (uint8_t)(used > 255 ? 255 : used);
                if (attempts_total) *attempts_total += (uint64_t)used;
                quat_mul(v, ud, a);                        // a = v u~^-1   (eq 14)
            } else {
                quat_mul(ud, ud, a);                       // a = (u~^-1)^2 (eq 17 per subgroup)
            }
            // eq 6: [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]]
            const cx<T> a00(a[0], a[3]), a01(a[2], a[1]), a10(-a[2], a[1]), a11(a[0], -a[3]);
            for (int c = 0; c < N; ++c) {
                cx<T> ui = U[i * N + c], uj = U[j * N + c];
                U[i * N + c] = a00 * ui + a01 * uj;
                U[j * N + c] = a10 * ui + a11 * uj;
                cx<T> wi = W[i * N + c], wj = W[j * N + c];
                W[i * N + c] = a00 * wi + a01 * wj;
                W[j * N + c] = a10 * wi + a11 * wj;
            }
        }
    return exhausted;
}

struct LatticeBase {
    virtual ~LatticeBase() {}
    virtual int init_cold(uint64_t seed) = 0;
    virtual int init_hot(uint64_t seed) = 0;
    virtual int set_rng(uint64_t seed, uint32_t sweep) = 0;
    virtual int sweep(double beta, int n_hb, int n_or) = 0;
    virtual int substep(double beta, int kind, int pass, int parity, int mu, uint8_t* attempts) = 0;
    virtual int plaquette(double* out) = 0;
    virtual int polyakov(double* out) = 0;
    virtual int reunitarize() = 0;
    virtual int export_links(double* dst, size_t n) = 0;
    virtual int import_links(const double* src, size_t n) = 0;
    virtual int counters(uint64_t* a, uint64_t* e) = 0;
    virtual int staple_out(size_t site, int mu, double* out) = 0;
};

template <class T> struct Lattice : LatticeBase {
    int N, L[4];
    size_t V;
    bool recon12, ready = false;
    std::vector<cx<T>> U;                      // [site][mu][N*N], site lexicographic, x fastest
    uint32_t key[2] = {0, 0};
    uint32_t sweep_counter = 0;
    uint64_t kp_attempts_total = 0, kp_exhausted = 0;

    Lattice(int Nc, int Lx, int Ly, int Lz, int Lt, bool r12) : N(Nc), recon12(r12) {
        L[0] = Lx; L[1] = Ly; L[2] = Lz; L[3] = Lt;
        V = (size_t)Lx * Ly * Lz * Lt;
        U.assign(V * 4 * N * N, cx<T>(0, 0));
    }
    cx<T>* link(size_t site, int mu) { return &U[(site * 4 + mu) * N * N]; }
    void coords(size_t i, int x[4]) const {
        x[0] = (int)(i % L[0]); i /= L[0];
        x[1] = (int)(i % L[1]); i /= L[1];
        x[2] = (int)(i % L[2]); i /= L[2];
        x[3] = (int)i;
    }
    size_t index(const int x[4]) const {
        return (size_t)x[0] + (size_t)L[0] * (x[1] + (size_t)L[1] * (x[2] + (size_t)L[2] * x[3]));
    }
    // periodic neighbour: site + dir * mu-hat
    size_t shift(size_t i, int mu, int dir) const {
        int x[4]; coords(i, x);
        x[mu] = (x[mu] + dir + L[mu]) % L[mu];
        return index(x);
    }
    void store_fix(cx<T>* u) { if (recon12) su3_third_row(u); }

    void set_key(uint64_t seed) { key[0] = (uint32_t)seed; key[1] = (uint32_t)(seed >> 32); }

    int init_cold(uint64_t seed) override {
        for (size_t l = 0; l < V * 4; ++l)
            for (int i = 0; i < N; ++i)
                for (int j = 0; j < N; ++j) U[l * N * N + i * N + j] = cx<T>(i == j ? 1 : 0, 0);
        set_key(seed); sweep_counter = 0; kp_attempts_total = kp_exhausted = 0; ready = true;
        return 0;
    }

    // Hot start (reading R12): Haar SU(Nc). Per link, Philox blocks (kind 2,
    // c3 = block number) -> uniforms in fours -> Box-Muller pairs -> 2Nc^2 Gaussians filling the
    // matrix row-major (re, im) -> modified Gram-Schmidt over rows -> last row * conj(det)/|det|.
    // Nc = 2: the first four Gaussians, normalised, are (a0..a3) of eq 6. Always computed in
    // double and rounded to T on store (reading R20).
    int init_hot(uint64_t seed) override {
        set_key(seed); sweep_counter = 0; kp_attempts_total = kp_exhausted = 0;
        const double TWO_PI = 6.283185307179586476925286766559;
        const int ng = (N == 2) ? 4 : 2 * N * N;
#pragma omp parallel for schedule(static)
        for (long long s = 0; s < (long long)V; ++s) {
            int x[4]; coords((size_t)s, x);
            int parity = (x[0] + x[1] + x[2] + x[3]) & 1;
            std::vector<double> g(ng + 4);
            std::vector<cx<double>> M(N * N);
            for (int mu = 0; mu < 4; ++mu) {
                for (int b = 0; 4 * b < ng; ++b) {
                    uint32_t ctr[4] = {(uint32_t)s, 0u, pack_c2(KIND_HOT, 0, parity, mu, 0), (uint32_t)b}, w[4];
                    philox4x32_10(ctr, key, w);
                    for (int h = 0; h < 2; ++h) {
                        double ua = uniform01<double>(w[2 * h]), ub = uniform01<double>(w[2 * h + 1]);
                        double rad = std::sqrt(-2.0 * std::log(ua));
                        g[4 * b + 2 * h]     = rad * std::cos(TWO_PI * ub);
                        g[4 * b + 2 * h + 1] = rad * std::sin(TWO_PI * ub);
                    }
                }
                if (N == 2) {
                    double n = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2] + g[3] * g[3]);
                    double a0 = g[0] / n, a1 = g[1] / n, a2 = g[2] / n, a3 = g[3] / n;
                    M[0] = cx<double>(a0, a3);  M[1] = cx<double>(a2, a1);
                    M[2] = cx<double>(-a2, a1); M[3] = cx<double>(a0, -a3);
                } else {
                    for (int e = 0; e < N * N; ++e) M[e] = cx<double>(g[2 * e], g[2 * e + 1]);
                    gram_schmidt_rows<double>(N, M.data(), N);
                    cx<double> d = mat_det<double>(N, M.data());
                    cx<double> ph = std::conj(d) / std::abs(d);
                    for (int k = 0; k < N; ++k) M[(N - 1) * N + k] *= ph;
                }
                cx<T>* u = link((size_t)s, mu);
                for (int e = 0; e < N * N; ++e) u[e] = cx<T>((T)M[e].real(), (T)M[e].imag());
                store_fix(u);
            }
        }
        ready = true;
        return 0;
    }

    int set_rng(uint64_t seed, uint32_t sweep) override { set_key(seed); sweep_counter = sweep; return 0; }

    // Staple of link (x, mu): eq 9 exactly as printed, nu ascending, upper term
    // before lower, products left to right.
    void staple(size_t x, int mu, cx<T>* S) {
        std::vector<cx<T>> A(N * N), B(N * N), D(N * N);
        for (int e = 0; e < N * N; ++e) S[e] = cx<T>(0, 0);
        const size_t xpmu = shift(x, mu, +1);
        for (int nu = 0; nu < 4; ++nu) {
            if (nu == mu) continue;
            // U_nu(x) U_mu(x+nu) U_nu(x+mu)^dagger
            mat_mul(N, link(x, nu), link(shift(x, nu, +1), mu), A.data());
            mat_dagger(N, link(xpmu, nu), D.data());
            mat_mul(N, A.data(), D.data(), B.data());
            mat_add(N, S, B.data());
            // U_nu(x-nu)^dagger U_mu(x-nu) U_nu(x-nu+mu)
            const size_t xmnu = shift(x, nu, -1);
            mat_dagger(N, link(xmnu, nu), D.data());
            mat_mul(N, D.data(), link(xmnu, mu), A.data());
            mat_mul(N, A.data(), link(shift(xmnu, mu, +1), nu), B.data());
            mat_add(N, S, B.data());
        }
    }

    int substep(double beta, int kind, int pass, int parity, int mu, uint8_t* attempts) override {
        if (!ready) return 5;
        if (!(beta >= 0) || !std::isfinite(beta) || kind < 0 || kind > 1 || parity < 0 || parity > 1 ||
            mu < 0 || mu > 3 || pass < 0 || pass > 255) return 1;
        const int nsub = N * (N - 1) / 2;
        const size_t half = V / 2;
        uint64_t att_total = 0, exh_total = 0;
#pragma omp parallel for schedule(static) reduction(+ : att_total, exh_total)
        for (long long s = 0; s < (long long)V; ++s) {
            int x[4]; coords((size_t)s, x);
            if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
            std::vector<cx<T>> S(N * N), Sd(N * N), W(N * N);
            std::vector<uint8_t> att(nsub);
            cx<T>* u = link((size_t)s, mu);
            staple((size_t)s, mu, S.data());                       // step 1
            mat_dagger(N, S.data(), Sd.data());
            mat_mul(N, u, Sd.data(), W.data());                    // step 2: U S^dagger
            uint64_t a_tot = 0;
            int exh = update_subgroups<T>(N, (T)beta, kind, key, (uint32_t)s, sweep_counter,
                                          pack_c2(0, pass, parity, mu, 0), u, W.data(), att.data(), &a_tot);
            store_fix(u);
            att_total += a_tot; exh_total += (uint64_t)exh;
            if (attempts)
                for (int q = 0; q < nsub; ++q) attempts[(size_t)q * half + (size_t)s / 2] = att[q];
        }
        kp_attempts_total += att_total; kp_exhausted += exh_total;
        return 0;
    }

    // Schedule (reading R6): all HB passes, then all OR passes; within
    // a pass parity 0 then 1, mu = 0..3 inside.
    int sweep(double beta, int n_hb, int n_or) override {
        if (!ready) return 5;
        if (n_hb < 0 || n_or < 0 || n_hb > 255) return 1;
        for (int pass = 0; pass < n_hb + n_or; ++pass) {
            int kind = pass < n_hb ? 0 : 1;
            for (int parity = 0; parity < 2; ++parity)
                for (int mu = 0; mu < 4; ++mu) {
                    int rc = substep(beta, kind, kind == 0 ? pass : 0, parity, mu, nullptr);
                    if (rc) return rc;
                }
        }
        ++sweep_counter;
        return 0;
    }

    // <P> = (1/(6 V Nc)) sum_x sum_{mu<nu} ReTr P_mu,nu(x), P of eq 4; fp64 sum.
    int plaquette(double* out) override {
        if (!ready) return 5;
        std::vector<double> per_site(V);
#pragma omp parallel for schedule(static)
        for (long long s = 0; s < (long long)V; ++s) {
            std::vector<cx<T>> A(N * N), B(N * N), D(N * N);
            double acc = 0;
            for (int mu = 0; mu < 4; ++mu)
                for (int nu = mu + 1; nu < 4; ++nu) {
                    // U_mu(s) U_nu(s+mu) U_mu(s+nu)^dagger U_nu(s)^dagger
                    mat_mul(N, link((size_t)s, mu), link(shift((size_t)s, mu, +1), nu), A.data());
                    mat_dagger(N, link(shift((size_t)s, nu, +1), mu), D.data());
                    mat_mul(N, A.data(), D.data(), B.data());
                    mat_dagger(N, link((size_t)s, nu), D.data());
                    mat_mul(N, B.data(), D.data(), A.data());
                    for (int i = 0; i < N; ++i) acc += (double)A[i * N + i].real();
                }
            per_site[s] = acc;
        }
        double sum = 0;
        for (size_t s = 0; s < V; ++s) sum += per_site[s];
        *out = sum / (6.0 * (double)V * (double)N);
        return 0;
    }

    // Polyakov loop (not in the paper; north_star, reading R9):
    // L = (1/(V_s Nc)) sum_{xvec} Tr prod_{t=0}^{Lt-1} U_3(xvec, t).
    int polyakov(double* out) override {
        if (!ready) return 5;
        const size_t Vs = (size_t)L[0] * L[1] * L[2];
        std::vector<double> re(Vs), im(Vs);
#pragma omp parallel for schedule(static)
        for (long long xs = 0; xs < (long long)Vs; ++xs) {
            std::vector<cx<T>> P(link((size_t)xs, 3), link((size_t)xs, 3) + N * N), Q(N * N);
            for (int t = 1; t < L[3]; ++t) {
                mat_mul(N, P.data(), link((size_t)xs + Vs * t, 3), Q.data());
                P = Q;
            }
            double r = 0, i = 0;
            for (int d = 0; d < N; ++d) { r += (double)P[d * N + d].real(); i += (double)P[d * N + d].imag(); }
            re[xs] = r; im[xs] = i;
        }
        double sr = 0, si = 0;
        for (size_t xs = 0; xs < Vs; ++xs) { sr += re[xs]; si += im[xs]; }
        out[0] = sr / ((double)Vs * N); out[1] = si / ((double)Vs * N);
        return 0;
    }

    int reunitarize() override {
        if (!ready) return 5;
#pragma omp parallel for schedule(static)
        for (long long l = 0; l < (long long)(V * 4); ++l) reunitarize_link<T>(N, &U[(size_t)l * N * N]);
        return 0;
    }

    int export_links(double* dst, size_t n) override {
        if (!ready) return 5;
        if (n != V * 4 * 2 * (size_t)N * N) return 1;
        for (size_t e = 0; e < V * 4 * (size_t)N * N; ++e) { dst[2 * e] = (double)U[e].real(); dst[2 * e + 1] = (double)U[e].imag(); }
        return 0;
    }
    int import_links(const double* src, size_t n) override {
        if (n != V * 4 * 2 * (size_t)N * N) return 1;
        for (size_t e = 0; e < V * 4 * (size_t)N * N; ++e) U[e] = cx<T>((T)src[2 * e], (T)src[2 * e + 1]);
        if (recon12) for (size_t l = 0; l < V * 4; ++l) su3_third_row(&U[l * N * N]);
        ready = true;
        return 0;
    }
    int counters(uint64_t* a, uint64_t* e) override {
        if (a) *a = kp_attempts_total;
        if (e) *e = kp_exhausted;
        return 0;
    }
    int staple_out(size_t site, int mu, double* out) override {
        if (!ready) return 5;
        if (site >= V || mu < 0 || mu > 3) return 1;
        std::vector<cx<T>> S(N * N);
        staple(site, mu, S.data());
        for (int e = 0; e < N * N; ++e) { out[2 * e] = (double)S[e].real(); out[2 * e + 1] = (double)S[e].imag(); }
        return 0;
    }
};

template <class T>
int kp_sample_impl(double alpha, uint64_t seed, size_t n, double* out_v, uint8_t* out_attempts) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (size_t i = 0; i < n; ++i) {
        T v[4] = {0, 0, 0, 0};
        int used = kp_draw<T>((T)alpha, key, (uint32_t)i, 0u, 0u, v);
        for (int c = 0; c < 4; ++c) out_v[4 * i + c] = (double)v[c];
        if (out_attempts) out_attempts[i] = (uint8_t)(used > 255 ? 255 : used);
    }
    return 0;
}

template <class T>
int update_matrix_impl(int N, double beta, int kind, uint64_t seed, uint32_t c0, uint32_t c1,
                       uint32_t c2_base, double* U, double* W, uint8_t* attempts) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    std::vector<cx<T>> u(N * N), w(N * N);
    for (int e = 0; e < N * N; ++e) { u[e] = cx<T>((T)U[2 * e], (T)U[2 * e + 1]); w[e] = cx<T>((T)W[2 * e], (T)W[2 * e + 1]); }
    update_subgroups<T>(N, (T)beta, kind, key, c0, c1, c2_base, u.data(), w.data(), attempts, nullptr);
    for (int e = 0; e < N * N; ++e) {
        U[2 * e] = (double)u[e].real(); U[2 * e + 1] = (double)u[e].imag();
        W[2 * e] = (double)w[e].real(); W[2 * e + 1] = (double)w[e].imag();
    }
    return 0;
}

}  // namespace

struct so_lattice { LatticeBase* impl; };

extern "C" {

int so_create(int Nc, int Lx, int Ly, int Lz, int Lt, int precision, int recon12, so_lattice** out) {
    if (!out) return 1;
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int d = 0; d < 4; ++d) if (L[d] < 2 || (L[d] & 1)) return 1;      // reading R7: even extents
    if (Nc < 2 || Nc > 64) return 1;
    if (precision != 0 && precision != 1) return 1;
    if (recon12 && Nc != 3) return 1;
    if ((double)Lx * Ly * Lz * Lt > 4294967295.0) return 1;               // site index is a 32-bit RNG word
    try {
        so_lattice* h = new so_lattice;
        if (precision == 0) h->impl = new Lattice<float>(Nc, Lx, Ly, Lz, Lt, recon12 != 0);
        else                h->impl = new Lattice<double>(Nc, Lx, Ly, Lz, Lt, recon12 != 0);
        *out = h;
    } catch (const std::bad_alloc&) { return 3; }
    return 0;
}
void so_destroy(so_lattice* h) { if (h) { delete h->impl; delete h; } }
int so_init_cold(so_lattice* h, uint64_t seed) { return h ? h->impl->init_cold(seed) : 1; }
int so_init_hot(so_lattice* h, uint64_t seed) { return h ? h->impl->init_hot(seed) : 1; }
int so_set_rng(so_lattice* h, uint64_t seed, uint32_t sweep) { return h ? h->impl->set_rng(seed, sweep) : 1; }
int so_sweep(so_lattice* h, double beta, int n_hb, int n_or) {
    if (!h || !(beta >= 0) || !std::isfinite(beta)) return 1;
    return h->impl->sweep(beta, n_hb, n_or);
}
int so_substep(so_lattice* h, double beta, int kind, int pass, int parity, int mu, uint8_t* attempts) {
    return h ? h->impl->substep(beta, kind, pass, parity, mu, attempts) : 1;
}
int so_plaquette(so_lattice* h, double* out) { return (h && out) ? h->impl->plaquette(out) : 1; }
int so_polyakov(so_lattice* h, double out[2]) { return (h && out) ? h->impl->polyakov(out) : 1; }
int so_reunitarize(so_lattice* h) { return h ? h->impl->reunitarize() : 1; }
int so_export_links(so_lattice* h, double* dst, size_t n) { return (h && dst) ? h->impl->export_links(dst, n) : 1; }
int so_import_links(so_lattice* h, const double* src, size_t n) { return (h && src) ? h->impl->import_links(src, n) : 1; }
int so_get_counters(so_lattice* h, uint64_t* a, uint64_t* e) { return h ? h->impl->counters(a, e) : 1; }

void so_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
double so_uniform(uint32_t w, int precision) {
    return precision == 0 ? (double)uniform01<float>(w) : uniform01<double>(w);
}
int so_staple(so_lattice* h, size_t site, int mu, double* out) { return (h && out) ? h->impl->staple_out(site, mu, out) : 1; }
int so_kp_sample(int precision, double alpha, uint64_t seed, size_t n, double* out_v, uint8_t* out_attempts) {
    if (!out_v) return 1;
    return precision == 0 ? kp_sample_impl<float>(alpha, seed, n, out_v, out_attempts)
                          : kp_sample_impl<double>(alpha, seed, n, out_v, out_attempts);
}
int so_update_matrix(int Nc, int precision, double beta, int kind, uint64_t seed, uint32_t c0, uint32_t c1,
                     uint32_t c2_base, double* U, double* W, uint8_t* attempts) {
    if (Nc < 2 || !U || !W || kind < 0 || kind > 1) return 1;
    return precision == 0 ? update_matrix_impl<float>(Nc, beta, kind, seed, c0, c1, c2_base, U, W, attempts)
                          : update_matrix_impl<double>(Nc, beta, kind, seed, c0, c1, c2_base, U, W, attempts);
}
int so_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
