// su_device.cuh — device-side building blocks of libsugauge (sm_100a).
// Complex Nc x Nc arithmetic in registers (UNR=true) or local arrays (UNR=false, generic kernel),
// checkerboard geometry, SoA link I/O, Philox4x32-10 and the Kennedy-Pendleton draw.
// Method: Cardoso & Bicudo, arXiv:1112.4533 (PAPER.md cited by line); readings R1..R20 in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
// -DSUG_CHECK=1 (a debug build: SUG_BUILD_VARIANT=check SUG_NVCC_EXTRA=-DSUG_CHECK=1): device-side asserts on every
// checkerboard index the kernels form (site, 8 neighbours, diagonal neighbour, halo copies) - the bounds check of
// our own that stands in for compute-sanitizer memcheck, which is closed on this pool (profiles/r02_sanitizers.md).
#if defined(SUG_CHECK) && SUG_CHECK
#include <cassert>
#define SUG_ASSERT(x) assert(x)
#else
#define SUG_ASSERT(x) ((void)0)
#endif

namespace sug {

enum : int { STORE_FULL = 0, STORE_RECON12 = 1, STORE_QUAT = 2 };
enum : int { KIND_HB = 0, KIND_OR = 1 };
enum : int { RNG_KP = 0, RNG_DIR = 1, RNG_HOT = 2 };
constexpr int KP_MAX_ATTEMPTS = 1024;   // reading R15
#ifndef SUG_KP_PRETEST
#define SUG_KP_PRETEST 1
#endif

template <class T> struct V2;
template <> struct V2<float>  { typedef float2  type; static __device__ __forceinline__ float2  make(float a, float b)   { return make_float2(a, b); } };
template <> struct V2<double> { typedef double2 type; static __device__ __forceinline__ double2 make(double a, double b) { return make_double2(a, b); } };

template <class T> struct cx { T re, im; };

template <class T> __device__ __forceinline__ cx<T> mk(T r, T i) { cx<T> c; c.re = r; c.im = i; return c; }
template <class T> __device__ __forceinline__ cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <class T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <class T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <class T> __device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b) { return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <class T> __device__ __forceinline__ cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.re, s * a.im); }
// acc += a b ; acc += a conj(b) ; acc += conj(a) b
template <class T> __device__ __forceinline__ void mad(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re += a.re * b.re; acc.re -= a.im * b.im; acc.im += a.re * b.im; acc.im += a.im * b.re;
}
template <class T> __device__ __forceinline__ void mad_cb(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re += a.re * b.re; acc.re += a.im * b.im; acc.im += a.im * b.re; acc.im -= a.re * b.im;
}
template <class T> __device__ __forceinline__ void mad_ca(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re += a.re * b.re; acc.re += a.im * b.im; acc.im += a.re * b.im; acc.im -= a.im * b.re;
}

// ------------------------------------------------------------------------------------------
// Geometry (readings R7): even extents, periodic, checkerboard index cb = i/2.
// ------------------------------------------------------------------------------------------
// sites per AoSoA tile of the link storage (32 = one warp-wide row per matrix element). Overridable for the layout
// ablation (profiles/r01f): 1 = array of structures, large = structure of arrays.
#ifndef SUG_LINK_TILE
#define SUG_LINK_TILE 32
#endif
constexpr int LINK_TILE = SUG_LINK_TILE;

struct Geom {
    int L[4];       // extents of the STORED lattice; L[3] includes the two halo time slices in slab mode
    int Lxh;        // Lx / 2
    unsigned Vh;    // stored sites per parity
    unsigned Vhp;   // Vh rounded up to a multiple of LINK_TILE = sites per stored plane
    int Zc;         // z-chunk of the update kernel's traversal order (divides Lz)
    // Block tiles of the register update kernels (su_set_option "block_tile"): the Wb warps
    // of a thread block work on the SAME 32-site x-y segments of Bz consecutive z-planes x Bt consecutive time slices
    // (Wb / (Bz Bt) consecutive segments each), so that links two of them need arrive in L1 once. Bz = Bt = 1: off
    // (a block is Wb consecutive segments of one plane). Only set in the copy a launch hands to k_update.
    int Bz, Bt, Wb;
    // t-slab decomposition: the handle owns Lt_int time slices of a global lattice of
    // Lt_glob slices and stores one halo slice below and above them (t_halo = 1). Without it: t_halo = 0,
    // Lt_int = L[3] = Lt_glob, t0g = 0 and the t direction wraps periodically inside the buffer.
    int t_halo;     // 0 or 1
    int Lt_int;     // interior (owned) time slices
    int Lt_glob;    // global time extent
    int t0g;        // global t of stored slice 0, in [0, Lt_glob)
    unsigned Vh_int;   // interior sites per parity = Lx Ly Lz Lt_int / 2
    unsigned Vsh;      // sites per parity of one time slice = Lx Ly Lz / 2
};

// parity of a stored site = parity of its GLOBAL coordinates (Lt_glob is even)
__device__ __forceinline__ int site_parity(const Geom& g, int x, int y, int z, int t_store) {
    return (x + y + z + t_store + g.t0g) & 1;
}
__device__ __forceinline__ int global_t(const Geom& g, int t_store) {
    const int t = t_store + g.t0g;             // can reach 2 Lt_glob (a single slab's upper halo)
    return t < g.Lt_glob ? t : t % g.Lt_glob;
}

__device__ __forceinline__ void decode_cb(const Geom& g, unsigned cb, int parity, int c[4]) {
    unsigned xh = cb % (unsigned)g.Lxh, r = cb / (unsigned)g.Lxh;
    c[1] = (int)(r % (unsigned)g.L[1]); r /= (unsigned)g.L[1];
    c[2] = (int)(r % (unsigned)g.L[2]);
    c[3] = (int)(r / (unsigned)g.L[2]);
    c[0] = 2 * (int)xh + ((c[1] + c[2] + c[3] + g.t0g + parity) & 1);
}
__device__ __forceinline__ unsigned cb_of(const Geom& g, int x, int y, int z, int t) {
    SUG_ASSERT(x >= 0 && x < g.L[0] && y >= 0 && y < g.L[1] && z >= 0 && z < g.L[2] && t >= 0 && t < g.L[3]);
    return (unsigned)(x >> 1) + (unsigned)g.Lxh * ((unsigned)y + (unsigned)g.L[1] * ((unsigned)z + (unsigned)g.L[2] * (unsigned)t));
}
// lexicographic index of a stored site in the GLOBAL lattice (the RNG counter word c0)
__device__ __forceinline__ unsigned lex_of(const Geom& g, const int c[4]) {
    return (unsigned)c[0] + (unsigned)g.L[0] * ((unsigned)c[1] + (unsigned)g.L[1] * ((unsigned)c[2] + (unsigned)g.L[2] * (unsigned)global_t(g, c[3])));
}
// checkerboard index of c + s1*e_{d1} + s2*e_{d2} (s in {-1,0,+1}), periodic wrap
__device__ __forceinline__ unsigned cb_shift(const Geom& g, const int c[4], int d1, int s1, int d2 = 0, int s2 = 0) {
    int n[4] = {c[0], c[1], c[2], c[3]};
    n[d1] += s1; if (n[d1] < 0) n[d1] += g.L[d1]; if (n[d1] >= g.L[d1]) n[d1] -= g.L[d1];
    n[d2] += s2; if (n[d2] < 0) n[d2] += g.L[d2]; if (n[d2] >= g.L[d2]) n[d2] -= g.L[d2];
    return cb_of(g, n[0], n[1], n[2], n[3]);
}

// ------------------------------------------------------------------------------------------
// Link I/O on the tiled structure-of-arrays layout
//     links[mu][parity][cb / 32][elem][cb % 32]   of (re,im) pairs:
// a warp reading one matrix element of 32 consecutive sites issues one coalesced 256 B (fp32) /
// 512 B (fp64) request, the E elements of a link sit at compile-time offsets e * 32 from one base
// address (one address computation per link instead of one per element), and the E rows of a
// tile are one contiguous E * 512 B piece of DRAM.
// ------------------------------------------------------------------------------------------
template <int NC, int STORE> struct LinkElems {
    static constexpr int E = (STORE == STORE_QUAT) ? 2 : ((STORE == STORE_RECON12) ? 6 : NC * NC);
};

template <class T> __device__ __forceinline__ void su3_third_row(cx<T>* m) {
    m[6] = conj(m[1] * m[5] - m[2] * m[4]);
    m[7] = conj(m[2] * m[3] - m[0] * m[5]);
    m[8] = conj(m[0] * m[4] - m[1] * m[3]);
}

// Load / store flavours: LD_PLAIN = ld.global (read-write data), LD_RO = ld.global.nc (neighbour links,
// read-only during a sub-step, kept in L1/L2 for re-use), LD_STREAM = ld.global.cs / st.global.cs (the
// link being updated: touched once per sub-step, so it should not displace re-used lines).
// LD_COHERENT = ld.relaxed.gpu (served by L2, never by a stale L1 line): links that another block may have
// rewritten earlier in the SAME launch (fused multi-sub-step launches, fused_schedule.h).
// LD_CG = ld.global.cg (cached in L2 only), LD_NA = ld.global.nc.L1::no_allocate (read-only path, no L1 line kept).
enum : int { LD_PLAIN = 0, LD_RO = 1, LD_STREAM = 2, LD_COHERENT = 3, LD_CG = 4, LD_NA = 5 };
__device__ __forceinline__ double2 ld_na(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_na(const float2* p) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ld_coherent(const double2* p) {
    double2 v;
    asm volatile("ld.relaxed.gpu.global.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ float2 ld_coherent(const float2* p) {
    float2 v;
    asm volatile("ld.relaxed.gpu.global.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p) : "memory");
    return v;
}
template <class T, int LD> __device__ __forceinline__ typename V2<T>::type ldg2(const typename V2<T>::type* p) {
    if (LD == LD_COHERENT) return ld_coherent(p);
    if (LD == LD_CG) return __ldcg(p);
    if (LD == LD_NA) return ld_na(p);
    return LD == LD_RO ? __ldg(p) : (LD == LD_STREAM ? __ldcs(p) : *p);
}
template <class T, bool STREAM> __device__ __forceinline__ void stg2(typename V2<T>::type* p, typename V2<T>::type v) {
    if (STREAM) __stcs(p, v); else *p = v;
}

template <int NC, class T, int STORE, bool UNR> struct LinkIO {
    typedef typename V2<T>::type T2;
    static constexpr int E = LinkElems<NC, STORE>::E;
    static_assert(STORE != STORE_QUAT || NC == 2, "quaternion storage is SU(2) only");
    static_assert(STORE != STORE_RECON12 || NC == 3, "two-row storage is SU(3) only");

    static __device__ __forceinline__ const T2* plane(const void* base, const Geom& g, int mu, int par) {
        return (const T2*)base + (size_t)(mu * 2 + par) * E * g.Vhp;
    }
    static __device__ __forceinline__ T2* plane(void* base, const Geom& g, int mu, int par) {
        return (T2*)base + (size_t)(mu * 2 + par) * E * g.Vhp;
    }
    // address of element 0 of site cb in a plane; element e is at + e * LINK_TILE
    static __device__ __forceinline__ const T2* site(const T2* pl, unsigned cb) {
        return pl + (size_t)(cb / LINK_TILE) * (E * LINK_TILE) + (cb % LINK_TILE);
    }
    static __device__ __forceinline__ T2* site(T2* pl, unsigned cb) {
        return pl + (size_t)(cb / LINK_TILE) * (E * LINK_TILE) + (cb % LINK_TILE);
    }
    template <int LD>
    static __device__ __forceinline__ void load(const T2* __restrict__ pl, unsigned cb, cx<T>* m) {
        pl = site(pl, cb);
        if (STORE == STORE_QUAT) {
            T2 v0 = ldg2<T, LD>(pl);
            T2 v1 = ldg2<T, LD>(pl + LINK_TILE);
            // eq 6: [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]], v0 = (a0,a1), v1 = (a2,a3)
            m[0] = mk<T>(v0.x, v1.y);  m[1] = mk<T>(v1.x, v0.y);
            m[2] = mk<T>(-v1.x, v0.y); m[3] = mk<T>(v0.x, -v1.y);
        } else {
#pragma unroll(UNR ? E : 1)
            for (int e = 0; e < E; ++e) {
                T2 v = ldg2<T, LD>(pl + e * LINK_TILE);
                m[e] = mk<T>(v.x, v.y);
            }
            if (STORE == STORE_RECON12) su3_third_row(m);
        }
    }
    // the E stored elements only (two-row storage: rows 0 and 1, no third-row reconstruction)
    template <int LD>
    static __device__ __forceinline__ void load_stored(const T2* __restrict__ pl, unsigned cb, cx<T>* m) {
        pl = site(pl, cb);
#pragma unroll(UNR ? E : 1)
        for (int e = 0; e < E; ++e) {
            T2 v = ldg2<T, LD>(pl + e * LINK_TILE);
            m[e] = mk<T>(v.x, v.y);
        }
    }
    template <bool STREAM = false>
    static __device__ __forceinline__ void store(T2* __restrict__ pl, unsigned cb, const cx<T>* m) {
        pl = site(pl, cb);
        if (STORE == STORE_QUAT) {
            stg2<T, STREAM>(pl,             V2<T>::make(m[0].re, m[1].im));
            stg2<T, STREAM>(pl + LINK_TILE, V2<T>::make(m[1].re, m[0].im));
        } else {
#pragma unroll(UNR ? E : 1)
            for (int e = 0; e < E; ++e) stg2<T, STREAM>(pl + e * LINK_TILE, V2<T>::make(m[e].re, m[e].im));
        }
    }
};

// ------------------------------------------------------------------------------------------
// Nc x Nc complex products, row-major. UNR: full unroll (registers) or rolled loops (local arrays).
// ------------------------------------------------------------------------------------------
template <int NC, class T, bool UNR> struct Mat {
    typedef cx<T> C;
    // O = A B
    static __device__ __forceinline__ void mul_nn(const C* A, const C* B, C* O) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i)
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad(s, A[i * NC + k], B[k * NC + j]);
                O[i * NC + j] = s;
            }
    }
    // O = A^dagger B
    static __device__ __forceinline__ void mul_dn(const C* A, const C* B, C* O) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i)
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_ca(s, A[k * NC + i], B[k * NC + j]);
                O[i * NC + j] = s;
            }
    }
    // O = A B^dagger
    static __device__ __forceinline__ void mul_nd(const C* A, const C* B, C* O) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i)
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_cb(s, A[i * NC + k], B[j * NC + k]);
                O[i * NC + j] = s;
            }
    }
    // S += A B
    static __device__ __forceinline__ void acc_nn(C* S, const C* A, const C* B) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i)
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = S[i * NC + j];
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad(s, A[i * NC + k], B[k * NC + j]);
                S[i * NC + j] = s;
            }
    }
    // S += A B^dagger
    static __device__ __forceinline__ void acc_nd(C* S, const C* A, const C* B) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i)
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = S[i * NC + j];
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_cb(s, A[i * NC + k], B[j * NC + k]);
                S[i * NC + j] = s;
            }
    }
    // S += (A B) C^dagger, one row of A B at a time: only B, C and S stay live across the rows, so the
    // loads of all three operands can be issued before the first product.
    // Same operation order per element as mul_nn followed by acc_nd.
    static __device__ __forceinline__ void acc_nnd(C* S, const C* A, const C* B, const C* D) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i) {
            C r[NC];
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad(s, A[i * NC + k], B[k * NC + j]);
                r[j] = s;
            }
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = S[i * NC + j];
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_cb(s, r[k], D[j * NC + k]);
                S[i * NC + j] = s;
            }
        }
    }
    // S += (A^dagger B) C, row by row; same operation order per element as mul_dn followed by acc_nn
    static __device__ __forceinline__ void acc_dnn(C* S, const C* A, const C* B, const C* D) {
#pragma unroll(UNR ? NC : 1)
        for (int i = 0; i < NC; ++i) {
            C r[NC];
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_ca(s, A[k * NC + i], B[k * NC + j]);
                r[j] = s;
            }
#pragma unroll(UNR ? NC : 1)
            for (int j = 0; j < NC; ++j) {
                C s = S[i * NC + j];
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad(s, r[k], D[k * NC + j]);
                S[i * NC + j] = s;
            }
        }
    }
    // B <- A^dagger B in place, column by column (column j of the product needs column j of B only); same sums as mul_dn
    static __device__ __forceinline__ void mul_dn_inplace(const C* A, C* B) {
#pragma unroll(UNR ? NC : 1)
        for (int j = 0; j < NC; ++j) {
            C col[NC];
#pragma unroll(UNR ? NC : 1)
            for (int i = 0; i < NC; ++i) {
                C s = mk<T>(0, 0);
#pragma unroll(UNR ? NC : 1)
                for (int k = 0; k < NC; ++k) mad_ca(s, A[k * NC + i], B[k * NC + j]);
                col[i] = s;
            }
#pragma unroll(UNR ? NC : 1)
            for (int i = 0; i < NC; ++i) B[i * NC + j] = col[i];
        }
    }
    // Re Tr (A B^dagger) = sum_ij Re(A_ij conj(B_ij))
    static __device__ __forceinline__ T retr_nd(const C* A, const C* B) {
        T s = 0;
#pragma unroll(UNR ? NC * NC : 1)
        for (int e = 0; e < NC * NC; ++e) s += A[e].re * B[e].re + A[e].im * B[e].im;
        return s;
    }
    static __device__ __forceinline__ void zero(C* S) {
#pragma unroll(UNR ? NC * NC : 1)
        for (int e = 0; e < NC * NC; ++e) S[e] = mk<T>(0, 0);
    }
};

// ------------------------------------------------------------------------------------------
// SU(3) staple terms on two-row operands (12-real storage): a product of SU(3) matrices is in SU(3),
// so only rows 0 and 1 of a three-link product are multiplied out and its third row is the conjugate cross
// product of those, exactly as for a stored link. An operand's third row is rebuilt only where the product sums
// over it. Per term: 2 x 72 multiply-adds + 3 (upper) or 4 (lower) third rows of 24, against 216 + 3 x 24 when
// every loaded link is completed first.
// ------------------------------------------------------------------------------------------
template <class T> struct Su3Rows {
    typedef cx<T> C;
    // S += (A B) C^dagger, A: rows 0,1; B, C: rows 0,1 stored, row 2 rebuilt here (B[6..8], C[6..8] are scratch)
    static __device__ __forceinline__ void acc_upper(C* S, const C* A, C* B, C* D) {
        su3_third_row(B);
        su3_third_row(D);
        C P[9];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            C r[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll
                for (int k = 0; k < 3; ++k) mad(s, A[i * 3 + k], B[k * 3 + j]);
                r[j] = s;
            }
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll
                for (int k = 0; k < 3; ++k) mad_cb(s, r[k], D[j * 3 + k]);
                P[i * 3 + j] = s;
            }
        }
        su3_third_row(P);
#pragma unroll
        for (int e = 0; e < 9; ++e) S[e] = S[e] + P[e];
    }
    // S += (A^dagger B) C, all three operands: rows 0,1 stored, row 2 rebuilt here
    static __device__ __forceinline__ void acc_lower(C* S, C* A, C* B, C* D) {
        su3_third_row(A);
        su3_third_row(B);
        su3_third_row(D);
        C P[9];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            C r[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll
                for (int k = 0; k < 3; ++k) mad_ca(s, A[k * 3 + i], B[k * 3 + j]);
                r[j] = s;
            }
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                C s = mk<T>(0, 0);
#pragma unroll
                for (int k = 0; k < 3; ++k) mad(s, r[k], D[k * 3 + j]);
                P[i * 3 + j] = s;
            }
        }
        su3_third_row(P);
#pragma unroll
        for (int e = 0; e < 9; ++e) S[e] = S[e] + P[e];
    }
};

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11): counter (c0..c3), key (k0,k1), 10 rounds.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// uniform in (0,1], exact in T: fp64 (w+1)/2^32, fp32 ((w>>8)+1)/2^24
template <class T> __device__ __forceinline__ T uniform01(uint32_t w);
template <> __device__ __forceinline__ double uniform01<double>(uint32_t w) { return ((double)w + 1.0) * (1.0 / 4294967296.0); }
template <> __device__ __forceinline__ float  uniform01<float >(uint32_t w) { return ((float)(w >> 8) + 1.0f) * (1.0f / 16777216.0f); }

// Counter word c2 = kind<<28 | pass<<20 | parity<<19 | mu<<17 | subgroup. pack_c2 fills
// the low 28 bits; the stream kind (RNG_KP / RNG_DIR / RNG_HOT) is ORed in by c2_kind where a block is drawn.
__device__ __forceinline__ uint32_t pack_c2(int pass, int parity, int mu, int subgroup) {
    return ((uint32_t)(pass & 0xff) << 20) | ((uint32_t)parity << 19) | ((uint32_t)mu << 17) | (uint32_t)subgroup;
}
__device__ __forceinline__ uint32_t c2_kind(uint32_t c2_low, int kind) { return c2_low | ((uint32_t)kind << 28); }

// ------------------------------------------------------------------------------------------
// Branch-free fp64 elementary functions for the Kennedy-Pendleton draw (-DSUG_FAST_MATH64=0: libdevice instead).
// The draw needs ln u, cos 2 pi u, sincos 2 pi u for u = (w + 1) / 2^32 with w a 32-bit Philox word, and square roots
// of numbers in [0, 1] / positive norms: no special cases, so no branches or slow-path calls - libdevice's versions
// carry both, which keeps the compiler from interleaving the chains of independent draws with each other or with loads
// (profiles/r02a, r02g). Accuracy <= 1 ulp-level (2.2e-16 relative for ln, 1.8e-16 absolute for sin / cos: checked against
// long double on 2^24 words and the edge words by tests/test_gpu_parity.py::test_fast_math_against_host).
// ------------------------------------------------------------------------------------------
#ifndef SUG_FAST_MATH64
#define SUG_FAST_MATH64 1
#endif
__device__ __forceinline__ double rcp_approx64(double x) { double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
__device__ __forceinline__ double rsqrt_approx64(double x) { double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }

// ln((w + 1) / 2^32): n = w + 1 = m 2^e with m in [sqrt(1/2), sqrt 2], ln m = 2 atanh(s), s = (m - 1) / (m + 1), by its
// Taylor series to s^21 (|s| <= 0.172: next term 2e-17 relative), the division by a Newton-refined reciprocal.
__device__ __forceinline__ double fast_log_u01(uint32_t w) {
    const double n = (__hiloint2double(0x43300000, (int)w) - 4503599627370496.0) + 1.0;      // exact: 1 ... 2^32
    const int hi = __double2hiint(n), lo = __double2loint(n);
    int e = (hi >> 20) - 1023;
    int mh = (hi & 0x000fffff) | 0x3ff00000;
    const int big = mh > 0x3ff6a09e ? 1 : 0;                        // m > sqrt 2 (to 2^-20): halve it
    mh -= big << 20; e += big;
    const double f = __hiloint2double(mh, lo) - 1.0, d = 2.0 + f;
    double r = rcp_approx64(d);
    r = __fma_rn(r, __fma_rn(-d, r, 1.0), r);
    r = __fma_rn(r, __fma_rn(-d, r, 1.0), r);
    double sq = f * r;
    sq = __fma_rn(__fma_rn(-d, sq, f), r, sq);
    const double z = sq * sq;
    double P = 0.09523809523809523;                                 // 2 / 21
    P = __fma_rn(P, z, 0.10526315789473684);
    P = __fma_rn(P, z, 0.11764705882352941);
    P = __fma_rn(P, z, 0.13333333333333333);
    P = __fma_rn(P, z, 0.15384615384615385);
    P = __fma_rn(P, z, 0.18181818181818182);
    P = __fma_rn(P, z, 0.2222222222222222);
    P = __fma_rn(P, z, 0.2857142857142857);
    P = __fma_rn(P, z, 0.4);
    P = __fma_rn(P, z, 0.6666666666666666);
    const double k = (double)(e - 32);
    // k ln2_hi is exact (ln2_hi has 32 trailing zero bits)
    return __fma_rn(k, 6.93147180369123816490e-01, __fma_rn(2.0, sq, __fma_rn(sq * z, P, k * 1.90821492927058770002e-10)));
}
// sin and cos of 2 pi (w + 1) / 2^32: the angle is an exact 32-bit fraction of the circle, so the quadrant and the
// remainder theta in [-pi/4, pi/4) come from integer arithmetic; Taylor series to theta^17 / theta^18.
__device__ __forceinline__ void fast_sincos2pi_u01(uint32_t w, double* sn, double* cs) {
    const uint32_t kp = (w + 1u) + 0x20000000u;
    const int q = (int)(kp >> 30), ri = (int)(kp & 0x3fffffffu) - 0x20000000;
    const double th = (double)ri * 1.4629180792671596e-09, t2 = th * th;      // pi / 2^31
    double S = 2.8114572543455206e-15;                              // 1 / 17!
    S = __fma_rn(S, t2, -7.647163731819816e-13);                    // -1 / 15!
    S = __fma_rn(S, t2, 1.6059043836821613e-10);                    // 1 / 13!
    S = __fma_rn(S, t2, -2.505210838544172e-08);                    // -1 / 11!
    S = __fma_rn(S, t2, 2.7557319223985893e-06);                    // 1 / 9!
    S = __fma_rn(S, t2, -0.0001984126984126984);                    // -1 / 7!
    S = __fma_rn(S, t2, 0.008333333333333333);                      // 1 / 5!
    S = __fma_rn(S, t2, -0.16666666666666666);                      // -1 / 3!
    S = __fma_rn(S * t2, th, th);
    double Cc = -1.5619206968586225e-16;                            // -1 / 18!
    Cc = __fma_rn(Cc, t2, 4.779477332387385e-14);                   // 1 / 16!
    Cc = __fma_rn(Cc, t2, -1.1470745597729725e-11);                 // -1 / 14!
    Cc = __fma_rn(Cc, t2, 2.08767569878681e-09);                    // 1 / 12!
    Cc = __fma_rn(Cc, t2, -2.755731922398589e-07);                  // -1 / 10!
    Cc = __fma_rn(Cc, t2, 2.48015873015873e-05);                    // 1 / 8!
    Cc = __fma_rn(Cc, t2, -0.001388888888888889);                   // -1 / 6!
    Cc = __fma_rn(Cc, t2, 0.041666666666666664);                    // 1 / 4!
    Cc = __fma_rn(Cc, t2, -0.5);
    Cc = __fma_rn(Cc, t2, 1.0);
    const double a = (q & 1) ? Cc : S, b = (q & 1) ? S : Cc;        // sin, cos of the quadrant-rotated angle, up to sign
    *sn = (q & 2) ? -a : a;
    *cs = ((q + 1) & 2) ? -b : b;
}
// sqrt(x) for 0 <= x <~ 1e300 and 1 / sqrt(x) for x > 0 (normal range): rsqrt seed + two coupled Newton steps + one correction
__device__ __forceinline__ double fast_sqrt64(double x) {
    const double xs = fmax(x, 1e-300);                              // sqrt(0) -> 1e-150, below anything it is added to
    const double y = rsqrt_approx64(xs);
    double g = xs * y, h = 0.5 * y, r = __fma_rn(-h, g, 0.5);
    g = __fma_rn(g, r, g); h = __fma_rn(h, r, h);
    r = __fma_rn(-h, g, 0.5);
    g = __fma_rn(g, r, g); h = __fma_rn(h, r, h);
    return __fma_rn(__fma_rn(-g, g, xs), h, g);
}
// 1 / x for x > 0 in the normal range: reciprocal seed + two Newton steps (<= 1 ulp), no slow path
__device__ __forceinline__ double fast_rcp64(double x) {
    double r = rcp_approx64(x);
    r = __fma_rn(r, __fma_rn(-x, r, 1.0), r);
    r = __fma_rn(r, __fma_rn(-x, r, 1.0), r);
    return r;
}
__device__ __forceinline__ double fast_rsqrt64(double x) {
    const double y = rsqrt_approx64(x);
    double g = x * y, h = 0.5 * y, r = __fma_rn(-h, g, 0.5);
    g = __fma_rn(g, r, g); h = __fma_rn(h, r, h);
    r = __fma_rn(-h, g, 0.5);
    h = __fma_rn(h, r, h);
    return 2.0 * h;
}

template <class T> struct Fn;
template <> struct Fn<float> {
    static __device__ __forceinline__ float log(float x) { return logf(x); }
    static __device__ __forceinline__ float cos(float x) { return cosf(x); }
    static __device__ __forceinline__ float sqrt(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float rsqrt(float x) { return rsqrtf(x); }
    static __device__ __forceinline__ void sincos(float x, float* s, float* c) { sincosf(x, s, c); }
    // cos / sincos of 2 pi u for u in (0,1]: the pi-scaled forms need no range reduction of an irrational multiple
    static __device__ __forceinline__ float cos2pi(float u) { return cospif(2.0f * u); }
    static __device__ __forceinline__ void sincos2pi(float u, float* s, float* c) { sincospif(2.0f * u, s, c); }
    // of the uniform of a Philox word (uniform01<float>): ln u, cos 2 pi u, sincos 2 pi u
    static __device__ __forceinline__ float log_w(uint32_t w) { return logf(((float)(w >> 8) + 1.0f) * (1.0f / 16777216.0f)); }
    static __device__ __forceinline__ float cos2pi_w(uint32_t w) { return cospif(2.0f * (((float)(w >> 8) + 1.0f) * (1.0f / 16777216.0f))); }
    static __device__ __forceinline__ void sincos2pi_w(uint32_t w, float* s, float* c) { sincospif(2.0f * (((float)(w >> 8) + 1.0f) * (1.0f / 16777216.0f)), s, c); }
    static __device__ __forceinline__ float sqrt01(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float rsqrt_pos(float x) { return rsqrtf(x); }
    static __device__ __forceinline__ float rcp_pos(float x) { return 1.0f / x; }
    static __device__ __forceinline__ float max0(float x) { return fmaxf(x, 0.0f); }
    static __device__ __forceinline__ bool finite(float x) { return isfinite(x); }
    // smallest k^2 a subgroup update is carried out for (see update_subgroups): below it 1 / k^2 overflows
    static __device__ __forceinline__ float min_norm2() { return 1.17549435e-38f; }      // FLT_MIN
};
template <> struct Fn<double> {
    static __device__ __forceinline__ double log(double x) { return ::log(x); }
    static __device__ __forceinline__ double cos(double x) { return ::cos(x); }
    static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
    static __device__ __forceinline__ double rsqrt(double x) { return ::rsqrt(x); }
    static __device__ __forceinline__ void sincos(double x, double* s, double* c) { ::sincos(x, s, c); }
    static __device__ __forceinline__ double cos2pi(double u) { return ::cospi(2.0 * u); }
    static __device__ __forceinline__ void sincos2pi(double u, double* s, double* c) { ::sincospi(2.0 * u, s, c); }
#if SUG_FAST_MATH64
    static __device__ __forceinline__ double log_w(uint32_t w) { return fast_log_u01(w); }
    static __device__ __forceinline__ double cos2pi_w(uint32_t w) { double s, c; fast_sincos2pi_u01(w, &s, &c); return c; }
    static __device__ __forceinline__ void sincos2pi_w(uint32_t w, double* s, double* c) { fast_sincos2pi_u01(w, s, c); }
    static __device__ __forceinline__ double sqrt01(double x) { return fast_sqrt64(x); }
    static __device__ __forceinline__ double rsqrt_pos(double x) { return fast_rsqrt64(x); }
    static __device__ __forceinline__ double rcp_pos(double x) { return fast_rcp64(x); }
#else
    static __device__ __forceinline__ double log_w(uint32_t w) { return ::log(((double)w + 1.0) * (1.0 / 4294967296.0)); }
    static __device__ __forceinline__ double cos2pi_w(uint32_t w) { return ::cospi(2.0 * (((double)w + 1.0) * (1.0 / 4294967296.0))); }
    static __device__ __forceinline__ void sincos2pi_w(uint32_t w, double* s, double* c) { ::sincospi(2.0 * (((double)w + 1.0) * (1.0 / 4294967296.0)), s, c); }
    static __device__ __forceinline__ double sqrt01(double x) { return ::sqrt(x); }
    static __device__ __forceinline__ double rsqrt_pos(double x) { return ::rsqrt(x); }
    static __device__ __forceinline__ double rcp_pos(double x) { return 1.0 / x; }
#endif
    static __device__ __forceinline__ double max0(double x) { return fmax(x, 0.0); }
    static __device__ __forceinline__ bool finite(double x) { return isfinite(x); }
    // smallest k^2 a subgroup update is carried out for: rcp / rsqrt.approx.ftz.f64 (the seeds of fast_rcp64 and
    // fast_rsqrt64) flush a subnormal argument to zero and the Newton steps then turn the infinite seed into NaN
    static __device__ __forceinline__ double min_norm2() { return 2.2250738585072014e-308; }      // DBL_MIN
};

// Kennedy-Pendleton draw of v = (a0, a): P(a0) ~ sqrt(1-a0^2) exp(alpha a0) (eq 13),
// a uniform on the sphere of radius sqrt(1-a0^2). Returns attempts used, 0 = none.
// m_inv2a = -1 / (2 alpha), supplied by the caller (it has 1/k already).
//
// fp64: the accept test r4^2 <= 1 - lambda^2  <=>  M = 2 alpha (1 - r4^2) + ln r1 + cos^2(2 pi r2) ln r3 >= 0
// is first evaluated in fp32 with the SFU approximations (|error of M| < 1e-4 + 2 alpha 5e-7). Only when
// |M| is inside a 10x wider band is the decision taken with the exact fp64 expression, so the decision is
// always the fp64 one, and the accepted attempt's lambda^2 is then evaluated in fp64 once, after the
// loop, by the whole warp together (a warp would otherwise run the fp64 log/log/cos body for every
// attempt any of its lanes needs: 1.9 times per draw at beta = 6 instead of once).
// Direction of the heatbath vector: a point uniform on the unit sphere from the "direction"
// Philox block of the draw. It does not depend on the links, so a kernel may evaluate it ahead of the
// staple (in the shadow of the first loads) and hand it to kp_draw.
template <class T>
__device__ __forceinline__ void kp_direction(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2_base, T n[3]) {
    uint32_t d[4];
    philox4x32_10(c0, c1, c2_kind(c2_base, RNG_DIR), 0u, k0, k1, d);
    const T u1 = uniform01<T>(d[0]);
    const T cos_t = (T)1 - (T)2 * u1;
    const T sin_t = Fn<T>::sqrt01(Fn<T>::max0((T)1 - cos_t * cos_t));
    T sp, cp;
    Fn<T>::sincos2pi_w(d[1], &sp, &cp);
    n[0] = sin_t * cp; n[1] = sin_t * sp; n[2] = cos_t;
}

// The link-independent part of attempt 0 of a draw: Q = ln r1 + cos^2(2 pi r2) ln r3 and R = r4^2, so that
// lambda^2 = -Q / (2 alpha) and the attempt is accepted iff R <= 1 - lambda^2 - the same expressions, in the
// same order and precision, as in the accept loop of kp_draw. A kernel evaluates this for all the subgroups of
// its link before the staple (with the Philox blocks of the subgroups interleaved, in the shadow of the first
// loads) and hands it to kp_draw as pre0 = {Q, R} at stride dir_stride; attempts >= 1 (a few percent of the
// draws) still run the loop.
template <class T>
__device__ __forceinline__ void kp_attempt0(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2_base, T& Q, T& R) {
    uint32_t w[4];
    philox4x32_10(c0, c1, c2_kind(c2_base, RNG_KP), 0u, k0, k1, w);
    const T r4 = uniform01<T>(w[3]);
    const T c = Fn<T>::cos2pi_w(w[1]);
    Q = Fn<T>::log_w(w[0]) + c * c * Fn<T>::log_w(w[2]);
    R = r4 * r4;
}

template <class T>
__device__ __forceinline__ int kp_draw(unsigned draw_mask, T alpha, T m_inv2a, uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                       uint32_t c2_base, T v[4], const T* dir = nullptr, int dir_stride = 0,
                                       const T* pre0 = nullptr) {
    const bool drawable = (alpha > (T)0) && Fn<T>::finite(alpha);
    const unsigned converged = __ballot_sync(draw_mask, drawable);
    if (!drawable) return 0;
    constexpr bool PRETEST = (sizeof(T) == 8) && (SUG_KP_PRETEST != 0);
    const float two_af = 2.0f * (float)alpha;
    const float band = 1e-3f + two_af * 4e-6f;
    T a0 = 0;
    int used = 0;
    uint32_t w[4];
    // attempt 0 precomputed by kp_attempt0 (link-independent part): only the scale by -1/(2 alpha) and the test remain
    bool from_pre = false;
    if (pre0) {
        const T lambda2 = pre0[0] * m_inv2a;
        if (pre0[dir_stride] <= (T)1 - lambda2) { a0 = (T)1 - (T)2 * lambda2; used = 1; from_pre = true; }
    }
    // lanes leave the accept loop after different numbers of attempts; without an explicit barrier the
    // compiler lets every exit group run the rest of the draw on its own (ncu: the direction part ran 1.6x
    // per warp). draw_mask = the lanes that call kp_draw for this subgroup, balloted by the caller BEFORE its
    // divergent branch (all of them reach the barrier: the early return above is taken before the loop by
    // lanes that then skip it, so they are excluded here).
    for (int n = pre0 ? 1 : 0; !from_pre && n < KP_MAX_ATTEMPTS; ++n) {
        philox4x32_10(c0, c1, c2_kind(c2_base, RNG_KP), (uint32_t)n, k0, k1, w);
        if (PRETEST) {
            const float S = 2.3283064365386963e-10f;      // 2^-32
            const float r1f = (__uint2float_rn(w[0]) + 1.0f) * S, r2f = (__uint2float_rn(w[1]) + 1.0f) * S;
            const float r3f = (__uint2float_rn(w[2]) + 1.0f) * S, r4f = (__uint2float_rn(w[3]) + 1.0f) * S;
            const float cf = __cosf(6.2831853071795865f * r2f);
            const float M = two_af * (1.0f - r4f * r4f) + (__logf(r1f) + cf * cf * __logf(r3f));
            if (M > band) { used = n + 1; break; }
            if (M < -band) continue;
        }
        T r4 = uniform01<T>(w[3]);
        T c = Fn<T>::cos2pi_w(w[1]);
        T lambda2 = (Fn<T>::log_w(w[0]) + c * c * Fn<T>::log_w(w[2])) * m_inv2a;
        if (r4 * r4 <= (T)1 - lambda2) { a0 = (T)1 - (T)2 * lambda2; used = n + 1; break; }
    }
    __syncwarp(converged);
    if (!used) return 0;
    if (PRETEST && !from_pre) {
        T c = Fn<T>::cos2pi_w(w[1]);
        T lambda2 = (Fn<T>::log_w(w[0]) + c * c * Fn<T>::log_w(w[2])) * m_inv2a;
        a0 = (T)1 - (T)2 * lambda2;
    }
    T n[3];
    if (dir) { n[0] = dir[0]; n[1] = dir[dir_stride]; n[2] = dir[2 * dir_stride]; }
    else kp_direction<T>(k0, k1, c0, c1, c2_base, n);
    const T rho = Fn<T>::sqrt01(Fn<T>::max0((T)1 - a0 * a0));
    v[0] = a0; v[1] = rho * n[0]; v[2] = rho * n[1]; v[3] = rho * n[2];
    return used;
}

// Explicitly fused / unfused scalar operations. Where an expression a b + c d leaves the compiler a choice of which
// product to fuse, two instances of the same source (plain, fused and cooperative kernels) can round differently in
// the last bit; the few such expressions of the update are written with these so that every instance is bitwise the same.
__device__ __forceinline__ float  fma_x(float a, float b, float c)    { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_x(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float  mul_x(float a, float b)   { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_x(double a, double b) { return __dmul_rn(a, b); }
// a0^2 + a1^2 + a2^2 + a3^2, summed left to right
template <class T> __device__ __forceinline__ T norm2_4(T a0, T a1, T a2, T a3) {
    return fma_x(a3, a3, fma_x(a2, a2, fma_x(a1, a1, mul_x(a0, a0))));
}

// quaternion product, U = a0 + i a.sigma (eq 6): (ab)_0 = a0 b0 - a.b, (ab)_vec = a0 b + b0 a - a x b
template <class T> __device__ __forceinline__ void quat_mul(const T a[4], const T b[4], T o[4]) {
    o[0] = fma_x(-a[3], b[3], fma_x(-a[2], b[2], fma_x(-a[1], b[1], mul_x(a[0], b[0]))));
    o[1] = fma_x(a[3], b[2], fma_x(-a[2], b[3], fma_x(b[0], a[1], mul_x(a[0], b[1]))));
    o[2] = fma_x(a[1], b[3], fma_x(-a[3], b[1], fma_x(b[0], a[2], mul_x(a[0], b[2]))));
    o[3] = fma_x(a[2], b[1], fma_x(-a[1], b[2], fma_x(b[0], a[3], mul_x(a[0], b[3]))));
}

// ------------------------------------------------------------------------------------------
// Steps 3-5 of the Cabibbo-Marinari procedure on one link (eqs 11-17): every
// SU(2) subgroup (i<j), lexicographic (reading R5): project the 2x2 block of W, heatbath
// (alpha = 2 beta k / Nc, reading R3) or overrelaxation, left-multiply rows i,j of U and W (eq 15).
// att: attempts per subgroup (NULL ok). Returns (attempts_total, exhausted) packed: lo 24 bits / hi 8.
// ------------------------------------------------------------------------------------------
template <int NC, class T, int KIND, bool UNR>
__device__ __forceinline__ void update_subgroups(cx<T>* U, cx<T>* W, T beta, uint32_t k0, uint32_t k1,
                                                 uint32_t c0, uint32_t c1, uint32_t c2_base,
                                                 uint8_t* att_out, size_t att_stride,
                                                 unsigned& att_total, unsigned& exhausted, unsigned warp_mask,
                                                 const T* dirs = nullptr, int dir_stride = 0, const T* pre = nullptr) {
    // warp_mask: the lanes of this warp that run the subgroup loop (balloted by the kernel where all of them
    // are converged); every one of them executes the ballots below, subgroup by subgroup
    int q = 0;
    const T two_beta_over_nc = (T)2 * beta / (T)NC;      // alpha = 2 beta k / Nc (reading R3)
    const T m_nc_over_4beta = (T)-0.25 * (T)NC / beta;   // -1 / (2 alpha) = this / k   (heatbath only)
#pragma unroll(UNR ? NC : 1)
    for (int i = 0; i < NC - 1; ++i) {
#pragma unroll(UNR ? NC : 1)
        for (int j = i + 1; j < NC; ++j, ++q) {
            const cx<T> wii = W[i * NC + i], wij = W[i * NC + j], wji = W[j * NC + i], wjj = W[j * NC + j];
            T r0 = (T)0.5 * (wii.re + wjj.re), r1 = (T)0.5 * (wij.im + wji.im);
            T r2 = (T)0.5 * (wij.re - wji.re), r3 = (T)0.5 * (wii.im - wjj.im);
            const T n2 = norm2_4(r0, r1, r2, r3);                        // k^2
            // k = 0 leaves the subgroup unchanged (reading R15); so does a k^2 below the normal range, where 1 / k and
            // 1 / k^2 are not representable (or not computable by the fast reciprocals): such a block carries no weight
            bool ok = (n2 >= Fn<T>::min_norm2()) && Fn<T>::finite(n2);
            T a[4] = {(T)1, (T)0, (T)0, (T)0};
            int used = 0;
            const unsigned draw_mask = (KIND == KIND_HB) ? __ballot_sync(warp_mask, ok) : 0u;
            if (ok) {
                if (KIND == KIND_HB) {
                    const T ik = Fn<T>::rsqrt_pos(n2), k = n2 * ik;      // 1/k and k without a division
                    T ud[4] = {r0 * ik, -r1 * ik, -r2 * ik, -r3 * ik};
                    T v[4];
                    used = kp_draw<T>(draw_mask, two_beta_over_nc * k, m_nc_over_4beta * ik, k0, k1, c0, c1,
                                      c2_base | (uint32_t)q, v, dirs ? dirs + 3 * q * dir_stride : nullptr, dir_stride,
                                      pre ? pre + 2 * q * dir_stride : nullptr);
                    if (used) quat_mul(v, ud, a); else ok = false;
                } else {
                    // a = (u~^dagger)^2 = conj(r)^2 / k^2 (eq 17): no square root, one reciprocal
                    const T in2 = Fn<T>::rcp_pos(n2), m2r0 = (T)-2 * r0 * in2;
                    a[0] = fma_x(r0, r0, -fma_x(r3, r3, fma_x(r2, r2, mul_x(r1, r1)))) * in2;
                    a[1] = m2r0 * r1; a[2] = m2r0 * r2; a[3] = m2r0 * r3;
                }
            }
            if (KIND == KIND_HB) {
                att_total += (unsigned)used;
                if (!ok) exhausted += 1u;
                if (att_out) att_out[(size_t)q * att_stride] = (uint8_t)(used > 255 ? 255 : used);
            }
            if (ok) {
                const cx<T> a00 = mk<T>(a[0], a[3]), a01 = mk<T>(a[2], a[1]);
                const cx<T> a10 = mk<T>(-a[2], a[1]), a11 = mk<T>(a[0], -a[3]);
#pragma unroll(UNR ? NC : 1)
                for (int c = 0; c < NC; ++c) {
                    cx<T> ui = U[i * NC + c], uj = U[j * NC + c];
                    U[i * NC + c] = a00 * ui + a01 * uj;
                    U[j * NC + c] = a10 * ui + a11 * uj;
                    cx<T> wi = W[i * NC + c], wj = W[j * NC + c];
                    W[i * NC + c] = a00 * wi + a01 * wj;
                    W[j * NC + c] = a10 * wi + a11 * wj;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Gram-Schmidt / determinant on a local matrix (rolled loops), used by reunitarise (Nc >= 4)
// and by the hot start (always double, reading R20).
// ------------------------------------------------------------------------------------------
template <int NC, class R, bool UNR = false>
__device__ __forceinline__ void gram_schmidt_rows(cx<R>* U, int nrows) {
#pragma unroll(UNR ? NC : 1)
    for (int r = 0; r < (UNR ? NC : nrows); ++r) {
#pragma unroll(UNR ? NC : 1)
        for (int p = 0; p < r; ++p) {
            cx<R> dot = mk<R>(0, 0);
#pragma unroll(UNR ? NC : 1)
            for (int k = 0; k < NC; ++k) mad_ca(dot, U[p * NC + k], U[r * NC + k]);
#pragma unroll(UNR ? NC : 1)
            for (int k = 0; k < NC; ++k) U[r * NC + k] = U[r * NC + k] - dot * U[p * NC + k];
        }
        R n2 = 0;
#pragma unroll(UNR ? NC : 1)
        for (int k = 0; k < NC; ++k) n2 += U[r * NC + k].re * U[r * NC + k].re + U[r * NC + k].im * U[r * NC + k].im;
        R inv = (R)1 / Fn<R>::sqrt(n2);
#pragma unroll(UNR ? NC : 1)
        for (int k = 0; k < NC; ++k) U[r * NC + k] = inv * U[r * NC + k];
    }
}

// det of a 4x4 complex matrix by the 2x2-minor (Laplace) expansion over rows {0,1} x {2,3}: no pivoting,
// no dynamic indexing, so it stays in registers (used for the phase conj(det)/|det| only).
template <class R>
__device__ __forceinline__ cx<R> determinant4(const cx<R>* A) {
    const cx<R> s0 = A[0] * A[5] - A[1] * A[4], s1 = A[0] * A[6] - A[2] * A[4], s2 = A[0] * A[7] - A[3] * A[4];
    const cx<R> s3 = A[1] * A[6] - A[2] * A[5], s4 = A[1] * A[7] - A[3] * A[5], s5 = A[2] * A[7] - A[3] * A[6];
    const cx<R> c5 = A[10] * A[15] - A[11] * A[14], c4 = A[9] * A[15] - A[11] * A[13], c3 = A[9] * A[14] - A[10] * A[13];
    const cx<R> c2 = A[8] * A[15] - A[11] * A[12], c1 = A[8] * A[14] - A[10] * A[12], c0 = A[8] * A[13] - A[9] * A[12];
    return (s0 * c5 - s1 * c4) + (s2 * c3 + s3 * c2) + (s5 * c0 - s4 * c1);
}

// SU(3) rows 0,1 by modified Gram-Schmidt in registers (same operation order as gram_schmidt_rows)
template <class T>
__device__ __forceinline__ void gram_schmidt_su3_two_rows(cx<T>* U) {
    T n2 = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) n2 += U[k].re * U[k].re + U[k].im * U[k].im;
    T inv = (T)1 / Fn<T>::sqrt(n2);
#pragma unroll
    for (int k = 0; k < 3; ++k) U[k] = inv * U[k];
    cx<T> dot = mk<T>(0, 0);
#pragma unroll
    for (int k = 0; k < 3; ++k) mad_ca(dot, U[k], U[3 + k]);
#pragma unroll
    for (int k = 0; k < 3; ++k) U[3 + k] = U[3 + k] - dot * U[k];
    n2 = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) n2 += U[3 + k].re * U[3 + k].re + U[3 + k].im * U[3 + k].im;
    inv = (T)1 / Fn<T>::sqrt(n2);
#pragma unroll
    for (int k = 0; k < 3; ++k) U[3 + k] = inv * U[3 + k];
}

// Reunitarisation of one link in registers, Nc <= 4 (reading R10): SU(2) normalise the first row
// (a0, a1, a2, a3) and rebuild the second, SU(3) Gram-Schmidt on rows 0, 1 + cross product, SU(4) Gram-Schmidt +
// phase of the determinant on the last row. Used by k_reunit and, on request, by the update kernels right before
// they store (su_set_option "reunit_on_store").
template <int NC, class T>
__device__ __forceinline__ void reunitarize_small(cx<T>* U) {
    static_assert(NC <= 4, "register-resident reunitarisation is for Nc <= 4");
    if (NC == 2) {
        T n = Fn<T>::sqrt((U[0].re * U[0].re + U[0].im * U[0].im) + (U[1].re * U[1].re + U[1].im * U[1].im));
        U[0] = mk<T>(U[0].re / n, U[0].im / n);
        U[1] = mk<T>(U[1].re / n, U[1].im / n);
        U[NC * NC - 2] = mk<T>(-U[1].re, U[1].im);
        U[NC * NC - 1] = mk<T>(U[0].re, -U[0].im);
    } else if (NC == 3) {
        gram_schmidt_su3_two_rows<T>(U);
        su3_third_row(U);
    } else {
        gram_schmidt_rows<NC, T, true>(U, NC);
        const cx<T> d = determinant4<T>(U);
        const T inv = (T)1 / Fn<T>::sqrt(d.re * d.re + d.im * d.im);
        const cx<T> ph = mk<T>(d.re * inv, -d.im * inv);
#pragma unroll
        for (int k = 0; k < NC; ++k) U[(NC - 1) * NC + k] = U[(NC - 1) * NC + k] * ph;
    }
}

// block-wide sum of doubles (warp shuffle, then shared memory across warps); result in thread 0
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) sh[w] = v;
    __syncthreads();
    v = (threadIdx.x < nw) ? sh[threadIdx.x] : 0.0;
    if (w == 0) for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace sug
