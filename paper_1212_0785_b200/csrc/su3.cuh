// su3.cuh — 3x3 complex algebra in registers, templated on the real type (double / float).
// Everything is fully unrolled with compile-time indices so matrices live in registers.
#pragma once

#include <cuda_runtime.h>

namespace qcd {

template <typename T> struct Pair;
template <> struct Pair<double> { using type = double2; };
template <> struct Pair<float> { using type = float2; };
template <typename T> using pair_t = typename Pair<T>::type;

template <typename T>
struct M3 {
    T re[9];
    T im[9];
};

template <typename T> __device__ __forceinline__ T fma_(T a, T b, T c);
template <> __device__ __forceinline__ double fma_<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }

template <typename T> __device__ __forceinline__ T rsqrt_(T a);
template <> __device__ __forceinline__ double rsqrt_<double>(double a) { return rsqrt(a); }  // <= 1 ulp
template <> __device__ __forceinline__ float rsqrt_<float>(float a) { return rsqrtf(a); }

// ---- global memory access.  Device layout (include/qcd.h): array of structures of arrays in chunks of 32
// checkerboard sites: unit k (of NC per site) of site cb at index ((cb >> 5)*NC + k)*32 + (cb & 31); a matrix
// field has NC = 36 complex pairs per site, k = mu*9 + e.  A warp reading one entry of 32 consecutive sites reads
// 512 contiguous bytes (fp64), and all 36 entries of a site sit at compile-time offsets (e*32 units) from one base:
// one address computation per neighbour site instead of one per load.  36 V < 2^32, so 32-bit indices suffice.
constexpr int CHUNK = 32;

__host__ __device__ __forceinline__ unsigned unit_index(int NC, int k, int cb) {
    return ((unsigned)(cb >> 5) * (unsigned)NC + (unsigned)k) * 32u + (unsigned)(cb & 31);
}

// read-only load that asks L1 to keep the line (ld.global.nc.L1::evict_last, SASS LDG.E.EL.CONSTANT): for the
// links of the stencil kernels, which neighbouring threads of the block read again within the same direction, while
// the streaming accesses around them (momenta, outputs: ld/st.global.cs) are marked evict-first
__device__ __forceinline__ double2 ldg_keep(const double2 *p) {
    double2 v;
    asm volatile("ld.global.nc.L1::evict_last.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ldg_keep(const float2 *p) {
    float2 v;
    asm volatile("ld.global.nc.L1::evict_last.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

template <typename T>
__device__ __forceinline__ void load_link(M3<T> &m, const pair_t<T> *__restrict__ f, int V, int mu, int cb) {
    const pair_t<T> *p = f + unit_index(36, mu * 9, cb);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        pair_t<T> v = ldg_keep(p + e * CHUNK);
        m.re[e] = v.x;
        m.im[e] = v.y;
    }
}

// streaming variants (ld.global.cs / st.global.cs): for data touched once per kernel (the momenta in the
// force kernel), so that it does not displace the neighbour links other threads of the block reuse from L1
template <typename T>
__device__ __forceinline__ void load_link_cs(M3<T> &m, const pair_t<T> *f, int V, int mu, int cb) {
    const pair_t<T> *p = f + unit_index(36, mu * 9, cb);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        pair_t<T> v = __ldcs(p + e * CHUNK);
        m.re[e] = v.x;
        m.im[e] = v.y;
    }
}

template <typename T>
__device__ __forceinline__ void store_link_cs(const M3<T> &m, pair_t<T> *f, int V, int mu, int cb) {
    pair_t<T> *p = f + unit_index(36, mu * 9, cb);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        pair_t<T> v;
        v.x = m.re[e];
        v.y = m.im[e];
        __stcs(p + e * CHUNK, v);
    }
}

// same, through the normal (coherent) path: for fields the kernel also writes
template <typename T>
__device__ __forceinline__ void load_link_rw(M3<T> &m, const pair_t<T> *f, int V, int mu, int cb) {
    const pair_t<T> *p = f + unit_index(36, mu * 9, cb);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        pair_t<T> v = p[e * CHUNK];
        m.re[e] = v.x;
        m.im[e] = v.y;
    }
}

template <typename T>
__device__ __forceinline__ void store_link(const M3<T> &m, pair_t<T> *f, int V, int mu, int cb) {
    pair_t<T> *p = f + unit_index(36, mu * 9, cb);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        pair_t<T> v;
        v.x = m.re[e];
        v.y = m.im[e];
        p[e * CHUNK] = v;
    }
}

// ---- products.  DA / DB: take the dagger of that operand.  ACC: C += ... instead of C = ...

template <bool DA, bool DB, bool ACC, typename T>
__device__ __forceinline__ void mul(M3<T> &C, const M3<T> &A, const M3<T> &B) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T cr = ACC ? C.re[3 * i + j] : T(0);
            T ci = ACC ? C.im[3 * i + j] : T(0);
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const int ia = DA ? 3 * k + i : 3 * i + k;
                const int ib = DB ? 3 * j + k : 3 * k + j;
                const T ar = A.re[ia], ai = DA ? -A.im[ia] : A.im[ia];
                const T br = B.re[ib], bi = DB ? -B.im[ib] : B.im[ib];
                cr = fma_(ar, br, cr);
                cr = fma_(-ai, bi, cr);
                ci = fma_(ar, bi, ci);
                ci = fma_(ai, br, ci);
            }
            C.re[3 * i + j] = cr;
            C.im[3 * i + j] = ci;
        }
}

// rows 0 and 1 of C = A B only (row 2 of C is left untouched): what reunit() needs of exp(i eps P) U, since it
// rebuilds the third row from the first two
template <typename T>
__device__ __forceinline__ void mul_top2(M3<T> &C, const M3<T> &A, const M3<T> &B) {
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T cr = T(0), ci = T(0);
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const T ar = A.re[3 * i + k], ai = A.im[3 * i + k];
                const T br = B.re[3 * k + j], bi = B.im[3 * k + j];
                cr = fma_(ar, br, cr);
                cr = fma_(-ai, bi, cr);
                ci = fma_(ar, bi, ci);
                ci = fma_(ai, br, ci);
            }
            C.re[3 * i + j] = cr;
            C.im[3 * i + j] = ci;
        }
}

// Re tr (A B^dagger) = sum_ij Re(A_ij conj(B_ij))
template <typename T>
__device__ __forceinline__ T retr_mul_dag(const M3<T> &A, const M3<T> &B) {
    T acc = T(0);
#pragma unroll
    for (int e = 0; e < 9; e++) {
        acc = fma_(A.re[e], B.re[e], acc);
        acc = fma_(A.im[e], B.im[e], acc);
    }
    return acc;
}

template <typename T>
__device__ __forceinline__ void zero(M3<T> &A) {
#pragma unroll
    for (int e = 0; e < 9; e++) A.re[e] = A.im[e] = T(0);
}

template <typename T>
__device__ __forceinline__ void scale(M3<T> &A, T w) {
#pragma unroll
    for (int e = 0; e < 9; e++) {
        A.re[e] *= w;
        A.im[e] *= w;
    }
}

// ---- projection (O7): F = (i c)[(W - W^dag) - (1/3) tr(W - W^dag)], c = beta/12.
// W - W^dag =: X is anti-Hermitian: X_ii = 2i Im W_ii, X_ij = W_ij - conj(W_ji).
// i*X is Hermitian; F_ii = -2c (Im W_ii - mean Im W_kk), F_ij = i c (W_ij - conj(W_ji)).
template <typename T>
__device__ __forceinline__ void project_force(M3<T> &F, const M3<T> &W, T c) {
    const T m = (W.im[0] + W.im[4] + W.im[8]) * T(1.0 / 3.0);
#pragma unroll
    for (int i = 0; i < 3; i++) {
        F.re[4 * i] = T(-2) * c * (W.im[4 * i] - m);
        F.im[4 * i] = T(0);
    }
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = i + 1; j < 3; j++) {
            const T xr = W.re[3 * i + j] - W.re[3 * j + i];
            const T xi = W.im[3 * i + j] + W.im[3 * j + i];
            // i c (xr + i xi) = -c xi + i c xr
            F.re[3 * i + j] = -c * xi;
            F.im[3 * i + j] = c * xr;
            F.re[3 * j + i] = -c * xi;
            F.im[3 * j + i] = -c * xr;
        }
}

// ---- reunitarisation (O9): row Gram-Schmidt, third row = conj(r0 x r1)
template <typename T>
__device__ __forceinline__ void reunit(M3<T> &M) {
    T n0 = T(0);
#pragma unroll
    for (int j = 0; j < 3; j++) n0 = fma_(M.re[j], M.re[j], fma_(M.im[j], M.im[j], n0));
    T s = rsqrt_(n0);
#pragma unroll
    for (int j = 0; j < 3; j++) {
        M.re[j] *= s;
        M.im[j] *= s;
    }
    // d = r0^dag . r1
    T dr = T(0), di = T(0);
#pragma unroll
    for (int j = 0; j < 3; j++) {
        dr = fma_(M.re[j], M.re[3 + j], dr);
        dr = fma_(M.im[j], M.im[3 + j], dr);
        di = fma_(M.re[j], M.im[3 + j], di);
        di = fma_(-M.im[j], M.re[3 + j], di);
    }
#pragma unroll
    for (int j = 0; j < 3; j++) {
        // r1 -= d r0
        M.re[3 + j] = fma_(-dr, M.re[j], fma_(di, M.im[j], M.re[3 + j]));
        M.im[3 + j] = fma_(-dr, M.im[j], fma_(-di, M.re[j], M.im[3 + j]));
    }
    T n1 = T(0);
#pragma unroll
    for (int j = 0; j < 3; j++) n1 = fma_(M.re[3 + j], M.re[3 + j], fma_(M.im[3 + j], M.im[3 + j], n1));
    s = rsqrt_(n1);
#pragma unroll
    for (int j = 0; j < 3; j++) {
        M.re[3 + j] *= s;
        M.im[3 + j] *= s;
    }
    // r2 = conj(r0 x r1): (a x b)_0 = a1 b2 - a2 b1, ...
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        const T pr = M.re[a] * M.re[3 + b] - M.im[a] * M.im[3 + b] - (M.re[b] * M.re[3 + a] - M.im[b] * M.im[3 + a]);
        const T pi = M.re[a] * M.im[3 + b] + M.im[a] * M.re[3 + b] - (M.re[b] * M.im[3 + a] + M.im[b] * M.re[3 + a]);
        M.re[6 + j] = pr;
        M.im[6 + j] = -pi;
    }
}

// ---- exp(iQ) for Hermitian traceless Q (O8), Cayley-Hamilton route.
// Q^3 = c1 Q + c0 with c1 = (1/2) tr Q^2, c0 = det Q = (1/3) tr Q^3 (both real), hence
// (iQ)^k / k! = a_k + b_k Q + c_k Q^2 with (a,b,c)_{k+1} = (i/(k+1)) (c0 c_k, a_k + c1 c_k, b_k).
// Q is first scaled by 2^-n so that ||Q||_F <= 1 (series terms decay from the start: no
// cancellation), the result squared n times.  NT = number of series terms kept.
// 1/k, k = 0..23 (entry 0 unused), correctly rounded doubles
__device__ __constant__ const double c_inv_k[24] = {0.0, 1.0, 1.0 / 2, 1.0 / 3, 1.0 / 4, 1.0 / 5, 1.0 / 6, 1.0 / 7, 1.0 / 8,
                                                    1.0 / 9, 1.0 / 10, 1.0 / 11, 1.0 / 12, 1.0 / 13, 1.0 / 14, 1.0 / 15,
                                                    1.0 / 16, 1.0 / 17, 1.0 / 18, 1.0 / 19, 1.0 / 20, 1.0 / 21, 1.0 / 22,
                                                    1.0 / 23};

template <typename T> struct ExpTerms;
template <> struct ExpTerms<double> { static constexpr int max_terms = 22; static constexpr double tol = 1e-18; };
template <> struct ExpTerms<float> { static constexpr int max_terms = 13; static constexpr float tol = 1e-9f; };

// E = exp(i eps P) for Hermitian traceless P; only the upper triangle of P is read (P_ji = conj P_ij).
// ROWS = 2: only rows 0 and 1 of E are formed (what reunit() needs of exp(i eps P) U, since it rebuilds the third
// row); ROWS = 3: all of E.
// Arithmetic per link: Q^2 is Hermitian (6 entries, 54 FMAs instead of 108); the series runs on REAL
// coefficients — Q^k/k! = al_k + be_k Q + ga_k Q^2 with (al,be,ga)_{k+1} = (c0 ga, al + c1 ga, be)/(k+1), and
// i^k only decides whether a term adds to the real or the imaginary part of f0, f1, f2 and with which sign.
template <int ROWS, typename T>
__device__ __forceinline__ void expi_herm_scaled(M3<T> &E, const M3<T> &P, const T eps) {
    // ||eps P||_F^2 from the upper triangle
    T n2 = T(0);
#pragma unroll
    for (int i = 0; i < 3; i++) n2 = fma_(P.re[4 * i], P.re[4 * i], n2);
    T off = T(0);
    const int I[3] = {0, 0, 1}, J[3] = {1, 2, 2};
#pragma unroll
    for (int p = 0; p < 3; p++) {
        const int e = 3 * I[p] + J[p];
        off = fma_(P.re[e], P.re[e], fma_(P.im[e], P.im[e], off));
    }
    n2 = fma_(T(2), off, n2) * eps * eps;
    int nsq = 0;
    T scale = eps;
    while (n2 > T(1)) {
        scale *= T(0.5);
        n2 *= T(0.25);
        nsq++;
    }
    // Q = scale * P: d[i] = Q_ii (real), (xr, xi)[p] = Q_ij for (ij) = (01), (02), (12)
    T d[3], xr[3], xi[3];
#pragma unroll
    for (int i = 0; i < 3; i++) d[i] = P.re[4 * i] * scale;
#pragma unroll
    for (int p = 0; p < 3; p++) {
        xr[p] = P.re[3 * I[p] + J[p]] * scale;
        xi[p] = P.im[3 * I[p] + J[p]] * scale;
    }
    // Q2 = Q Q, Hermitian: D[i] = sum_k |Q_ik|^2; (Xr, Xi)[p] = sum_k Q_ik Q_kj
    const T a01 = fma_(xr[0], xr[0], xi[0] * xi[0]);
    const T a02 = fma_(xr[1], xr[1], xi[1] * xi[1]);
    const T a12 = fma_(xr[2], xr[2], xi[2] * xi[2]);
    T D[3], Xr[3], Xi[3];
    D[0] = fma_(d[0], d[0], a01 + a02);
    D[1] = fma_(d[1], d[1], a01 + a12);
    D[2] = fma_(d[2], d[2], a02 + a12);
    // (01): Q00 Q01 + Q01 Q11 + Q02 Q21,  Q21 = conj Q12
    Xr[0] = fma_(d[0] + d[1], xr[0], fma_(xr[1], xr[2], xi[1] * xi[2]));
    Xi[0] = fma_(d[0] + d[1], xi[0], fma_(xi[1], xr[2], -xr[1] * xi[2]));
    // (02): Q00 Q02 + Q01 Q12 + Q02 Q22
    Xr[1] = fma_(d[0] + d[2], xr[1], fma_(xr[0], xr[2], -xi[0] * xi[2]));
    Xi[1] = fma_(d[0] + d[2], xi[1], fma_(xr[0], xi[2], xi[0] * xr[2]));
    // (12): Q10 Q02 + Q11 Q12 + Q12 Q22,  Q10 = conj Q01
    Xr[2] = fma_(d[1] + d[2], xr[2], fma_(xr[0], xr[1], xi[0] * xi[1]));
    Xi[2] = fma_(d[1] + d[2], xi[2], fma_(xr[0], xi[1], -xi[0] * xr[1]));
    const T c1 = T(0.5) * n2;
    // c0 = det Q = (1/3) tr(Q Q2) = (1/3) [sum_i Q_ii Q2_ii + 2 sum_{i<j} Re(Q_ij conj Q2_ij)]
    T c0 = T(0), c0o = T(0);
#pragma unroll
    for (int i = 0; i < 3; i++) c0 = fma_(d[i], D[i], c0);
#pragma unroll
    for (int p = 0; p < 3; p++) c0o = fma_(xr[p], Xr[p], fma_(xi[p], Xi[p], c0o));
    c0 = fma_(T(2), c0o, c0) * T(1.0 / 3.0);
    // series, two terms per round: odd k adds to the imaginary parts, even k to the real parts; the sign pattern
    // + - - + of i^k is folded into the recurrence (every even step carries a factor -1)
    T al = T(1), be = T(0), ga = T(0);
    T f0r = T(1), f0i = T(0), f1r = T(0), f1i = T(0), f2r = T(0), f2i = T(0);
    T bound = T(1);  // x^k / k!, x = ||Q||_F <= 1
    for (int k = 1; k <= ExpTerms<T>::max_terms; k += 2) {
        const T inv1 = (T)c_inv_k[k], inv2 = (T)c_inv_k[k + 1];  // 1/k from a table: an fp64 division is a dozen instructions
        T na = c0 * ga * inv1, nb = fma_(c1, ga, al) * inv1, nc = be * inv1;
        f0i += na;
        f1i += nb;
        f2i += nc;
        al = -c0 * nc * inv2;
        be = -fma_(c1, nc, na) * inv2;
        ga = -nb * inv2;
        f0r += al;
        f1r += be;
        f2r += ga;
        bound *= n2 * inv1 * inv2;
        if (bound < ExpTerms<T>::tol) break;
    }
    // E = f0 + f1 Q + f2 Q2
    const int rows = nsq > 0 ? 3 : ROWS;  // squaring needs the whole matrix
#pragma unroll
    for (int i = 0; i < 3; i++) {
        if (i < rows) {
            E.re[4 * i] = fma_(f1r, d[i], fma_(f2r, D[i], f0r));
            E.im[4 * i] = fma_(f1i, d[i], fma_(f2i, D[i], f0i));
        }
    }
#pragma unroll
    for (int p = 0; p < 3; p++) {
        const int i = I[p], j = J[p];
        // (i,j): Q_ij = xr + i xi
        E.re[3 * i + j] = fma_(f1r, xr[p], fma_(-f1i, xi[p], fma_(f2r, Xr[p], -f2i * Xi[p])));
        E.im[3 * i + j] = fma_(f1r, xi[p], fma_(f1i, xr[p], fma_(f2r, Xi[p], f2i * Xr[p])));
        // (j,i): Q_ji = xr - i xi
        if (j < rows) {
            E.re[3 * j + i] = fma_(f1r, xr[p], fma_(f1i, xi[p], fma_(f2r, Xr[p], f2i * Xi[p])));
            E.im[3 * j + i] = fma_(-f1r, xi[p], fma_(f1i, xr[p], fma_(-f2r, Xi[p], f2i * Xr[p])));
        }
    }
    for (int k = 0; k < nsq; k++) {
        M3<T> S;
        mul<false, false, false>(S, E, E);
        E = S;
    }
}

template <typename T>
__device__ __forceinline__ void expi_herm(M3<T> &E, const M3<T> &Q) {
    expi_herm_scaled<3>(E, Q, T(1));
}

// Q = sum_a q_a T_a (O2), T_a = Gell-Mann / 2
template <typename T>
__device__ __forceinline__ void herm_from_coeffs(M3<T> &Q, const double q[8]) {
    const double is3 = 0.57735026918962576451;  // 1/sqrt(3)
    Q.re[0] = T(q[2] / 2 + q[7] * is3 / 2);
    Q.re[4] = T(-q[2] / 2 + q[7] * is3 / 2);
    Q.re[8] = T(-q[7] * is3);
    Q.im[0] = Q.im[4] = Q.im[8] = T(0);
    Q.re[1] = T(q[0] / 2); Q.im[1] = T(-q[1] / 2);
    Q.re[2] = T(q[3] / 2); Q.im[2] = T(-q[4] / 2);
    Q.re[5] = T(q[5] / 2); Q.im[5] = T(-q[6] / 2);
    Q.re[3] = Q.re[1]; Q.im[3] = -Q.im[1];
    Q.re[6] = Q.re[2]; Q.im[6] = -Q.im[2];
    Q.re[7] = Q.re[5]; Q.im[7] = -Q.im[5];
}

}  // namespace qcd
