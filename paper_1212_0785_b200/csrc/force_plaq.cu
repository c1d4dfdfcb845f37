// force_plaq.cu — Wilson gauge force by plaquette sharing, subset ALL.
//
// Same result as force.cu (O7) for unitary links, reached with far fewer products and loads.  Every
// plaquette is computed ONCE, by the (site y, plane mu<nu) work item, from its four links
//     U1 = U_mu(y), U2 = U_nu(y+mu), U3 = U_nu(y), U4 = U_mu(y+nu),   a = U1 U2,  b = U3 U4,
// and feeds all four links it contains.  With TA(M) = (M - M^dag)/2 - tr(..)/6 (linear, TA(M^dag) = -TA(M)):
//     link (y,mu):      W += a b^dag                               -> up[mu][y]      += TA(a b^dag)
//     link (y,nu):      W += b a^dag = (a b^dag)^dag               -> up[nu][y]      -= TA(a b^dag)
//     link (y+nu, mu):  W += U4 a^dag U3 = U4 (a^dag b) U4^dag     -> G[mu][y+nu]    += TA(a^dag b)
//     link (y+mu, nu):  W += U2 b^dag U1 = U2 (a^dag b)^dag U2^dag -> G[nu][y+mu]    -= TA(a^dag b)
// (the last two use U3 = b U4^dag and U1 = a U2^dag, i.e. unitarity of the links, exact to rounding on
// an MD trajectory), and finally  F_mu(x) = (i beta/6) [ up[mu][x] + U_mu(x) G[mu][x] U_mu(x)^dag ].
// 3.7 products per plaquette + 1.5 per link instead of 13 per link.
//
// A block owns a 4-D tile; up[] and G[] live in shared memory as 8 reals (anti-Hermitian traceless) per
// (mu, site).  Work proceeds in six plane phases separated by __syncthreads(); within a phase every
// accumulator entry is touched by exactly one thread, so the summation order is fixed (deterministic).
// Contributions that enter the tile from plaquettes based one site outside it (the -mu and -nu faces)
// are recomputed by extra "halo" items instead of being exchanged between blocks.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

constexpr int FP_THREADS = 384;

// anti-Hermitian traceless 3x3 as 8 reals: diag = i*(d0, d1, -d0-d1); x01, x02, x12 complex (x_ji = -conj x_ij)
template <typename T>
struct AH {
    T d0, d1;
    T r01, i01, r02, i02, r12, i12;
};

// t = TA(A B^dag)  (DA = false)   or   t = TA(A^dag B)  (DA = true)
//   M_ij = sum_k A_ik conj(B_jk)   (DA false);   M_ij = sum_k conj(A_ki) B_kj   (DA true)
template <bool DA, typename T>
__device__ __forceinline__ void ta_mul(AH<T> &t, const M3<T> &A, const M3<T> &B) {
    T dim[3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        T s = T(0);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const int e = DA ? 3 * k + i : 3 * i + k;
            // Im(A conj B) = Ai Br - Ar Bi ;  Im(conj A B) = Ar Bi - Ai Br
            if (DA) s = fma_(A.re[e], B.im[e], fma_(-A.im[e], B.re[e], s));
            else s = fma_(A.im[e], B.re[e], fma_(-A.re[e], B.im[e], s));
        }
        dim[i] = s;
    }
    const T m = (dim[0] + dim[1] + dim[2]) * T(1.0 / 3.0);
    t.d0 = dim[0] - m;
    t.d1 = dim[1] - m;
    T xr[3], xi[3];
#pragma unroll
    for (int p = 0; p < 3; p++) {
        const int i = p == 2 ? 1 : 0, j = p == 0 ? 1 : 2;
        T mr = T(0), mi = T(0), nr = T(0), ni = T(0);  // M_ij, M_ji
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (DA) {
                // M_ij += conj(A_ki) B_kj ; M_ji += conj(A_kj) B_ki
                const T ar = A.re[3 * k + i], ai = A.im[3 * k + i], br = B.re[3 * k + j], bi = B.im[3 * k + j];
                mr = fma_(ar, br, fma_(ai, bi, mr));
                mi = fma_(ar, bi, fma_(-ai, br, mi));
                const T cr = A.re[3 * k + j], ci = A.im[3 * k + j], dr = B.re[3 * k + i], di = B.im[3 * k + i];
                nr = fma_(cr, dr, fma_(ci, di, nr));
                ni = fma_(cr, di, fma_(-ci, dr, ni));
            } else {
                // M_ij += A_ik conj(B_jk) ; M_ji += A_jk conj(B_ik)
                const T ar = A.re[3 * i + k], ai = A.im[3 * i + k], br = B.re[3 * j + k], bi = B.im[3 * j + k];
                mr = fma_(ar, br, fma_(ai, bi, mr));
                mi = fma_(ai, br, fma_(-ar, bi, mi));
                const T cr = A.re[3 * j + k], ci = A.im[3 * j + k], dr = B.re[3 * i + k], di = B.im[3 * i + k];
                nr = fma_(cr, dr, fma_(ci, di, nr));
                ni = fma_(ci, dr, fma_(-cr, di, ni));
            }
        }
        // X_ij = (M_ij - conj(M_ji)) / 2
        xr[p] = T(0.5) * (mr - nr);
        xi[p] = T(0.5) * (mi + ni);
    }
    t.r01 = xr[0]; t.i01 = xi[0];
    t.r02 = xr[1]; t.i02 = xi[1];
    t.r12 = xr[2]; t.i12 = xi[2];
}

// shared-memory accumulators: entry (arr, mu, k, slot) is one pair; arr 0 = up, 1 = G; k = 16-byte chunk.
// Consecutive slots are consecutive pairs: conflict-free for a warp of consecutive sites.
template <typename T>
struct Acc {
    pair_t<T> *base;
    int nsite;
    __device__ __forceinline__ pair_t<T> *p(int arr, int mu, int slot) const {
        return base + (size_t)((arr * 4 + mu) * 4) * nsite + slot;
    }
    // sign +1/-1; first: assign instead of accumulate
    __device__ __forceinline__ void add(int arr, int mu, int slot, const AH<T> &t, T sign, bool first) const {
        pair_t<T> *q = p(arr, mu, slot);
        pair_t<T> v0, v1, v2, v3;
        if (first) {
            v0.x = v0.y = v1.x = v1.y = v2.x = v2.y = v3.x = v3.y = T(0);
        } else {
            v0 = q[0]; v1 = q[nsite]; v2 = q[2 * nsite]; v3 = q[3 * nsite];
        }
        v0.x = fma_(sign, t.d0, v0.x);  v0.y = fma_(sign, t.d1, v0.y);
        v1.x = fma_(sign, t.r01, v1.x); v1.y = fma_(sign, t.i01, v1.y);
        v2.x = fma_(sign, t.r02, v2.x); v2.y = fma_(sign, t.i02, v2.y);
        v3.x = fma_(sign, t.r12, v3.x); v3.y = fma_(sign, t.i12, v3.y);
        q[0] = v0; q[nsite] = v1; q[2 * nsite] = v2; q[3 * nsite] = v3;
    }
    __device__ __forceinline__ void get(int arr, int mu, int slot, AH<T> &t) const {
        const pair_t<T> *q = p(arr, mu, slot);
        const pair_t<T> v0 = q[0], v1 = q[nsite], v2 = q[2 * nsite], v3 = q[3 * nsite];
        t.d0 = v0.x; t.d1 = v0.y; t.r01 = v1.x; t.i01 = v1.y; t.r02 = v2.x; t.i02 = v2.y; t.r12 = v3.x; t.i12 = v3.y;
    }
};

__device__ __forceinline__ int sel4(const int a[4], int i) { return i == 0 ? a[0] : i == 1 ? a[1] : i == 2 ? a[2] : a[3]; }

// tile-local coordinates (c[d] in [-1, T[d]]) -> global site (periodic)
__device__ __forceinline__ Site tile_global_site(const LatP &lat, const int o[4], const int c[4]) {
    Site st;
    int sum = 0, s = 0;
#pragma unroll
    for (int d = 0; d < 4; d++) {
        int g = o[d] + c[d];
        g = g < 0 ? g + lat.L[d] : g >= lat.L[d] ? g - lat.L[d] : g;
        st.c[d] = g;
        sum += g;
        s += g * lat.stride[d];
    }
    st.s = s;
    st.par = sum & 1;
    return st;
}

__device__ __forceinline__ int slot_of(const TileP &tile, const int c[4], int par) {
    return par * tile.tsp + (c[0] >> 1) + (tile.T[0] >> 1) * (c[1] + tile.T[1] * (c[2] + tile.T[2] * c[3]));
}

// slot -> tile-local coordinates; osum = o[1]+o[2]+o[3] (o[0] is even)
__device__ __forceinline__ int coords_of_slot(const TileP &tile, int slot, int osum, int c[4]) {
    const int par = slot >= tile.tsp ? 1 : 0;
    int r = slot - par * tile.tsp;
    const int hx = tile.T[0] >> 1;
    const int jx = r % hx;
    r /= hx;
    c[1] = r % tile.T[1];
    r /= tile.T[1];
    c[2] = r % tile.T[2];
    c[3] = r / tile.T[2];
    c[0] = 2 * jx + ((c[1] + c[2] + c[3] + osum + par) & 1);
    return par;
}

__device__ __forceinline__ void tile_origin(const TileP &tile, int b, int o[4]) {
    o[0] = (b % tile.nt[0]) * tile.T[0];
    b /= tile.nt[0];
    o[1] = (b % tile.nt[1]) * tile.T[1];
    b /= tile.nt[1];
    o[2] = (b % tile.nt[2]) * tile.T[2];
    o[3] = (b / tile.nt[2]) * tile.T[3];
}

template <typename T, bool FUSED>
__global__ void __launch_bounds__(FP_THREADS) force_plaq_kernel(const LatP lat, const TileP tile, const T c6 /* beta/6 */,
                                                                const T eps, const pair_t<T> *__restrict__ U,
                                                                pair_t<T> *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nsite = 2 * tile.tsp;
    const Acc<T> acc{(pair_t<T> *)smem_raw, nsite};
    const int V = lat.V;
    int o[4];
    tile_origin(tile, blockIdx.x, o);
    const int osum = o[1] + o[2] + o[3];

#pragma unroll 1
    for (int ph = 0; ph < 6; ph++) {
        // planes (0,1) (0,2) (0,3) (1,2) (1,3) (2,3); an accumulator array is first touched (assigned)
        // in the first phase that contains its direction
        const int mu = ph < 3 ? 0 : ph < 5 ? 1 : 2;
        const int nu = ph < 3 ? ph + 1 : ph < 5 ? ph - 1 : 3;
        const bool first_mu = ph == 0, first_nu = ph < 3;
        const int Tmu = sel4(tile.T, mu), Tnu = sel4(tile.T, nu);
        const int nA = nsite / Tnu;  // halo items based on the -nu face
        const int nB = nsite / Tmu;  // halo items based on the -mu face
#pragma unroll 1
        for (int it = threadIdx.x; it < nsite + nA + nB; it += FP_THREADS) {
            int c[4];
            int kind;  // 0 main, 1 face -nu, 2 face -mu
            if (it < nsite) {
                kind = 0;
                coords_of_slot(tile, it, osum, c);
            } else {
                kind = it < nsite + nA ? 1 : 2;
                int h = kind == 1 ? it - nsite : it - nsite - nA;
                const int fixed = kind == 1 ? nu : mu;
#pragma unroll
                for (int d = 0; d < 4; d++) {
                    if (d == fixed) {
                        c[d] = -1;
                    } else {
                        c[d] = h % tile.T[d];
                        h /= tile.T[d];
                    }
                }
            }
            const Site y = tile_global_site(lat, o, c);
            const int cb = cb_of(lat, y.s, y.par);
            int df[4];
#pragma unroll
            for (int d = 0; d < 4; d++) df[d] = dfwd(lat, y, d);
            const int cb_pm = cb_of(lat, y.s + sel4(df, mu), y.par ^ 1);
            const int cb_pn = cb_of(lat, y.s + sel4(df, nu), y.par ^ 1);
            M3<T> a, b;
            {
                M3<T> X, Y;
                load_link(X, U, V, mu, cb);
                load_link(Y, U, V, nu, cb_pm);
                mul<false, false, false>(a, X, Y);
                load_link(X, U, V, nu, cb);
                load_link(Y, U, V, mu, cb_pn);
                mul<false, false, false>(b, X, Y);
            }
            const int cmu = sel4(c, mu), cnu = sel4(c, nu);
            if (kind == 0) {
                AH<T> tP;
                ta_mul<false>(tP, a, b);
                const int sl = slot_of(tile, c, y.par);
                acc.add(0, mu, sl, tP, T(1), first_mu);
                acc.add(0, nu, sl, tP, T(-1), first_nu);
            }
            AH<T> tR;
            ta_mul<true>(tR, a, b);
            if (kind != 2 && cnu + 1 < Tnu) {  // link (y+nu, mu)
                int cc[4];
#pragma unroll
                for (int d = 0; d < 4; d++) cc[d] = c[d] + (d == nu ? 1 : 0);
                acc.add(1, mu, slot_of(tile, cc, y.par ^ 1), tR, T(1), first_mu);
            }
            if (kind != 1 && cmu + 1 < Tmu) {  // link (y+mu, nu)
                int cc[4];
#pragma unroll
                for (int d = 0; d < 4; d++) cc[d] = c[d] + (d == mu ? 1 : 0);
                acc.add(1, nu, slot_of(tile, cc, y.par ^ 1), tR, T(-1), first_nu);
            }
        }
        __syncthreads();
    }

    // ---- finalize: F_mu(x) = (i beta/6) [ up + U G U^dag ]
#pragma unroll 1
    for (int it = threadIdx.x; it < 4 * nsite; it += FP_THREADS) {
        const int mu = it / nsite;
        const int sl = it - mu * nsite;
        int c[4];
        const int par = coords_of_slot(tile, sl, osum, c);
        const Site x = tile_global_site(lat, o, c);
        const int cb = cb_of(lat, x.s, par);
        M3<T> Um, G, Vm;
        load_link(Um, U, V, mu, cb);
        AH<T> g, u;
        acc.get(1, mu, sl, g);
        acc.get(0, mu, sl, u);
        G.re[0] = T(0); G.im[0] = g.d0;
        G.re[4] = T(0); G.im[4] = g.d1;
        G.re[8] = T(0); G.im[8] = -(g.d0 + g.d1);
        G.re[1] = g.r01; G.im[1] = g.i01; G.re[3] = -g.r01; G.im[3] = g.i01;
        G.re[2] = g.r02; G.im[2] = g.i02; G.re[6] = -g.r02; G.im[6] = g.i02;
        G.re[5] = g.r12; G.im[5] = g.i12; G.re[7] = -g.r12; G.im[7] = g.i12;
        mul<false, false, false>(Vm, Um, G);
        AH<T> h;
        ta_mul<false>(h, Vm, Um);  // TA(V U^dag)
        // H = u + h;  F = i c6 H:  F_ii = -c6 d_i,  F_ij = c6 (-Im H_ij + i Re H_ij),  F_ji = conj(F_ij)
        const T d0 = u.d0 + h.d0, d1 = u.d1 + h.d1;
        const T r01 = u.r01 + h.r01, i01 = u.i01 + h.i01;
        const T r02 = u.r02 + h.r02, i02 = u.i02 + h.i02;
        const T r12 = u.r12 + h.r12, i12 = u.i12 + h.i12;
        M3<T> F;
        F.re[0] = -c6 * d0; F.im[0] = T(0);
        F.re[4] = -c6 * d1; F.im[4] = T(0);
        F.re[8] = c6 * (d0 + d1); F.im[8] = T(0);
        F.re[1] = -c6 * i01; F.im[1] = c6 * r01; F.re[3] = -c6 * i01; F.im[3] = -c6 * r01;
        F.re[2] = -c6 * i02; F.im[2] = c6 * r02; F.re[6] = -c6 * i02; F.im[6] = -c6 * r02;
        F.re[5] = -c6 * i12; F.im[5] = c6 * r12; F.re[7] = -c6 * i12; F.im[7] = -c6 * r12;
        if (FUSED) {
            M3<T> P;
            load_link_rw(P, out, V, mu, cb);
#pragma unroll
            for (int e = 0; e < 9; e++) {
                P.re[e] = fma_(eps, F.re[e], P.re[e]);
                P.im[e] = fma_(eps, F.im[e], P.im[e]);
            }
            store_link(P, out, V, mu, cb);
        } else {
            store_link(F, out, V, mu, cb);
        }
    }
}

// ---- host side ------------------------------------------------------------------------------------

// tile for the plaquette kernel: at most max_sites sites, T0 even and as long as possible up to 16
// (coalescing: T0/2 consecutive sites of a parity are contiguous), then the smallest halo sum 1/T_d.
// QCD_TILE="tx,ty,tz,tt" overrides (block-shape sweeps).
static TileP choose_plaq_tile(const LatP &lat, int max_sites) {
    TileP tp;
    tp.npar = 2;
    tp.par0 = 0;
    int best[4] = {2, 1, 1, 1};
    const char *env = getenv("QCD_TILE");
    int e[4];
    bool have = false;
    if (env && sscanf(env, "%d,%d,%d,%d", &e[0], &e[1], &e[2], &e[3]) == 4) {
        have = true;
        for (int d = 0; d < 4; d++)
            if (e[d] < 1 || lat.L[d] % e[d]) have = false;
        if (e[0] & 1) have = false;
        if (have && (long)e[0] * e[1] * e[2] * e[3] > max_sites) have = false;
        if (have) memcpy(best, e, sizeof e);
    }
    if (!have) {
        double best_score = -1e300;
        for (int a = 2; a <= lat.L[0]; a += 2)
            for (int b = 1; b <= lat.L[1]; b++)
                for (int c = 1; c <= lat.L[2]; c++)
                    for (int d = 1; d <= lat.L[3]; d++) {
                        if (lat.L[0] % a || lat.L[1] % b || lat.L[2] % c || lat.L[3] % d) continue;
                        const long n = (long)a * b * c * d;
                        if (n > max_sites) continue;
                        const double halo = 1.0 / a + 1.0 / b + 1.0 / c + 1.0 / d;
                        const double score = (a >= 16 ? 16 : a) * 1e3 - halo * 100.0 + n * 1e-3;
                        if (score > best_score) {
                            best_score = score;
                            best[0] = a; best[1] = b; best[2] = c; best[3] = d;
                        }
                    }
    }
    for (int d = 0; d < 4; d++) {
        tp.T[d] = best[d];
        tp.nt[d] = lat.L[d] / best[d];
    }
    tp.tsp = (tp.T[0] / 2) * tp.T[1] * tp.T[2] * tp.T[3];
    return tp;
}

constexpr int FP_MAX_SITES = 256;

template <typename T, bool FUSED>
static void launch_plaq_v(const qcd_lattice *lat, T c6, T eps, const pair_t<T> *U, pair_t<T> *out, cudaStream_t st) {
    const TileP tp = choose_plaq_tile(lat->p, FP_MAX_SITES);
    const int nsite = 2 * tp.tsp;
    const size_t smem = (size_t)32 * nsite * sizeof(pair_t<T>);
    static bool attr_set = false;  // per instantiation
    if (!attr_set) {
        cudaFuncSetAttribute(force_plaq_kernel<T, FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             32 * FP_MAX_SITES * (int)sizeof(pair_t<T>));
        attr_set = true;
    }
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    force_plaq_kernel<T, FUSED><<<blocks, FP_THREADS, smem, st>>>(lat->p, tp, c6, eps, U, out);
}

int launch_gauge_force_plaq(const qcd_lattice *lat, int prec, double beta, double eps, const void *U, void *out,
                            bool fused_mom, cudaStream_t st) {
    if (prec == QCD_F64) {
        if (fused_mom) launch_plaq_v<double, true>(lat, beta / 6.0, eps, (const double2 *)U, (double2 *)out, st);
        else launch_plaq_v<double, false>(lat, beta / 6.0, eps, (const double2 *)U, (double2 *)out, st);
    } else {
        if (fused_mom) launch_plaq_v<float, true>(lat, (float)(beta / 6.0), (float)eps, (const float2 *)U, (float2 *)out, st);
        else launch_plaq_v<float, false>(lat, (float)(beta / 6.0), (float)eps, (const float2 *)U, (float2 *)out, st);
    }
    return check_launch(fused_mom ? "force_mom_update(plaq)" : "gauge_force(plaq)");
}

}  // namespace qcd
