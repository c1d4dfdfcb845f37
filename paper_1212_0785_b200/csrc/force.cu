// force.cu — Wilson gauge force (O7; "force term calculation", "projection of
// fields"), optionally fused with the momentum update P += eps*F (fewer site loops) and with
// the link update of the same step (single pass).
//
// One thread per site of the subset, all four directions.  A thread block owns the
// sites of a compact 4-D tile so that the neighbour links a site needs are shared through L1.
//
// Two kernels compute the same force:
//   force_plane_kernel  (default)  the six planes are visited once each: the open plaquette
//                       S = U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag closed with U_mu(x) serves F_mu(x) AND,
//                       daggered, F_nu(x); only the down staples are summed per direction.  46 products and
//                       64 link loads per site instead of 52 and 76.  Exact for arbitrary 3x3 matrices.
//   force_kernel        the definition: 6 staples x 2 products per direction, then U_mu(x) A.  Kept as the
//                       tuner's alternative (QCD_FORCE_STAPLE) and as an in-library cross-check.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"
#include "tmem.cuh"

#define QCD_TRY_RC(expr)               \
    do {                               \
        const int rc_ = (expr);        \
        if (rc_ != QCD_OK) return rc_; \
    } while (0)


namespace qcd {

constexpr int FORCE_NT = 128;  // threads per block of the stencil kernels (168 registers in fp64 -> 3 blocks per SM)

// Launch order -> canonical block index bx + nt0 (by + nt1 (bz + nt2 bt)).  On lattices whose timeslices are large
// the blocks are launched z-block by z-block: inside a z-block of tile.zb tiles the order is x, y, z, t, so the
// links a block shares with its t and z neighbours are still in L2 when they are needed again, because T3 + 2
// timeslices of the z-block, not of the whole lattice, pass through it (host side: tile_from_extents).
__device__ __forceinline__ int canonical_block(const TileP &tile, int b) {
    if (tile.zb == tile.nt[2]) return b;
    const int nxy = tile.nt[0] * tile.nt[1];
    const int nin = nxy * tile.zb;
    const int q = b / (nin * tile.nt[3]);
    int r = b - q * nin * tile.nt[3];
    const int bt = r / nin;
    r -= bt * nin;
    const int bz = q * tile.zb + r / nxy;
    return (r % nxy) + nxy * (bz + tile.nt[2] * bt);
}

// thread -> site of the tile of (canonical) block b
__device__ __forceinline__ Site tile_site(const LatP &lat, const TileP &tile, int j, int b) {
    int par = tile.par0;
    if (tile.npar == 2) {
        par = j >= tile.tsp ? 1 : 0;
        j -= par * tile.tsp;
    }
    const int hx = tile.T[0] >> 1;
    int r = j / hx;
    const int jx = j - r * hx;
    const int jy = r % tile.T[1];
    r /= tile.T[1];
    const int jz = r % tile.T[2];
    const int jt = r / tile.T[2];
    const int bx = b % tile.nt[0];
    b /= tile.nt[0];
    const int by = b % tile.nt[1];
    b /= tile.nt[1];
    const int bz = b % tile.nt[2];
    const int bt = b / tile.nt[2];
    Site st;
    st.par = par;
    st.c[1] = by * tile.T[1] + jy;
    st.c[2] = bz * tile.T[2] + jz;
    st.c[3] = lat.t0 + bt * tile.T[3] + jt;  // the interior timeslices [t0, t1) of a slab lattice; t0 = 0 otherwise
    st.c[0] = bx * tile.T[0] + 2 * jx + ((st.c[1] + st.c[2] + st.c[3] + par) & 1);
    st.s = st.c[0] + lat.L[0] * (st.c[1] + lat.L[1] * (st.c[2] + lat.L[2] * st.c[3]));
    return st;
}

// Lexicographic offsets of the periodic hops x -> x +- e_d for the direction d = (mu + k) & 3, mu the (rolled) loop
// variable.  Picking them from a per-thread register array with a run-time index compiles to branches, which keep the
// compiler from moving the next product's loads above the current one.  The two possible hops per direction are
// block-uniform, so they sit in shared memory, tab[d] = stride_d, tab[4 + d] = -(L_d - 1) stride_d, and a thread keeps
// eight wrap bits.  (Register arrays rotated once per direction were 2 % faster in fp32 while the plane loop was
// unrolled; with it rolled the table wins in both precisions: profiles/r02_force_limiters.md.)
struct Hops {
    const int *tab;  // shared, 8 ints
    unsigned wrap;   // bit d: c[d] == L[d] - 1;  bit 4 + d: c[d] == 0
    // every thread of the block calls init before the first use; the caller synchronises the block
    __device__ __forceinline__ void init(const LatP &lat, const Site &st, int *t) {
        // strided: a tuned tile may give a block fewer than four threads (tile (2,1,1,1): two)
        for (int d = threadIdx.x; d < 4; d += blockDim.x) {
            t[d] = lat.stride[d];
            t[4 + d] = -(lat.L[d] - 1) * lat.stride[d];
        }
        tab = t;
        wrap = 0;
#pragma unroll
        for (int d = 0; d < 4; d++) wrap |= (st.c[d] == lat.L[d] - 1 ? 1u << d : 0u) | (st.c[d] == 0 ? 16u << d : 0u);
    }
    __device__ __forceinline__ int fwd(int mu, int k) const {
        const int d = (mu + k) & 3;
        return tab[d + 4 * ((wrap >> d) & 1u)];
    }
    __device__ __forceinline__ int bwd(int mu, int k) const {
        const int d = (mu + k) & 3;
        return -tab[d + 4 * ((wrap >> (4 + d)) & 1u)];
    }
};

// Fixed-order sum of one double per thread over a block of ANY size (partial last warp included: no shuffle
// reads a lane that was never launched).  Result valid in thread 0.  buf: NT doubles of shared memory.
template <int NT>
__device__ __forceinline__ double block_sum_any(double v, double *buf) {
    __syncthreads();  // buf may still be read from a previous call
    buf[threadIdx.x] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x < 32) {
        for (int i = threadIdx.x; i < (int)blockDim.x; i += 32) s += buf[i];
    }
    __syncthreads();
    if (threadIdx.x < 32) buf[threadIdx.x] = s;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) {
        const int n = blockDim.x < 32 ? (int)blockDim.x : 32;
        for (int i = 0; i < n; i++) r += buf[i];
    }
    return r;
}

// The same for blocks of whole warps (at most 32 of them): shuffle tree per warp, then the warp sums in warp order.
// buf: 32 doubles of shared memory (the NT-double buffer of block_sum_any would move the L1 carve-out of the
// stencil kernels: profiles/r02_force_limiters.md section 4).
__device__ __forceinline__ double block_sum_warps(double v, double *buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();  // buf may still be read from a previous call
    if ((threadIdx.x & 31) == 0) buf[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) r += buf[w];
    return r;
}

// Halo transport from inside the single-pass step on a slab lattice (SURVEY.md 8(e) "peer stores"):
// where the new links of the slab's first / last interior timeslice also go — the upper halo of the lower
// neighbour's output field (spatial links) and the lower halo of the upper neighbour's (all four).  Pointers may be
// peer-GPU memory; NULL: no neighbour on that side.
struct PushP {
    void *lo_U, *hi_U;
    int lo_Vh, lo_L3, hi_Vh;
};

// the momentum update, the sums and the link update that follow the force of one direction (shared by both kernels)
// PUSH: cb_lo / cb_hi = this site's checkerboard index in the neighbour's halo, or -1 (most sites)
template <typename T, bool FUSED, bool EARLYP, bool LINK, bool SUMS, bool PUSH = false>
__device__ __forceinline__ void finish_direction(const M3<T> &F, const M3<T> &Pm, const M3<T> &Um, const T eps,
                                                 const T eps_u, pair_t<T> *__restrict__ out,
                                                 pair_t<T> *__restrict__ Uout, int V, int mu, int cb, double &sumK,
                                                 pair_t<T> *lo_U = nullptr, int cb_lo = -1, pair_t<T> *hi_U = nullptr,
                                                 int cb_hi = -1) {
    if (FUSED) {
        M3<T> P;
        if (EARLYP) P = Pm;
        else load_link_cs(P, out, V, mu, cb);
#pragma unroll
        for (int e = 0; e < 9; e++) {
            P.re[e] = fma_(eps, F.re[e], P.re[e]);
            P.im[e] = fma_(eps, F.im[e], P.im[e]);
        }
        store_link_cs(P, out, V, mu, cb);
        if (SUMS) {  // |P_mu(x)|^2 in the field's precision (R14), accumulated over links and sites in fp64 (R12)
            T k2 = T(0);
#pragma unroll
            for (int e = 0; e < 9; e++) k2 = fma_(P.re[e], P.re[e], fma_(P.im[e], P.im[e], k2));
            sumK += (double)k2;
        }
        if (LINK) {
            M3<T> E, R;
            expi_herm_scaled<2>(E, P, eps_u);
            mul_top2(R, E, Um);  // reunit rebuilds row 2
            reunit(R);
            store_link_cs(R, Uout, V, mu, cb);
            if (PUSH) {  // the thread that has the boundary link in registers sends it
                if (cb_lo >= 0 && mu < 3) store_link_cs(R, lo_U, V, mu, cb_lo);
                if (cb_hi >= 0) store_link_cs(R, hi_U, V, mu, cb_hi);
            }
        }
    } else {
        store_link_cs(F, out, V, mu, cb);
    }
}

// ---- the plane-sharing kernel ----------------------------------------------------------------------
//
// Only the traceless anti-Hermitian part of W_mu(x) = U_mu(x) A_mu(x) enters the force (O7), and that part is
// linear in W, so W is never formed: nine reals per direction ("TA part": Im W_ii, Re/Im of W_ij - conj W_ji
// for ij = 01, 02, 12) are accumulated.  For a plane mu < nu the closed plaquette
//     Pl = U_mu(x) [U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]
// is the up-staple term of W_mu(x), and Pl^dag is the up-staple term of W_nu(x); TA(Pl^dag) = -TA(Pl).  So the
// plane costs three products for both directions (instead of 2 x 2 + the share of U A), and the contribution to
// the direction handled later waits in shared memory: FORCE_NT x 4 x 9 reals per block.
template <typename T>
struct TA {
    T v[9];  // [0..2] Im W_ii;  [3..5] Re (W_ij - conj W_ji), (ij) = (01), (02), (12);  [6..8] Im of the same
};

// t (+)= TA(A B); returns Re tr(A B) when TR (else 0).  90 FMAs (+18 with TR) against 108 for the full product.
template <bool ACC, bool TR, typename T>
__device__ __forceinline__ T mul_ta(TA<T> &t, const M3<T> &A, const M3<T> &B) {
    T tr = T(0);
#pragma unroll
    for (int i = 0; i < 3; i++) {
        T im = ACC ? t.v[i] : T(0);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            im = fma_(A.re[3 * i + k], B.im[3 * k + i], im);
            im = fma_(A.im[3 * i + k], B.re[3 * k + i], im);
            if (TR) {
                tr = fma_(A.re[3 * i + k], B.re[3 * k + i], tr);
                tr = fma_(-A.im[3 * i + k], B.im[3 * k + i], tr);
            }
        }
        t.v[i] = im;
    }
    const int I[3] = {0, 0, 1}, J[3] = {1, 2, 2};
#pragma unroll
    for (int p = 0; p < 3; p++) {
        const int i = I[p], j = J[p];
        T xr = ACC ? t.v[3 + p] : T(0), xi = ACC ? t.v[6 + p] : T(0);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            // + (A B)_ij
            xr = fma_(A.re[3 * i + k], B.re[3 * k + j], xr);
            xr = fma_(-A.im[3 * i + k], B.im[3 * k + j], xr);
            xi = fma_(A.re[3 * i + k], B.im[3 * k + j], xi);
            xi = fma_(A.im[3 * i + k], B.re[3 * k + j], xi);
            // - conj (A B)_ji
            xr = fma_(-A.re[3 * j + k], B.re[3 * k + i], xr);
            xr = fma_(A.im[3 * j + k], B.im[3 * k + i], xr);
            xi = fma_(A.re[3 * j + k], B.im[3 * k + i], xi);
            xi = fma_(A.im[3 * j + k], B.re[3 * k + i], xi);
        }
        t.v[3 + p] = xr;
        t.v[6 + p] = xi;
    }
    return tr;
}

// F = (i c)[(W - W^dag) - tr/3] from the TA part of W (same formulas as project_force)
template <typename T>
__device__ __forceinline__ void force_from_ta(M3<T> &F, const TA<T> &a, T c) {
    const T m = (a.v[0] + a.v[1] + a.v[2]) * T(1.0 / 3.0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        F.re[4 * k] = T(-2) * c * (a.v[k] - m);
        F.im[4 * k] = T(0);
    }
    const int I[3] = {0, 0, 1}, J[3] = {1, 2, 2};
#pragma unroll
    for (int k = 0; k < 3; k++) {
        F.re[3 * I[k] + J[k]] = -c * a.v[6 + k];
        F.im[3 * I[k] + J[k]] = c * a.v[3 + k];
        F.re[3 * J[k] + I[k]] = -c * a.v[6 + k];
        F.im[3 * J[k] + I[k]] = -c * a.v[3 + k];
    }
}

// The pending TA parts, four directions x nine reals per thread.  TMEM = true: in Tensor Memory (tmem.cuh; the
// block must be whole warps, at most four); false: in shared memory, component j of direction d at
// [(d*9 + j)*FORCE_NT + thread].
template <typename T, bool TMEM>
struct Pend {
    T *p;        // shared
    uint32_t a;  // tensor memory address of this thread's lane, column 0 of the block's allocation
    static constexpr int WPD = 9 * (int)sizeof(T) / 4;  // 32-bit words per direction

    __device__ __forceinline__ void zero() {
        if (TMEM) {
            TA<T> z;
#pragma unroll
            for (int k = 0; k < 9; k++) z.v[k] = T(0);
#pragma unroll
            for (int d = 0; d < 4; d++) tmem_store9(a + d * WPD, z.v);
        } else {
#pragma unroll
            for (int j = 0; j < 36; j++) p[j * FORCE_NT] = T(0);
        }
    }
    __device__ __forceinline__ void load(int d, TA<T> &t) const {
        if (TMEM) {
            tmem_wait_st();
            tmem_load9(a + d * WPD, t.v);
        } else {
#pragma unroll
            for (int k = 0; k < 9; k++) t.v[k] = p[(d * 9 + k) * FORCE_NT];
        }
    }
    template <int SGN>
    __device__ __forceinline__ void add(int d, const TA<T> &t) {
        if (TMEM) {
            TA<T> o;
            load(d, o);
#pragma unroll
            for (int k = 0; k < 9; k++) o.v[k] += T(SGN) * t.v[k];
            tmem_store9(a + d * WPD, o.v);
        } else {
#pragma unroll
            for (int k = 0; k < 9; k++) p[(d * 9 + k) * FORCE_NT] += T(SGN) * t.v[k];
        }
    }
};

// FUSED: out = P, P += eps F; else out = F.  LINK (needs FUSED): the whole MD step in one pass (SURVEY.md 8(a)
// "single pass, ping-pong U"): Uout_mu(x) = reunit(exp(i eps_u P_mu(x)) U_mu(x)) is written to a second gauge
// field (neighbouring threads still read the old U).  ANISO (R19): the staples of plane
// (mu,nu) carry the weight wt if mu or nu is the time direction, else ws (c is then 1/12); planes of weight zero
// are skipped.  SUMS (needs FUSED): sum_{mu<nu} Re tr P_mu_nu(x) over the block's sites (the closed plaquettes are
// exactly the six based at x, so a block whose tile lies in one timeslice also yields that timeslice's share,
// R13) and K = sum |P_ij|^2 of the updated momenta as by-products (PAPER.md:26 fused as in PAPER.md:32), one fp64
// partial pair per block.
template <typename T, bool FUSED, bool EARLYP, bool LINK, bool ANISO, bool SUMS, bool TMEM, bool PUSH = false>
// resident blocks per SM: 3 in fp64 (168 registers), 4 in fp32 (128 registers) — measured best of 2..6
__global__ void __launch_bounds__(FORCE_NT, sizeof(T) == 8 ? 3 : 4)
    force_plane_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */, const T eps,
                       const pair_t<T> *__restrict__ U, pair_t<T> *__restrict__ out, const T eps_u,
                       pair_t<T> *__restrict__ Uout, const T ws, const T wt, double *__restrict__ partial,
                       const PushP push) {
    constexpr int TMEM_COLS = sizeof(T) == 8 ? 128 : 64;  // 4 x 18 (fp64) or 4 x 9 (fp32) words per thread
    __shared__ T pend_s[TMEM ? 1 : 4 * 9 * FORCE_NT];
    __shared__ uint32_t tmem_base;
    __shared__ int hop_tab[8];
    Pend<T, TMEM> pend;
    const int bc = canonical_block(tile, blockIdx.x);
    const Site st = tile_site(lat, tile, threadIdx.x, bc);
    Hops hop;
    hop.init(lat, st, hop_tab);
    if (TMEM) {
        if (threadIdx.x < 32) tmem_alloc<TMEM_COLS>(&tmem_base);
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        pend.a = tmem_base + ((threadIdx.x & ~31u) << 16);
    } else {
        __syncthreads();
        pend.p = pend_s + threadIdx.x;
    }
    double sumW = 0.0, sumK = 0.0;
    const int V = lat.V;
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);
    int cb_lo = -1, cb_hi = -1;
    if (PUSH) {  // sites of the slab's first / last interior timeslice: where they sit in the neighbours' halos
        const int sx = st.c[0] + lat.L[0] * (st.c[1] + lat.L[1] * st.c[2]), sp = st.c[0] + st.c[1] + st.c[2];
        if (st.c[3] == 1 && push.lo_U) {
            const int tp = push.lo_L3 - 1;
            cb_lo = ((sp + tp) & 1) * push.lo_Vh + ((sx + lat.stride[3] * tp) >> 1);
        }
        if (st.c[3] == lat.L[3] - 2 && push.hi_U) cb_hi = (sp & 1) * push.hi_Vh + (sx >> 1);
    }
    pend.zero();

#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int dfm = hop.fwd(mu, 0);
        const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);  // x + mu
        M3<T> Pm;
        if (FUSED && EARLYP) load_link_cs(Pm, out, V, mu, cb);
        // planes (mu, nu), nu = mu + k > mu: closed plaquette -> TA parts of W_mu (+) and of W_nu (-)
        // this loop is rolled: its bodies are separated by the uniform trip count anyway (nothing is scheduled across
        // them), and one copy instead of three brings the kernel from 53 to 40 kB of code (instruction cache:
        // -1.5 % in fp64, -5 % in fp32, profiles/r02_force_limiters.md); the staple loop below stays unrolled
        // (rolled: +1 % in fp64) because ptxas starts the next staple's loads under the current product
#pragma unroll 1
        for (int k = 1; k <= 3 - mu; k++) {
            const int nu = mu + k;
            const T w = ANISO ? (nu == 3 ? wt : ws) : T(1);
            if (ANISO && w == T(0)) continue;
            const int cb_pn = cb_of(lat, st.s + hop.fwd(mu, k), par ^ 1);  // x + nu
            M3<T> X, Y, Z;
            load_link(X, U, V, nu, cb_pm);
            load_link(Y, U, V, mu, cb_pn);
            mul<false, true, false>(Z, X, Y);  // U_nu(x+mu) U_mu(x+nu)^dag
            load_link(X, U, V, nu, cb);
            mul<false, true, false>(Y, Z, X);  // ... U_nu(x)^dag: the up staple of (mu, nu)
            if (ANISO) scale(Y, w);
            load_link(X, U, V, mu, cb);
            TA<T> t;
            const T tr = mul_ta<false, SUMS>(t, X, Y);
            if (SUMS) sumW += (double)tr;  // Re tr P_mu_nu(x): the six plaquettes based at x, each exactly once
            pend.template add<1>(mu, t);
            pend.template add<-1>(nu, t);
        }
        // down staples of direction mu
        M3<T> A;
        zero(A);
#pragma unroll
        for (int k = 1; k < 4; k++) {
            const int nu = (mu + k) & 3;
            const T w = ANISO ? ((mu == 3 || nu == 3) ? wt : ws) : T(1);
            if (ANISO && w == T(0)) continue;  // warp-uniform
            const int dbn = hop.bwd(mu, k);
            const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);      // x - nu
            const int cb_pmmn = cb_of(lat, st.s + dfm + dbn, par);  // x + mu - nu
            M3<T> X, Y, Z;
            // U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
            load_link(X, U, V, nu, cb_pmmn);
            load_link(Y, U, V, mu, cb_mn);
            mul<true, true, false>(Z, X, Y);
            if (ANISO) scale(Z, w);
            load_link(X, U, V, nu, cb_mn);
            mul<false, false, true>(A, Z, X);
        }
        M3<T> Um, F;
        load_link(Um, U, V, mu, cb);
        TA<T> acc;
        mul_ta<false, false>(acc, Um, A);
        {  // the parts that waited in Tensor Memory join after the product: their load is off the critical path
            TA<T> w;
            pend.load(mu, w);
#pragma unroll
            for (int j = 0; j < 9; j++) acc.v[j] += w.v[j];
        }
        force_from_ta(F, acc, c);
        finish_direction<T, FUSED, EARLYP, LINK, SUMS, PUSH>(F, Pm, Um, eps, eps_u, out, Uout, V, mu, cb, sumK,
                                                             (pair_t<T> *)push.lo_U, cb_lo, (pair_t<T> *)push.hi_U, cb_hi);
    }
    if (TMEM) {
        tmem_wait_st();
        tmem_fence_before_sync();
        __syncthreads();
        if (threadIdx.x < 32) tmem_dealloc<TMEM_COLS>(tmem_base);
    }
    if (SUMS) {
        // one plaquette partial per (timeslice of the tile, block), stored timeslice-major: the partials of one
        // timeslice are consecutive whatever the tile's t extent (R13); then one K partial per block
        __shared__ double red[TMEM ? 32 : FORCE_NT];  // TMEM: the block is whole warps
        const int nxyz = tile.nt[0] * tile.nt[1] * tile.nt[2];
        const int bt = bc / nxyz, bxyz = bc - bt * nxyz;
        const int jt = st.c[3] - lat.t0 - bt * tile.T[3];
        for (int q = 0; q < tile.T[3]; q++) {
            const double v = jt == q ? sumW : 0.0;
            const double a = TMEM ? block_sum_warps(v, red) : block_sum_any<FORCE_NT>(v, red);
            if (threadIdx.x == 0) partial[(bt * tile.T[3] + q) * nxyz + bxyz] = a;
        }
        const double b = TMEM ? block_sum_warps(sumK, red) : block_sum_any<FORCE_NT>(sumK, red);
        if (threadIdx.x == 0) partial[gridDim.x * tile.T[3] + bc] = b;
    }
}

// ---- the definition kernel -------------------------------------------------------------------------
template <typename T, bool FUSED, bool EARLYP, bool LINK, bool ANISO, bool SUMS>
__global__ void __launch_bounds__(FORCE_NT, 3)
    force_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */, const T eps,
                 const pair_t<T> *__restrict__ U, pair_t<T> *__restrict__ out, const T eps_u,
                 pair_t<T> *__restrict__ Uout, const T ws, const T wt, double *__restrict__ partial) {
    __shared__ int hop_tab[8];
    double sumW = 0.0, sumK = 0.0;
    const Site st = tile_site(lat, tile, threadIdx.x, blockIdx.x);
    Hops hop;
    hop.init(lat, st, hop_tab);
    __syncthreads();
    const int V = lat.V;
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);

#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int dfm = hop.fwd(mu, 0);
        const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);  // x + mu
        M3<T> A, Pm;
        // the momenta come straight from HBM (no reuse): with registers to spare (fp32) their loads are issued
        // before the staple work so the DRAM latency is hidden behind it
        if (FUSED && EARLYP) load_link_cs(Pm, out, V, mu, cb);
        zero(A);
#pragma unroll
        for (int k = 1; k < 4; k++) {
            const int nu = (mu + k) & 3;
            const T w = ANISO ? ((mu == 3 || nu == 3) ? wt : ws) : T(1);
            if (ANISO && w == T(0)) continue;  // warp-uniform
            const int dfn = hop.fwd(mu, k);
            const int dbn = hop.bwd(mu, k);
            const int cb_pn = cb_of(lat, st.s + dfn, par ^ 1);      // x + nu
            const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);      // x - nu
            const int cb_pmmn = cb_of(lat, st.s + dfm + dbn, par);  // x + mu - nu
            M3<T> X, Y, Z;
            // up staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
            {
                load_link(X, U, V, nu, cb_pm);
                load_link(Y, U, V, mu, cb_pn);
            }
            mul<false, true, false>(Z, X, Y);
            if (ANISO) scale(Z, w);
            load_link(X, U, V, nu, cb);
            mul<false, true, true>(A, Z, X);
            // down staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
            load_link(X, U, V, nu, cb_pmmn);
            load_link(Y, U, V, mu, cb_mn);
            mul<true, true, false>(Z, X, Y);
            if (ANISO) scale(Z, w);
            load_link(X, U, V, nu, cb_mn);
            mul<false, false, true>(A, Z, X);
        }
        M3<T> Um, W, F;
        load_link(Um, U, V, mu, cb);
        mul<false, false, false>(W, Um, A);
        project_force(F, W, c);
        if (SUMS) sumW += (double)W.re[0] + (double)W.re[4] + (double)W.re[8];
        finish_direction<T, FUSED, EARLYP, LINK, SUMS>(F, Pm, Um, eps, eps_u, out, Uout, V, mu, cb, sumK);
    }
    if (SUMS) {
        __shared__ double red[FORCE_NT];
        const double a = block_sum_any<FORCE_NT>(sumW, red);
        const double b = block_sum_any<FORCE_NT>(sumK, red);
        if (threadIdx.x == 0) {
            partial[blockIdx.x] = a;
            partial[gridDim.x + blockIdx.x] = b;
        }
    }
}

// ---- host side: tile choice -------------------------------------------------------------------

// all divisors of n (even ones only if `even`)
static int divisors(int n, bool even, int *out) {
    int k = 0;
    for (int d = 1; d <= n; d++)
        if (n % d == 0 && (!even || (d & 1) == 0)) out[k++] = d;
    return k;
}

static void tile_from_extents(const LatP &lat, int prec, int subset, const int t[4], TileP &tp) {
    tp.npar = subset == QCD_ALL ? 2 : 1;
    tp.par0 = subset == QCD_ODD ? 1 : 0;
    for (int d = 0; d < 4; d++) {
        tp.T[d] = t[d];
        tp.nt[d] = (d == 3 ? lat.t1 - lat.t0 : lat.L[d]) / t[d];
    }
    tp.tsp = (tp.T[0] / 2) * tp.T[1] * tp.T[2] * tp.T[3];
    // Launch order (canonical_block).  While a row of tiles in t is worked on, T3 + 2 timeslices of the gauge field
    // are live in L2; measured on B200 the step loses 11 ... 23 % per site once they exceed about 60 MB (32^3 x Lt
    // is below: plain order).  Above, z-blocks are cut so that the live part — (z extent + 2) planes of T3 + 2
    // timeslices — stays under 48 MB: -11 % at 32x64x64x32 and 64^3x32, -3 % at 48^3x96 (profiles/r02_shapes.md).
    tp.zb = tp.nt[2];
    const double plane = (double)lat.L[0] * lat.L[1] * (tp.T[3] + 2) * 72.0 * (prec == QCD_F64 ? 8 : 4);
    if (plane * lat.L[2] > 60e6) {
        for (int z = tp.nt[2]; z >= 1; z--)
            if (tp.nt[2] % z == 0 && (z == 1 || plane * (z * tp.T[2] + 2) <= 48e6)) {
                tp.zb = z;
                break;
            }
    }
}

// Tile extents dividing L with T0 even and threads = T0/2*T1*T2*T3*npar as close to FORCE_NT as possible (never
// above it), preferring a long x extent (coalescing: T0/2 consecutive sites are contiguous in memory) and then the
// smallest surface (L1 reuse of neighbour links).  Called once per lattice (qcd_lattice_create).
void default_force_tile(const LatP &lat, int npar, int out[4]) {
    int best[4] = {2, 1, 1, 1};
    int dv[4][128], nd[4];
    for (int d = 0; d < 4; d++) nd[d] = divisors(d == 3 ? lat.t1 - lat.t0 : lat.L[d], d == 0, dv[d]);
    double best_score = -1e300;
    for (int a = 0; a < nd[0]; a++)
        for (int b = 0; b < nd[1]; b++)
            for (int cc = 0; cc < nd[2]; cc++)
                for (int d = 0; d < nd[3]; d++) {
                    const int t[4] = {dv[0][a], dv[1][b], dv[2][cc], dv[3][d]};
                    const long threads = (long)(t[0] / 2) * t[1] * t[2] * t[3] * npar;
                    if (threads > FORCE_NT) continue;
                    const double vol = (double)t[0] * t[1] * t[2] * t[3];
                    double surf = 0;
                    for (int k = 0; k < 4; k++) surf += vol / t[k];
                    // more threads first; then x extent up to 32 (256-byte rows per parity in fp64; measured best on
                    // B200); then compactness; among equals the extent goes to y before z before t: consecutive
                    // threads of a warp are then consecutive in memory (the site index runs x, y, z, t), and a tile
                    // inside one timeslice gives per-timeslice sums as a by-product (32x2x2x1 beats 32x1x2x2 by 3.5 %
                    // at 32^3x64 inside the MD-step loop)
                    const double score = threads * 1e6 + (t[0] >= 32 ? 32 : t[0]) * 1e3 - surf / vol * 100.0 +
                                         t[1] * 1e-2 + t[2] * 1e-4;
                    if (score > best_score) {
                        best_score = score;
                        memcpy(best, t, sizeof best);
                    }
                }
    memcpy(out, best, sizeof best);
}

// kernel variant and tile for this launch: the tuner's database entry (tune.cu), else the lattice's defaults
struct ForceSel {
    int variant;
    TileP tp;
};

static ForceSel force_sel(const qcd_lattice *lat, int prec, int subset) {
    ForceSel fs;
    fs.variant = QCD_FORCE_PLANE;
    const int *t = subset == QCD_ALL ? lat->tile_all : lat->tile_par;
    TuneCfg cfg;
    if (tune_lookup(lat, prec, subset, QCD_KERNEL_FORCE, cfg)) {
        fs.variant = cfg.variant;
        // validated by qcd_tune_set for the lattice it was set on; a view of fewer timeslices keeps its own default
        if (cfg.tile[0] && (lat->p.t1 - lat->p.t0) % cfg.tile[3] == 0) t = cfg.tile;
    }
    tile_from_extents(lat->p, prec, subset, t, fs.tp);
    return fs;
}

template <typename T, bool FUSED, bool LINK, bool ANISO, bool SUMS>
static void launch_force_k(const qcd_lattice *lat, const ForceSel &fs, T c, T eps, const pair_t<T> *U, pair_t<T> *out,
                           T eps_u, pair_t<T> *Uout, T ws, T wt, double *partial, cudaStream_t st,
                           const PushP *push = nullptr) {
    const TileP &tp = fs.tp;
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    const int threads = tp.tsp * tp.npar;
    // fp32 has the registers to hold the momenta from the start of a direction (-5 %); fp64 does not (+12 %)
    constexpr bool EARLYP = FUSED && sizeof(T) == 4;
    const PushP none = {nullptr, nullptr, 0, 0, 0};
    if constexpr (LINK && !ANISO && !SUMS) {
        if (push) {  // single-pass step that also stores its boundary timeslices into the neighbours' halos
            if (threads % 32 == 0)
                force_plane_kernel<T, FUSED, EARLYP, LINK, ANISO, SUMS, true, true><<<blocks, threads, 0, st>>>(
                    lat->p, tp, c, eps, U, out, eps_u, Uout, ws, wt, partial, *push);
            else
                force_plane_kernel<T, FUSED, EARLYP, LINK, ANISO, SUMS, false, true><<<blocks, threads, 0, st>>>(
                    lat->p, tp, c, eps, U, out, eps_u, Uout, ws, wt, partial, *push);
            return;
        }
    }
    if (fs.variant == QCD_FORCE_STAPLE)
        force_kernel<T, FUSED, EARLYP, LINK, ANISO, SUMS><<<blocks, threads, 0, st>>>(lat->p, tp, c, eps, U, out, eps_u,
                                                                                        Uout, ws, wt, partial);
    else if (threads % 32 == 0)  // whole warps: the pending parts live in Tensor Memory
        force_plane_kernel<T, FUSED, EARLYP, LINK, ANISO, SUMS, true><<<blocks, threads, 0, st>>>(
            lat->p, tp, c, eps, U, out, eps_u, Uout, ws, wt, partial, none);
    else
        force_plane_kernel<T, FUSED, EARLYP, LINK, ANISO, SUMS, false><<<blocks, threads, 0, st>>>(
            lat->p, tp, c, eps, U, out, eps_u, Uout, ws, wt, partial, none);
}

template <typename T>
static int launch_force_t(const qcd_lattice *lat, int subset, const ForceSel &fs, double beta, double eps,
                          const void *U, void *out, bool fused, cudaStream_t st) {
    const T c = (T)(beta / 12.0);
    if (fused)
        launch_force_k<T, true, false, false, false>(lat, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0),
                                                     nullptr, T(0), T(0), nullptr, st);
    else
        launch_force_k<T, false, false, false, false>(lat, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0),
                                                      nullptr, T(0), T(0), nullptr, st);
    return check_launch(fused ? "force_mom_update" : "gauge_force");
}

int launch_gauge_force(const qcd_lattice *lat, int prec, int subset, double beta, double eps, const void *U,
                       void *out, bool fused_mom, cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, subset);
    return prec == QCD_F64 ? launch_force_t<double>(lat, subset, fs, beta, eps, U, out, fused_mom, st)
                           : launch_force_t<float>(lat, subset, fs, beta, eps, U, out, fused_mom, st);
}

// Anisotropic force (plane weights ws, wt; eps = 1 folds a step size into the weights)
template <typename T>
static int launch_force_aniso_t(const qcd_lattice *lat, int subset, const ForceSel &fs, double ws, double wt,
                                double eps, const void *U, void *out, bool fused, cudaStream_t st) {
    const T c = (T)(1.0 / 12.0);
    if (fused)
        launch_force_k<T, true, false, true, false>(lat, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0),
                                                    nullptr, (T)ws, (T)wt, nullptr, st);
    else
        launch_force_k<T, false, false, true, false>(lat, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0),
                                                     nullptr, (T)ws, (T)wt, nullptr, st);
    return check_launch(fused ? "force_mom_update_aniso" : "gauge_force_aniso");
}

int launch_gauge_force_aniso(const qcd_lattice *lat, int prec, int subset, double ws, double wt, double eps,
                             const void *U, void *out, bool fused_mom, cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, subset);
    return prec == QCD_F64 ? launch_force_aniso_t<double>(lat, subset, fs, ws, wt, eps, U, out, fused_mom, st)
                           : launch_force_aniso_t<float>(lat, subset, fs, ws, wt, eps, U, out, fused_mom, st);
}

// doubles of workspace the by-product sums write: the plane kernel one plaquette partial per (block, timeslice of
// its tile) and one K partial per block, the staple kernel two per block
static size_t force_sums_doubles(const ForceSel &fs) {
    const size_t blocks = (size_t)fs.tp.nt[0] * fs.tp.nt[1] * fs.tp.nt[2] * fs.tp.nt[3];
    return blocks * (fs.variant == QCD_FORCE_STAPLE ? 2 : fs.tp.T[3] + 1);
}

int force_sums_check(const qcd_lattice *lat, int prec) {
    const ForceSel fs = force_sel(lat, prec, QCD_ALL);
    if (force_sums_doubles(fs) + 8 > lat->workspace_doubles) {
        set_error("force sums: the workspace cannot hold the per-block partials of the tuned tile");
        return QCD_EWORKSPACE;
    }
    return QCD_OK;
}

// Force + momentum update (+ link update when Uout != NULL) with the plaquette and kinetic-energy sums as
// by-products (subset ALL).  out_plaq[0] = plaquette average of U, out_K[0] = K of the updated P, out_per_t (or
// NULL) = plaquette average per timeslice (Lt doubles).  Returns -1 (nothing enqueued) when out_per_t is asked
// for but the launch configuration cannot give it (staple variant, or a tile that spans several timeslices).
template <typename T>
static int launch_force_sums_t(const qcd_lattice *lat, const ForceSel &fs, double beta, double eps_p, double eps_u,
                               const void *U, void *P, void *Uout, double *out_plaq, double *out_K, double *out_per_t,
                               double *ws, cudaStream_t st) {
    const int blocks = fs.tp.nt[0] * fs.tp.nt[1] * fs.tp.nt[2] * fs.tp.nt[3];
    if (force_sums_doubles(fs) + 8 > lat->workspace_doubles) {
        set_error("force sums: workspace too small");
        return QCD_EWORKSPACE;
    }
    const bool plane = fs.variant != QCD_FORCE_STAPLE;
    const bool slab = lat->p.t0 != 0 || lat->p.t1 != lat->p.L[3];
    if (out_per_t && !(plane && !slab)) return -1;
    const int nW = plane ? blocks * fs.tp.T[3] : blocks;  // plaquette partials
    const T c = (T)(beta / 12.0);
    if (Uout)
        launch_force_k<T, true, true, false, true>(lat, fs, c, (T)eps_p, (const pair_t<T> *)U, (pair_t<T> *)P, (T)eps_u,
                                                   (pair_t<T> *)Uout, T(0), T(0), ws, st);
    else
        launch_force_k<T, true, false, false, true>(lat, fs, c, (T)eps_p, (const pair_t<T> *)U, (pair_t<T> *)P, T(0),
                                                    nullptr, T(0), T(0), ws, st);
    QCD_TRY_RC(check_launch("force sums"));
    // plane kernel: sum of the six plaquette traces per site; staple kernel: sum_mu Re tr W_mu = 4 x that
    // a slab lattice sums (and averages) over its interior timeslices only
    const double V = (double)(lat->p.V / lat->p.L[3]) * (double)(lat->p.t1 - lat->p.t0);
    QCD_TRY_RC(launch_sum_partials(ws, 1, nW, 1.0 / ((plane ? 18.0 : 72.0) * V), out_plaq, st));
    if (out_per_t) {  // the partials of one timeslice are consecutive (timeslice-major order in the kernel)
        const int Lt = lat->p.L[3];
        QCD_TRY_RC(launch_sum_partials(ws, Lt, nW / Lt, (double)Lt / (18.0 * V), out_per_t, st));
    }
    return launch_sum_partials(ws + nW, 1, blocks, 1.0, out_K, st);
}

int launch_force_sums(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U, void *P,
                      void *Uout, double *out_plaq, double *out_K, double *out_per_t, double *ws, cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, QCD_ALL);
    return prec == QCD_F64
               ? launch_force_sums_t<double>(lat, fs, beta, eps_p, eps_u, U, P, Uout, out_plaq, out_K, out_per_t, ws, st)
               : launch_force_sums_t<float>(lat, fs, beta, eps_p, eps_u, U, P, Uout, out_plaq, out_K, out_per_t, ws, st);
}

// Single-pass MD step: P += eps_p F(U); Uout = reunit(exp(i eps_u P) U).  Subset ALL only (every link moves).
template <typename T>
static int launch_md_single_t(const qcd_lattice *lat, const ForceSel &fs, double beta, double eps_p, double eps_u,
                              const void *U, void *P, void *Uout, cudaStream_t st, const PushP *push) {
    launch_force_k<T, true, true, false, false>(lat, fs, (T)(beta / 12.0), (T)eps_p, (const pair_t<T> *)U,
                                                (pair_t<T> *)P, (T)eps_u, (pair_t<T> *)Uout, T(0), T(0), nullptr, st,
                                                push);
    return check_launch(push ? "md_step_single_pass_push" : "md_step_single_pass");
}

int launch_md_single(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U, void *P,
                     void *Uout, cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, QCD_ALL);
    return prec == QCD_F64 ? launch_md_single_t<double>(lat, fs, beta, eps_p, eps_u, U, P, Uout, st, nullptr)
                           : launch_md_single_t<float>(lat, fs, beta, eps_p, eps_u, U, P, Uout, st, nullptr);
}

// the same on a slab lattice, storing the new links of its boundary timeslices into the neighbours' output fields too
int launch_md_single_push(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U,
                          void *P, void *Uout, const qcd_lattice *lo, void *lo_U, const qcd_lattice *hi, void *hi_U,
                          cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, QCD_ALL);
    const PushP push = {lo_U, hi_U, lo ? lo->p.Vh : 0, lo ? lo->p.L[3] : 0, hi ? hi->p.Vh : 0};
    return prec == QCD_F64 ? launch_md_single_t<double>(lat, fs, beta, eps_p, eps_u, U, P, Uout, st, &push)
                           : launch_md_single_t<float>(lat, fs, beta, eps_p, eps_u, U, P, Uout, st, &push);
}

}  // namespace qcd
