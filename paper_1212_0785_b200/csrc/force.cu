// force.cu — Wilson gauge force (O7; "force term calculation", "projection of
// fields"), optionally fused with the momentum update P += eps*F (fewer site loops).
//
// One thread per site of the subset, all four directions.  A thread block owns the
// sites of a compact 4-D tile so that the 44 neighbour links a site needs are shared through L1.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

#define QCD_TRY_RC(expr)               \
    do {                               \
        const int rc_ = (expr);        \
        if (rc_ != QCD_OK) return rc_; \
    } while (0)

namespace qcd {

// thread -> site of the block's tile
__device__ __forceinline__ Site tile_site(const LatP &lat, const TileP &tile, int j) {
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
    int b = blockIdx.x;
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
    st.c[3] = bt * tile.T[3] + jt;
    st.c[0] = bx * tile.T[0] + 2 * jx + ((st.c[1] + st.c[2] + st.c[3] + par) & 1);
    st.s = st.c[0] + lat.L[0] * (st.c[1] + lat.L[1] * (st.c[2] + lat.L[2] * st.c[3]));
    return st;
}

// F_mu(x) for mu = 0..3 at the thread's site; FUSED: out = P, P += eps F; else out = F.
// LINK (needs FUSED): the whole MD step in one pass over the lattice (SURVEY.md 8(a) "single pass, ping-pong U"):
// with the updated momentum still in registers, Uout_mu(x) = reunit(exp(i eps_u P_mu(x)) U_mu(x)) is written
// to a second gauge field (neighbouring threads still read the old U, so the update cannot be in place).
template <bool REC, typename T>
__device__ __forceinline__ void ldU(M3<T> &m, const pair_t<T> *__restrict__ f, int V, int mu, int cb) {
    if (REC) load_link_su3(m, f, V, mu, cb);
    else load_link(m, f, V, mu, cb);
}

// ANISO (R19; "anisotropic Wilson" action): the staples of plane (mu,nu) carry the weight
// wt if mu or nu is the time direction, else ws (c is then 1/12); planes of weight zero are skipped, which
// is what the levels of the multi-timescale integrator (space-space planes only / space-time planes only) use.
template <typename T, bool FUSED, bool EARLYP, bool LINK, int NT = 256, int MINB = 1, bool REC = false,
          bool ANISO = false, bool SUMS = false>
__global__ void __launch_bounds__(NT, MINB) force_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */,
                                                    const T eps, const pair_t<T> *__restrict__ U,
                                                    pair_t<T> *__restrict__ out, const T eps_u,
                                                    pair_t<T> *__restrict__ Uout, const T ws, const T wt,
                                                    double *__restrict__ partial = nullptr) {
    // SUMS (needs FUSED): the two sums the Hamiltonian needs are by-products (PAPER.md:26 reductions, fused
    // as in PAPER.md:32): sum Re tr W_mu(x) = 4 sum_{mu<nu} Re tr P_mu_nu (every plaquette closes four staple
    // loops) and K = sum |P_ij|^2 of the updated momenta.  One fp64 partial pair per block, fixed order.
    double sumW = 0.0, sumK = 0.0;
    const Site st = tile_site(lat, tile, threadIdx.x);
    const int V = lat.V;
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);
    int df[4], db[4];
#pragma unroll
    for (int d = 0; d < 4; d++) {
        df[d] = dfwd(lat, st, d);
        db[d] = dbwd(lat, st, d);
    }

#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int dfm = mu == 0 ? df[0] : mu == 1 ? df[1] : mu == 2 ? df[2] : df[3];
        const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);  // x + mu
        M3<T> A, Pm;
        // the momenta come straight from HBM (no reuse): issue their loads before the staple work so the
        // DRAM latency is hidden behind it (measured: -9 % kernel time at 32^3x64 fp64)
        if (FUSED && EARLYP) load_link_cs(Pm, out, V, mu, cb);
        zero(A);
#pragma unroll
        for (int k = 1; k < 4; k++) {
            const int nu = (mu + k) & 3;
            const T w = ANISO ? ((mu == 3 || nu == 3) ? wt : ws) : T(1);
            if (ANISO && w == T(0)) continue;  // warp-uniform
            const int dfn = nu == 0 ? df[0] : nu == 1 ? df[1] : nu == 2 ? df[2] : df[3];
            const int dbn = nu == 0 ? db[0] : nu == 1 ? db[1] : nu == 2 ? db[2] : db[3];
            const int cb_pn = cb_of(lat, st.s + dfn, par ^ 1);      // x + nu
            const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);      // x - nu
            const int cb_pmmn = cb_of(lat, st.s + dfm + dbn, par);  // x + mu - nu
            M3<T> X, Y, Z;
            // up staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
            ldU<REC>(X, U, V, nu, cb_pm);
            ldU<REC>(Y, U, V, mu, cb_pn);
            mul<false, true, false>(Z, X, Y);
            if (ANISO) scale(Z, w);
            ldU<REC>(X, U, V, nu, cb);
            mul<false, true, true>(A, Z, X);
            // down staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
            ldU<REC>(X, U, V, nu, cb_pmmn);
            ldU<REC>(Y, U, V, mu, cb_mn);
            mul<true, true, false>(Z, X, Y);
            if (ANISO) scale(Z, w);
            ldU<REC>(X, U, V, nu, cb_mn);
            mul<false, false, true>(A, Z, X);
        }
        M3<T> Um, W;
        ldU<REC>(Um, U, V, mu, cb);
        mul<false, false, false>(W, Um, A);
        M3<T> F;
        project_force(F, W, c);
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
            if (SUMS) {
                sumW += (double)W.re[0] + (double)W.re[4] + (double)W.re[8];
#pragma unroll
                for (int e = 0; e < 9; e++) {
                    sumK = fma((double)P.re[e], (double)P.re[e], sumK);
                    sumK = fma((double)P.im[e], (double)P.im[e], sumK);
                }
            }
            if (LINK) {
#pragma unroll
                for (int e = 0; e < 9; e++) {
                    P.re[e] *= eps_u;
                    P.im[e] *= eps_u;
                }
                M3<T> E, R;
                expi_herm(E, P);
                mul_top2(R, E, Um);  // reunit rebuilds row 2
                reunit(R);
                store_link_cs(R, Uout, V, mu, cb);
            }
        } else {
            store_link_cs(F, out, V, mu, cb);
        }
    }
    if (SUMS) {
        __shared__ double part[2][NT / 32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sumW += __shfl_down_sync(0xffffffffu, sumW, o);
            sumK += __shfl_down_sync(0xffffffffu, sumK, o);
        }
        if ((threadIdx.x & 31) == 0) {
            part[0][threadIdx.x >> 5] = sumW;
            part[1][threadIdx.x >> 5] = sumK;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double a = 0.0, b = 0.0;
            for (int w = 0; w < (int)(blockDim.x + 31) / 32; w++) {
                a += part[0][w];
                b += part[1][w];
            }
            partial[blockIdx.x] = a;
            partial[gridDim.x + blockIdx.x] = b;
        }
    }
}

// Variant "pipe": the same staple arithmetic as force_kernel, with the link loads software-pipelined by hand.
// Each staple is Z = op(a) op(b); A += Z op(c).  With 254 registers only 8 warps are resident per SM, so a
// wait on a group of loads is exposed; here the (a, b) links of the NEXT staple are requested before the
// second product of the current one and c before its first product, so every load has one 3x3 product
// (216 DFMA) of cover.  Live matrices at a product: A, Pm, Z, c and the two in flight = 216 registers (fp64).
template <typename T, bool FUSED>
__global__ void __launch_bounds__(256) force_pipe_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */,
                                                         const T eps, const pair_t<T> *__restrict__ U,
                                                         pair_t<T> *__restrict__ out) {
    const Site st = tile_site(lat, tile, threadIdx.x);
    const int V = lat.V;
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);
    int df[4], db[4];
#pragma unroll
    for (int d = 0; d < 4; d++) {
        df[d] = dfwd(lat, st, d);
        db[d] = dbwd(lat, st, d);
    }
    auto fwd = [&](int d) { return d == 0 ? df[0] : d == 1 ? df[1] : d == 2 ? df[2] : df[3]; };
    auto bwd = [&](int d) { return d == 0 ? db[0] : d == 1 ? db[1] : d == 2 ? db[2] : db[3]; };

    M3<T> Xa, Xb;  // operands (a, b) of the next staple, in flight across loop iterations
    load_link(Xa, U, V, 1, cb_of(lat, st.s + df[0], par ^ 1));  // mu = 0, nu = 1: U_nu(x+mu)
    load_link(Xb, U, V, 0, cb_of(lat, st.s + df[1], par ^ 1));  //                 U_mu(x+nu)

#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int dfm = fwd(mu);
        const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);  // x + mu
        M3<T> A, Pm, Um, Z, C;
        if (FUSED) load_link_rw(Pm, out, V, mu, cb);
        zero(A);
#pragma unroll
        for (int k = 1; k < 4; k++) {
            const int nu = (mu + k) & 3;
            const int dbn = bwd(nu);
            const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);  // x - nu
            // up staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
            load_link(C, U, V, nu, cb);
            mul<false, true, false>(Z, Xa, Xb);
            load_link(Xa, U, V, nu, cb_of(lat, st.s + dfm + dbn, par));  // U_nu(x+mu-nu)
            load_link(Xb, U, V, mu, cb_mn);                              // U_mu(x-nu)
            mul<false, true, true>(A, Z, C);
            // down staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
            load_link(C, U, V, nu, cb_mn);
            mul<true, true, false>(Z, Xa, Xb);
            if (k < 3) {
                const int nn = (mu + k + 1) & 3;
                load_link(Xa, U, V, nn, cb_pm);                                   // U_nn(x+mu)
                load_link(Xb, U, V, mu, cb_of(lat, st.s + fwd(nn), par ^ 1));     // U_mu(x+nn)
            } else {
                load_link(Um, U, V, mu, cb);
            }
            mul<false, false, true>(A, Z, C);
        }
        if (mu < 3) {  // first staple of the next direction: mu' = mu+1, nu' = mu+2
            const int m1 = mu + 1, n1 = (mu + 2) & 3;
            load_link(Xa, U, V, n1, cb_of(lat, st.s + fwd(m1), par ^ 1));
            load_link(Xb, U, V, m1, cb_of(lat, st.s + fwd(n1), par ^ 1));
        }
        M3<T> W, F;
        mul<false, false, false>(W, Um, A);
        project_force(F, W, c);
        if (FUSED) {
#pragma unroll
            for (int e = 0; e < 9; e++) {
                Pm.re[e] = fma_(eps, F.re[e], Pm.re[e]);
                Pm.im[e] = fma_(eps, F.im[e], Pm.im[e]);
            }
            store_link(Pm, out, V, mu, cb);
        } else {
            store_link(F, out, V, mu, cb);
        }
    }
}

// Variant "plane": the force assembled plane by plane from closed loops W = U_mu(x) * staple, so that the
// (mu,nu) plaquette at x serves both F_mu(x) (+) and F_nu(x) (its dagger, -) and each own link starts two
// chains: 10 link loads and 9 products per plane = 60 loads + 54 products per site instead of 80 + 52.
// The kernel is bound by bytes through the L1 load path, so fewer loads is the lever.
// Only the anti-Hermitian traceless part of each loop enters F (the projection is linear), so the four
// accumulators are 9 reals each (3 diagonal imaginary parts, 3 complex off-diagonal differences).
template <typename T>
struct TAcc {
    T d[3];   // sum Im W_ii
    T xr[3];  // sum Re (W_ij - conj W_ji) for (ij) = (01), (02), (12)
    T xi[3];  // sum Im (W_ij - conj W_ji)
};

template <typename T>
__device__ __forceinline__ void tacc_zero(TAcc<T> &a) {
#pragma unroll
    for (int k = 0; k < 3; k++) a.d[k] = a.xr[k] = a.xi[k] = T(0);
}

// a += sgn * antiHermitian part of W (sgn = -1 adds the part of W^dagger)
template <int SGN, typename T>
__device__ __forceinline__ void tacc_add(TAcc<T> &a, const M3<T> &W) {
    const T s = T(SGN);
#pragma unroll
    for (int k = 0; k < 3; k++) a.d[k] += s * W.im[4 * k];
    const int I[3] = {0, 0, 1}, J[3] = {1, 2, 2};
#pragma unroll
    for (int k = 0; k < 3; k++) {
        a.xr[k] += s * (W.re[3 * I[k] + J[k]] - W.re[3 * J[k] + I[k]]);
        a.xi[k] += s * (W.im[3 * I[k] + J[k]] + W.im[3 * J[k] + I[k]]);
    }
}

// F = (i c)[(W - W^dag) - tr/3] from the accumulated parts (same formulas as project_force)
template <typename T>
__device__ __forceinline__ void tacc_force(M3<T> &F, const TAcc<T> &a, T c) {
    const T m = (a.d[0] + a.d[1] + a.d[2]) * T(1.0 / 3.0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        F.re[4 * k] = T(-2) * c * (a.d[k] - m);
        F.im[4 * k] = T(0);
    }
    const int I[3] = {0, 0, 1}, J[3] = {1, 2, 2};
#pragma unroll
    for (int k = 0; k < 3; k++) {
        F.re[3 * I[k] + J[k]] = -c * a.xi[k];
        F.im[3 * I[k] + J[k]] = c * a.xr[k];
        F.re[3 * J[k] + I[k]] = -c * a.xi[k];
        F.im[3 * J[k] + I[k]] = -c * a.xr[k];
    }
}

// all loops of the (mu,nu) plane through x that contain U_mu(x) or U_nu(x)
template <typename T>
__device__ __forceinline__ void plane_loops(TAcc<T> &am, TAcc<T> &an, const LatP &lat, const Site &st, int V,
                                            const pair_t<T> *__restrict__ U, int mu, int nu, int dfm, int dbm,
                                            int dfn, int dbn) {
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);
    const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);  // x - nu
    const int cb_mm = cb_of(lat, st.s + dbm, par ^ 1);  // x - mu
    M3<T> Uo, B, M, N;
    // lower loop of U_mu(x):  U_mu(x) U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
    load_link(Uo, U, V, mu, cb);
    load_link(B, U, V, nu, cb_of(lat, st.s + dfm + dbn, par));
    mul<false, true, false>(M, Uo, B);
    load_link(B, U, V, mu, cb_mn);
    mul<false, true, false>(N, M, B);
    load_link(B, U, V, nu, cb_mn);
    mul<false, false, false>(M, N, B);
    tacc_add<1>(am, M);
    // plaquette:  U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag  -> +F_mu, its dagger -> F_nu
    load_link(B, U, V, nu, cb_of(lat, st.s + dfm, par ^ 1));
    mul<false, false, false>(M, Uo, B);
    load_link(B, U, V, mu, cb_of(lat, st.s + dfn, par ^ 1));
    mul<false, true, false>(N, M, B);
    load_link(Uo, U, V, nu, cb);  // U_nu(x): closes the plaquette, then starts the lower loop of U_nu(x)
    mul<false, true, false>(M, N, Uo);
    tacc_add<1>(am, M);
    tacc_add<-1>(an, M);
    // lower loop of U_nu(x):  U_nu(x) U_mu(x+nu-mu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    load_link(B, U, V, mu, cb_of(lat, st.s + dfn + dbm, par));
    mul<false, true, false>(M, Uo, B);
    load_link(B, U, V, nu, cb_mm);
    mul<false, true, false>(N, M, B);
    load_link(B, U, V, mu, cb_mm);
    mul<false, false, false>(M, N, B);
    tacc_add<1>(an, M);
}

template <typename T, bool FUSED>
__global__ void __launch_bounds__(256) force_plane_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */,
                                                          const T eps, const pair_t<T> *__restrict__ U,
                                                          pair_t<T> *__restrict__ out) {
    const Site st = tile_site(lat, tile, threadIdx.x);
    const int V = lat.V;
    const int cb = cb_of(lat, st.s, st.par);
    int df[4], db[4];
#pragma unroll
    for (int d = 0; d < 4; d++) {
        df[d] = dfwd(lat, st, d);
        db[d] = dbwd(lat, st, d);
    }
    // a0..a3 belong to directions mu, mu+1, mu+2, mu+3 (mod 4) of the current iteration: the accumulators
    // rotate by register moves so that the loop body is compiled once
    TAcc<T> a0, a1, a2, a3;
    tacc_zero(a0);
    tacc_zero(a1);
    tacc_zero(a2);
    tacc_zero(a3);
#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int n1 = (mu + 1) & 3, n2 = (mu + 2) & 3;
        const int dfm = mu == 0 ? df[0] : mu == 1 ? df[1] : mu == 2 ? df[2] : df[3];
        const int dbm = mu == 0 ? db[0] : mu == 1 ? db[1] : mu == 2 ? db[2] : db[3];
        const int df1 = n1 == 0 ? df[0] : n1 == 1 ? df[1] : n1 == 2 ? df[2] : df[3];
        const int db1 = n1 == 0 ? db[0] : n1 == 1 ? db[1] : n1 == 2 ? db[2] : db[3];
        plane_loops(a0, a1, lat, st, V, U, mu, n1, dfm, dbm, df1, db1);  // planes (0,1) (1,2) (2,3) (3,0)
        if (mu < 2) {                                                      // planes (0,2) (1,3)
            const int df2 = n2 == 0 ? df[0] : n2 == 1 ? df[1] : n2 == 2 ? df[2] : df[3];
            const int db2 = n2 == 0 ? db[0] : n2 == 1 ? db[1] : n2 == 2 ? db[2] : db[3];
            plane_loops(a0, a2, lat, st, V, U, mu, n2, dfm, dbm, df2, db2);
        }
        const TAcc<T> t = a0;
        a0 = a1;
        a1 = a2;
        a2 = a3;
        a3 = t;
    }
    // after four rotations a_k is direction k again
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        M3<T> F;
        tacc_force(F, mu == 0 ? a0 : mu == 1 ? a1 : mu == 2 ? a2 : a3, c);
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

// Variant "link": one thread per (site, mu).  The block owns the same 4-D tile; thread j < nsite handles
// mu = 0, the next nsite threads mu = 1, ... (mu is warp-uniform when nsite is a multiple of 32).  A
// quarter of the per-thread state of the per-site variant: more warps in flight per SM.
template <typename T, bool FUSED, int NT>
__global__ void __launch_bounds__(NT) force_link_kernel(const LatP lat, const TileP tile, const T c, const T eps,
                                                       const pair_t<T> *__restrict__ U,
                                                       pair_t<T> *__restrict__ out) {
    const int nsite = tile.tsp * tile.npar;
    const int mu = threadIdx.x / nsite;
    const Site st = tile_site(lat, tile, threadIdx.x - mu * nsite);
    const int V = lat.V;
    const int par = st.par;
    const int cb = cb_of(lat, st.s, par);
    int df[4], db[4];
#pragma unroll
    for (int d = 0; d < 4; d++) {
        df[d] = dfwd(lat, st, d);
        db[d] = dbwd(lat, st, d);
    }
    const int dfm = mu == 0 ? df[0] : mu == 1 ? df[1] : mu == 2 ? df[2] : df[3];
    const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);  // x + mu
    M3<T> A;
    zero(A);
#pragma unroll 1
    for (int k = 1; k < 4; k++) {
        const int nu = (mu + k) & 3;
        const int dfn = nu == 0 ? df[0] : nu == 1 ? df[1] : nu == 2 ? df[2] : df[3];
        const int dbn = nu == 0 ? db[0] : nu == 1 ? db[1] : nu == 2 ? db[2] : db[3];
        const int cb_pn = cb_of(lat, st.s + dfn, par ^ 1);      // x + nu
        const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);      // x - nu
        const int cb_pmmn = cb_of(lat, st.s + dfm + dbn, par);  // x + mu - nu
        M3<T> X, Y, Z;
        load_link(X, U, V, nu, cb_pm);
        load_link(Y, U, V, mu, cb_pn);
        mul<false, true, false>(Z, X, Y);
        load_link(X, U, V, nu, cb);
        mul<false, true, true>(A, Z, X);
        load_link(X, U, V, nu, cb_pmmn);
        load_link(Y, U, V, mu, cb_mn);
        mul<true, true, false>(Z, X, Y);
        load_link(X, U, V, nu, cb_mn);
        mul<false, false, true>(A, Z, X);
    }
    M3<T> Um, W;
    load_link(Um, U, V, mu, cb);
    mul<false, false, false>(W, Um, A);
    M3<T> F;
    project_force(F, W, c);
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

// ---- host side: tile choice -------------------------------------------------------------------

// all divisors of n (even ones only if `even`)
static int divisors(int n, bool even, int *out) {
    int k = 0;
    for (int d = 1; d <= n; d++)
        if (n % d == 0 && (!even || (d & 1) == 0)) out[k++] = d;
    return k;
}

// Pick tile extents dividing L with T0 even and `threads` = T0/2*T1*T2*T3*npar as close to the target
// as possible (never above it), preferring a long x extent (coalescing: T0/2 consecutive sites are
// contiguous in memory) and then the smallest surface (L1 reuse of neighbour links).
// QCD_TILE="tx,ty,tz,tt" overrides for block-shape sweeps (the paper's N_t tuning).
static TileP choose_tile(const LatP &lat, int subset, int target, const int *tuned = nullptr) {
    TileP tp;
    tp.npar = subset == QCD_ALL ? 2 : 1;
    tp.par0 = subset == QCD_ODD ? 1 : 0;
    int best[4] = {2, 1, 1, 1};
    const char *env = getenv("QCD_TILE");
    int e[4];
    bool have = false;
    // the environment (sweeps) wins over the tuner's database entry, which wins over the heuristic below
    bool given = env && sscanf(env, "%d,%d,%d,%d", &e[0], &e[1], &e[2], &e[3]) == 4;
    if (!given && tuned && tuned[0]) {
        memcpy(e, tuned, sizeof e);
        given = true;
    }
    if (given) {
        have = true;
        for (int d = 0; d < 4; d++)
            if (e[d] < 1 || lat.L[d] % e[d]) have = false;
        if (e[0] & 1) have = false;
        if (have && (long)(e[0] / 2) * e[1] * e[2] * e[3] * tp.npar > target) have = false;
        if (have) memcpy(best, e, sizeof e);
    }
    if (!have) {
        int dv[4][128], nd[4];
        for (int d = 0; d < 4; d++) nd[d] = divisors(lat.L[d], d == 0, dv[d]);
        double best_score = -1e300;
        for (int a = 0; a < nd[0]; a++)
            for (int b = 0; b < nd[1]; b++)
                for (int cc = 0; cc < nd[2]; cc++)
                    for (int d = 0; d < nd[3]; d++) {
                        const int t[4] = {dv[0][a], dv[1][b], dv[2][cc], dv[3][d]};
                        const long threads = (long)(t[0] / 2) * t[1] * t[2] * t[3] * tp.npar;
                        if (threads > target) continue;
                        const double vol = (double)t[0] * t[1] * t[2] * t[3];
                        double surf = 0;
                        for (int k = 0; k < 4; k++) surf += vol / t[k];
                        // more threads first; then x extent up to 32 (256-byte rows per parity in fp64; measured best on
                        // B200, profiles/r01c_force_sweeps.md); then compactness
                        const double score = threads * 1e6 + (t[0] >= 32 ? 32 : t[0]) * 1e3 - surf / vol * 100.0;
                        if (score > best_score) {
                            best_score = score;
                            memcpy(best, t, sizeof t);
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

// QCD_FORCE_VARIANT selects the kernel for block-shape / mapping sweeps (the paper's N_t tuning,
// PAPER.md:57): "site" (default) = one thread per site, 128-thread blocks; "site256" = the same kernel in
// 256-thread blocks with the momenta loaded early; "pipe" / "plane" = the hand-pipelined and the plane-wise
// kernels above; "link" = one thread per (site, mu) with QCD_FORCE_THREADS in {256, 512} threads per block.
// kernel variant and tile for this launch: QCD_FORCE_VARIANT (sweeps) > tuner database (tune.cu) > default
struct ForceSel {
    int variant;
    int tile[4];
};
static const char *const kVariantNames[] = {"site", "site256", "pipe", "plane", "link", "tile", "plaq"};

static ForceSel force_sel(const qcd_lattice *lat, int prec, int subset) {
    ForceSel fs = {QCD_FORCE_SITE, {0, 0, 0, 0}};
    TuneCfg cfg;
    if (tune_lookup(lat, prec, subset, QCD_KERNEL_FORCE, cfg)) {
        fs.variant = cfg.variant;
        memcpy(fs.tile, cfg.tile, sizeof fs.tile);
    }
    const char *v = getenv("QCD_FORCE_VARIANT");
    if (v) {
        fs.variant = QCD_FORCE_SITE;
        for (int k = 0; k <= QCD_FORCE_PLAQ; k++)
            if (!strcmp(v, kVariantNames[k])) fs.variant = k;
    }
    return fs;
}

template <typename T, bool FUSED>
static void launch_force_v(const qcd_lattice *lat, int subset, const ForceSel &fs, T c, T eps, const pair_t<T> *U,
                           pair_t<T> *out, cudaStream_t st) {
    const int *tuned = fs.tile;
    const int var = fs.variant;
    if (var != QCD_FORCE_SITE256 && var != QCD_FORCE_PLANE && var != QCD_FORCE_PIPE && var != QCD_FORCE_LINK) {
        // default: 128-thread blocks, three per SM (168 registers in fp64, 12 warps/SM); measured best at
        // 32^3x64 in both precisions (profiles/r01c_force_sweeps.md)
        const TileP tp = choose_tile(lat->p, subset, 128, tuned);
        const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
        if (getenv("QCD_SU3_REC"))  // sweep knob: SU(3) links only (two-row loads); measured no gain, off by default
            force_kernel<T, FUSED, false, false, 128, 3, true><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out, T(0), nullptr, T(0), T(0));
        else  // fp32 has the registers to hold the momenta from the start of a direction (-5 %); fp64 does not (+12 %)
            force_kernel<T, FUSED, sizeof(T) == 4, false, 128, 3><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out, T(0), nullptr, T(0), T(0));
        return;
    }
    if (var == QCD_FORCE_SITE256) {  // 256-thread blocks, one per SM in fp64 (254 registers), momenta loaded early
        const TileP tp = choose_tile(lat->p, subset, 256, tuned);
        const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
        const char *pm = getenv("QCD_EARLY_P");  // sweep knob; default on
        if (!pm || atoi(pm))
            force_kernel<T, FUSED, true, false><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out, T(0), nullptr, T(0), T(0));
        else
            force_kernel<T, FUSED, false, false><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out, T(0), nullptr, T(0), T(0));
        return;
    }
    if (var == QCD_FORCE_PLANE) {
        const TileP tp = choose_tile(lat->p, subset, 256, tuned);
        const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
        force_plane_kernel<T, FUSED><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out);
        return;
    }
    if (var == QCD_FORCE_PIPE) {
        const TileP tp = choose_tile(lat->p, subset, 256, tuned);
        const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
        force_pipe_kernel<T, FUSED><<<blocks, tp.tsp * tp.npar, 0, st>>>(lat->p, tp, c, eps, U, out);
        return;
    }
    const char *t = getenv("QCD_FORCE_THREADS");
    const int nt = t ? atoi(t) : 512;
    const TileP tp = choose_tile(lat->p, subset, nt == 256 ? 64 : 128, tuned);
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    const int threads = 4 * tp.tsp * tp.npar;
    if (nt == 256) force_link_kernel<T, FUSED, 256><<<blocks, threads, 0, st>>>(lat->p, tp, c, eps, U, out);
    else force_link_kernel<T, FUSED, 512><<<blocks, threads, 0, st>>>(lat->p, tp, c, eps, U, out);
}

template <typename T>
static int launch_force_t(const qcd_lattice *lat, int subset, const ForceSel &fs, double beta, double eps,
                          const void *U, void *out, bool fused, cudaStream_t st) {
    const T c = (T)(beta / 12.0);
    if (fused) launch_force_v<T, true>(lat, subset, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, st);
    else launch_force_v<T, false>(lat, subset, fs, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, st);
    return check_launch(fused ? "force_mom_update" : "gauge_force");
}

// Anisotropic force (plane weights ws, wt; eps = 1 folds a step size into the weights)
template <typename T>
static int launch_force_aniso_t(const qcd_lattice *lat, int subset, double ws, double wt, double eps, const void *U,
                                void *out, bool fused, cudaStream_t st) {
    const TileP tp = choose_tile(lat->p, subset, 128);
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    const T c = (T)(1.0 / 12.0);
    if (fused)
        force_kernel<T, true, false, false, 128, 3, false, true><<<blocks, tp.tsp * tp.npar, 0, st>>>(
            lat->p, tp, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0), nullptr, (T)ws, (T)wt);
    else
        force_kernel<T, false, false, false, 128, 3, false, true><<<blocks, tp.tsp * tp.npar, 0, st>>>(
            lat->p, tp, c, (T)eps, (const pair_t<T> *)U, (pair_t<T> *)out, T(0), nullptr, (T)ws, (T)wt);
    return check_launch(fused ? "force_mom_update_aniso" : "gauge_force_aniso");
}

int launch_gauge_force_aniso(const qcd_lattice *lat, int prec, int subset, double ws, double wt, double eps,
                             const void *U, void *out, bool fused_mom, cudaStream_t st) {
    return prec == QCD_F64 ? launch_force_aniso_t<double>(lat, subset, ws, wt, eps, U, out, fused_mom, st)
                           : launch_force_aniso_t<float>(lat, subset, ws, wt, eps, U, out, fused_mom, st);
}

// Force + momentum update with the plaquette and kinetic-energy sums as by-products (subset ALL).
// out[0] = plaquette average of U, out[1] = K of the updated P.  ws: 2 x blocks doubles.
template <typename T>
static int launch_force_sums_t(const qcd_lattice *lat, double beta, double eps, const void *U, void *P, double *out,
                               double *ws, cudaStream_t st) {
    const TileP tp = choose_tile(lat->p, QCD_ALL, 128);
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    if ((size_t)2 * blocks > lat->workspace_doubles) {
        set_error("force_mom_update_sums: workspace too small");
        return QCD_EWORKSPACE;
    }
    force_kernel<T, true, false, false, 128, 3, false, false, true><<<blocks, tp.tsp * tp.npar, 0, st>>>(
        lat->p, tp, (T)(beta / 12.0), (T)eps, (const pair_t<T> *)U, (pair_t<T> *)P, T(0), nullptr, T(0), T(0), ws);
    QCD_TRY_RC(check_launch("force_mom_update_sums"));
    QCD_TRY_RC(launch_sum_partials(ws, blocks, 1.0 / (72.0 * (double)lat->p.V), out, st));
    return launch_sum_partials(ws + blocks, blocks, 1.0, out + 1, st);
}

int launch_force_sums(const qcd_lattice *lat, int prec, double beta, double eps, const void *U, void *P, double *out,
                      double *ws, cudaStream_t st) {
    return prec == QCD_F64 ? launch_force_sums_t<double>(lat, beta, eps, U, P, out, ws, st)
                           : launch_force_sums_t<float>(lat, beta, eps, U, P, out, ws, st);
}

// Single-pass MD step: P += eps_p F(U); Uout = reunit(exp(i eps_u P) U).  Subset ALL only (every link moves).
template <typename T>
static int launch_md_single_t(const qcd_lattice *lat, double beta, double eps_p, double eps_u, const void *U, void *P,
                              void *Uout, cudaStream_t st) {
    const TileP tp = choose_tile(lat->p, QCD_ALL, 128);
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    force_kernel<T, true, sizeof(T) == 4, true, 128, 3><<<blocks, tp.tsp * tp.npar, 0, st>>>(
        lat->p, tp, (T)(beta / 12.0), (T)eps_p, (const pair_t<T> *)U, (pair_t<T> *)P, (T)eps_u, (pair_t<T> *)Uout, T(0), T(0));
    return check_launch("md_step_single_pass");
}

int launch_md_single(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U, void *P,
                     void *Uout, cudaStream_t st) {
    return prec == QCD_F64 ? launch_md_single_t<double>(lat, beta, eps_p, eps_u, U, P, Uout, st)
                           : launch_md_single_t<float>(lat, beta, eps_p, eps_u, U, P, Uout, st);
}

// Kernel choice.  Default: the plain staple kernels of this file (the definition, valid for arbitrary 3x3
// matrices and for subsets).  QCD_FORCE_VARIANT = site | site256 | pipe | plane | link | tile | plaq selects a variant for the
// block-shape / mapping sweeps (the paper's N_t auto-tuning); tile (force_tile.cu) and plaq
// (force_plaq.cu, needs unitary links) exist for subset ALL only.  DESIGN.md section 6 has the measurements.
int launch_gauge_force(const qcd_lattice *lat, int prec, int subset, double beta, double eps, const void *U,
                       void *out, bool fused_mom, cudaStream_t st) {
    const ForceSel fs = force_sel(lat, prec, subset);
    if (subset == QCD_ALL && fs.variant == QCD_FORCE_PLAQ)
        return launch_gauge_force_plaq(lat, prec, beta, eps, U, out, fused_mom, st);
    if (subset == QCD_ALL && fs.variant == QCD_FORCE_TILE) {
        const int rc = launch_gauge_force_tile(lat, prec, beta, eps, U, out, fused_mom, st);
        if (rc >= 0) return rc;
    }
    return prec == QCD_F64 ? launch_force_t<double>(lat, subset, fs, beta, eps, U, out, fused_mom, st)
                           : launch_force_t<float>(lat, subset, fs, beta, eps, U, out, fused_mom, st);
}

}  // namespace qcd
