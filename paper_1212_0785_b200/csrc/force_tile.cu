// force_tile.cu — Wilson gauge force (O7), staple form, with the tile's own links staged in shared memory.
//
// Measured on B200 (profiles/r01b_*): the staple kernels of force.cu are bound by the L1 global-load path,
// not by HBM or the FP64 pipe — an LDG costs about two cycles per 128-byte line it touches whatever its
// width, i.e. at most ~62 B/clk/SM, while shared memory delivers 128 B/clk/SM.  A site needs 80 link
// loads (6 per staple pair + U_mu(x), for 4 x 3 (mu,nu)), and about 70 % of them hit links of the block's
// own 4-D tile.  So the block first copies the four own links of each of its sites into shared memory
// (one coalesced pass), and every later load of a link whose site lies inside the tile is an LDS; only
// links of sites outside the tile (the halo) still go through L1 as LDGs.
//
// One thread per site, subset ALL; arithmetic identical to force_kernel in force.cu.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

constexpr int FT_MAX_SITES = 256;

template <typename T>
__device__ __forceinline__ void lds_link(M3<T> &m, const pair_t<T> *s, int N, int mu, int slot) {
    const pair_t<T> *p = s + (mu * 9) * N + slot;
#pragma unroll
    for (int e = 0; e < 9; e++) {
        const pair_t<T> v = p[e * N];
        m.re[e] = v.x;
        m.im[e] = v.y;
    }
}

// link `mu` of a neighbour: from the tile copy if it lies in the tile (slot >= 0), else from global memory
template <typename T>
__device__ __forceinline__ void get_link(M3<T> &m, const pair_t<T> *s, int N, const pair_t<T> *__restrict__ U, int V,
                                         int mu, int slot, int cb) {
    if (slot >= 0) lds_link(m, s, N, mu, slot);
    else load_link(m, U, V, mu, cb);
}

__device__ __forceinline__ int pick4(const int a[4], int i) { return i == 0 ? a[0] : i == 1 ? a[1] : i == 2 ? a[2] : a[3]; }

template <typename T, bool FUSED>
__global__ void __launch_bounds__(FT_MAX_SITES) force_tile_kernel(const LatP lat, const TileP tile, const T c /* beta/12 */,
                                                                  const T eps, const pair_t<T> *__restrict__ U,
                                                                  pair_t<T> *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    pair_t<T> *sU = (pair_t<T> *)smem_raw;
    const int N = 2 * tile.tsp;
    const int V = lat.V;
    const int j = threadIdx.x;  // slot: parity-major, x fastest

    // tile-local coordinates of slot j
    int o[4], cl[4];
    {
        int b = blockIdx.x;
        o[0] = (b % tile.nt[0]) * tile.T[0];
        b /= tile.nt[0];
        o[1] = (b % tile.nt[1]) * tile.T[1];
        b /= tile.nt[1];
        o[2] = (b % tile.nt[2]) * tile.T[2];
        o[3] = (b / tile.nt[2]) * tile.T[3];
    }
    const int par = j >= tile.tsp ? 1 : 0;
    const int hx = tile.T[0] >> 1;
    const int lin = j - par * tile.tsp;
    {
        int r = lin;
        const int jx = r % hx;
        r /= hx;
        cl[1] = r % tile.T[1];
        r /= tile.T[1];
        cl[2] = r % tile.T[2];
        cl[3] = r / tile.T[2];
        cl[0] = 2 * jx + ((cl[1] + cl[2] + cl[3] + o[1] + o[2] + o[3] + par) & 1);
    }
    Site st;
    st.par = par;
    st.s = 0;
#pragma unroll
    for (int d = 0; d < 4; d++) {
        st.c[d] = o[d] + cl[d];
        st.s += st.c[d] * lat.stride[d];
    }
    const int cb = cb_of(lat, st.s, par);

    // stage the own links
    {
        const pair_t<T> *g = U + unit_index(36, 0, cb);
        pair_t<T> *s = sU + j;
#pragma unroll 12
        for (int e = 0; e < 36; e++) s[e * N] = __ldg(g + e * CHUNK);
    }

    // neighbour bookkeeping: global index steps, tile-slot steps (within the parity block), in-tile flags
    int df[4], db[4], sf[4], sb[4];
    bool okf[4], okb[4];
    {
        const int sd[4] = {0, hx, hx * tile.T[1], hx * tile.T[1] * tile.T[2]};
#pragma unroll
        for (int d = 0; d < 4; d++) {
            df[d] = dfwd(lat, st, d);
            db[d] = dbwd(lat, st, d);
            okf[d] = cl[d] + 1 < tile.T[d];
            okb[d] = cl[d] > 0;
            sf[d] = d == 0 ? (cl[0] & 1) : sd[d];
            sb[d] = d == 0 ? -((cl[0] & 1) ^ 1) : -sd[d];
        }
    }
    const int base_same = par * tile.tsp + lin;        // slot of a site of the same parity, before steps
    const int base_opp = (par ^ 1) * tile.tsp + lin;   // slot of a site of the opposite parity, before steps
    __syncthreads();

#pragma unroll 1
    for (int mu = 0; mu < 4; mu++) {
        const int dfm = pick4(df, mu), sfm = pick4(sf, mu);
        const bool okm = mu == 0 ? okf[0] : mu == 1 ? okf[1] : mu == 2 ? okf[2] : okf[3];
        const int cb_pm = cb_of(lat, st.s + dfm, par ^ 1);
        const int sl_pm = okm ? base_opp + sfm : -1;
        M3<T> A;
        zero(A);
#pragma unroll 1
        for (int k = 1; k < 4; k++) {
            const int nu = (mu + k) & 3;
            const int dfn = pick4(df, nu), dbn = pick4(db, nu), sfn = pick4(sf, nu), sbn = pick4(sb, nu);
            const bool okfn = nu == 0 ? okf[0] : nu == 1 ? okf[1] : nu == 2 ? okf[2] : okf[3];
            const bool okbn = nu == 0 ? okb[0] : nu == 1 ? okb[1] : nu == 2 ? okb[2] : okb[3];
            const int cb_pn = cb_of(lat, st.s + dfn, par ^ 1);
            const int cb_mn = cb_of(lat, st.s + dbn, par ^ 1);
            const int cb_pmmn = cb_of(lat, st.s + dfm + dbn, par);
            const int sl_pn = okfn ? base_opp + sfn : -1;
            const int sl_mn = okbn ? base_opp + sbn : -1;
            const int sl_pmmn = (okm && okbn) ? base_same + sfm + sbn : -1;
            M3<T> X, Y, Z;
            // up staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
            get_link(X, sU, N, U, V, nu, sl_pm, cb_pm);
            get_link(Y, sU, N, U, V, mu, sl_pn, cb_pn);
            mul<false, true, false>(Z, X, Y);
            lds_link(X, sU, N, nu, j);
            mul<false, true, true>(A, Z, X);
            // down staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
            get_link(X, sU, N, U, V, nu, sl_pmmn, cb_pmmn);
            get_link(Y, sU, N, U, V, mu, sl_mn, cb_mn);
            mul<true, true, false>(Z, X, Y);
            get_link(X, sU, N, U, V, nu, sl_mn, cb_mn);
            mul<false, false, true>(A, Z, X);
        }
        M3<T> Um, W;
        lds_link(Um, sU, N, mu, j);
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
}

// tile: exactly the block's threads = sites (both parities), T0 even and long (coalescing), compact otherwise.
// Returns false if the lattice has no tile of at least 32 sites that divides it (tiny lattices: caller falls
// back to force.cu).  QCD_TILE="tx,ty,tz,tt" overrides (block-shape sweeps).
static bool choose_tile_sites(const LatP &lat, TileP &tp) {
    tp.npar = 2;
    tp.par0 = 0;
    int best[4] = {0, 0, 0, 0};
    const char *env = getenv("QCD_TILE");
    int e[4];
    bool have = false;
    if (env && sscanf(env, "%d,%d,%d,%d", &e[0], &e[1], &e[2], &e[3]) == 4) {
        have = true;
        for (int d = 0; d < 4; d++)
            if (e[d] < 1 || lat.L[d] % e[d]) have = false;
        if (e[0] & 1) have = false;
        if (have && (long)e[0] * e[1] * e[2] * e[3] > FT_MAX_SITES) have = false;
        if (have) memcpy(best, e, sizeof e);
    }
    if (!have) {
        double best_score = -1e300;
        for (int a = 2; a <= lat.L[0]; a += 2)
            for (int b = 1; b <= lat.L[1]; b++)
                for (int cc = 1; cc <= lat.L[2]; cc++)
                    for (int d = 1; d <= lat.L[3]; d++) {
                        if (lat.L[0] % a || lat.L[1] % b || lat.L[2] % cc || lat.L[3] % d) continue;
                        const long n = (long)a * b * cc * d;
                        if (n > FT_MAX_SITES) continue;
                        const double halo = 1.0 / a + 1.0 / b + 1.0 / cc + 1.0 / d;
                        const double score = n * 1e3 + (a >= 16 ? 16 : a) * 10.0 - halo;
                        if (score > best_score) {
                            best_score = score;
                            best[0] = a; best[1] = b; best[2] = cc; best[3] = d;
                        }
                    }
    }
    if (best[0] == 0) return false;
    for (int d = 0; d < 4; d++) {
        tp.T[d] = best[d];
        tp.nt[d] = lat.L[d] / best[d];
    }
    tp.tsp = (tp.T[0] / 2) * tp.T[1] * tp.T[2] * tp.T[3];
    return 2 * tp.tsp >= 32;
}

template <typename T, bool FUSED>
static void launch_tile_v(const qcd_lattice *lat, const TileP &tp, T c, T eps, const pair_t<T> *U, pair_t<T> *out,
                          cudaStream_t st) {
    const int N = 2 * tp.tsp;
    const size_t smem = (size_t)36 * N * sizeof(pair_t<T>);
    static bool attr_set = false;  // per instantiation
    if (!attr_set) {
        cudaFuncSetAttribute(force_tile_kernel<T, FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             36 * FT_MAX_SITES * (int)sizeof(pair_t<T>));
        attr_set = true;
    }
    const int blocks = tp.nt[0] * tp.nt[1] * tp.nt[2] * tp.nt[3];
    force_tile_kernel<T, FUSED><<<blocks, N, smem, st>>>(lat->p, tp, c, eps, U, out);
}

// returns QCD_OK, QCD_ECUDA, or -1 if this kernel does not apply to the lattice
int launch_gauge_force_tile(const qcd_lattice *lat, int prec, double beta, double eps, const void *U, void *out,
                            bool fused_mom, cudaStream_t st) {
    TileP tp;
    if (!choose_tile_sites(lat->p, tp)) return -1;
    const double c = beta / 12.0;
    if (prec == QCD_F64) {
        if (fused_mom) launch_tile_v<double, true>(lat, tp, c, eps, (const double2 *)U, (double2 *)out, st);
        else launch_tile_v<double, false>(lat, tp, c, eps, (const double2 *)U, (double2 *)out, st);
    } else {
        if (fused_mom) launch_tile_v<float, true>(lat, tp, (float)c, (float)eps, (const float2 *)U, (float2 *)out, st);
        else launch_tile_v<float, false>(lat, tp, (float)c, (float)eps, (const float2 *)U, (float2 *)out, st);
    }
    return check_launch(fused_mom ? "force_mom_update(tile)" : "gauge_force(tile)");
}

}  // namespace qcd
