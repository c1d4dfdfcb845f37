// update.cu — site-local updates: momentum update P += eps*F (O10), link update
// U <- exp(i eps P) U (O8, O10) and reunitarisation (O9), the last two fused in registers on request.
// One thread per link; every load and store is a coalesced 16-byte (fp64) / 8-byte (fp32) access.
#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

// MODE 0: U <- exp(i eps P) U;  1: same, then reunitarise;  2: reunitarise only
template <typename T, int MODE>
__global__ void __launch_bounds__(256) link_update_kernel(const int V, const int begin, const int count, const T eps,
                                                          const pair_t<T> *__restrict__ P, pair_t<T> *__restrict__ U) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const int cb = begin + i;
    const int mu = blockIdx.y;
    M3<T> R;
    if (MODE == 2) {
        load_link_rw(R, U, V, mu, cb);
    } else {
        M3<T> Q, Ul, E;
        load_link_cs(Q, P, V, mu, cb);  // touched once: streaming
        load_link_rw(Ul, U, V, mu, cb);
        if (MODE == 1) {
            expi_herm_scaled<2>(E, Q, eps);
            mul_top2(R, E, Ul);  // reunit rebuilds row 2
        } else {
            expi_herm_scaled<3>(E, Q, eps);
            mul<false, false, false>(R, E, Ul);
        }
    }
    if (MODE >= 1) reunit(R);
    store_link(R, U, V, mu, cb);
}

// Link update of the interior timeslices of a slab lattice fused with the halo transport ("one
// exchange per force evaluation ... over NVLink peer stores"): the thread that has the new link of a
// boundary timeslice in registers also stores it into the neighbour's halo — the first interior timeslice (te = 1)
// into the upper halo of `lo` (spatial links only: nobody reads a halo's time links from below), the last interior
// timeslice into the lower halo of `hi` (all four).  lo_U / hi_U may be peer-GPU memory or NULL.  The slab's own
// halos are NOT written (the neighbours' launches write them).  MODE as in link_update_kernel (0 or 1).
template <typename T, int MODE>
__global__ void __launch_bounds__(256) link_update_push_kernel(const LatP lat, const T eps,
                                                               const pair_t<T> *__restrict__ P,
                                                               pair_t<T> *__restrict__ U, const LatP lo,
                                                               pair_t<T> *__restrict__ lo_U, const LatP hi,
                                                               pair_t<T> *__restrict__ hi_U) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= lat.V) return;
    const Site st = site_of_cb(lat, cb);
    const int t = st.c[3];
    if (t < lat.t0 || t >= lat.t1) return;
    const int mu = blockIdx.y;
    M3<T> Q, Ul, E, R;
    load_link_cs(Q, P, lat.V, mu, cb);
    load_link_rw(Ul, U, lat.V, mu, cb);
    if (MODE == 1) {
        expi_herm_scaled<2>(E, Q, eps);
        mul_top2(R, E, Ul);
        reunit(R);
    } else {
        expi_herm_scaled<3>(E, Q, eps);
        mul<false, false, false>(R, E, Ul);
    }
    store_link(R, U, lat.V, mu, cb);
    const int sx = st.c[0] + lat.L[0] * (st.c[1] + lat.L[1] * st.c[2]);  // spatial index, the same on every slab
    const int Vs = lat.L[0] * lat.L[1] * lat.L[2];
    if (t == 1 && lo_U != nullptr && mu < 3) {
        const int tp = lo.L[3] - 1;
        const int par = (st.c[0] + st.c[1] + st.c[2] + tp) & 1;
        store_link(R, lo_U, lo.V, mu, par * lo.Vh + ((sx + Vs * tp) >> 1));
    }
    if (t == lat.L[3] - 2 && hi_U != nullptr) {
        const int par = (st.c[0] + st.c[1] + st.c[2]) & 1;  // tp = 0
        store_link(R, hi_U, hi.V, mu, par * hi.Vh + (sx >> 1));
    }
}

template <typename T>
__global__ void __launch_bounds__(256) mom_update_kernel(const int V, const int begin, const int count, const T eps,
                                                         const pair_t<T> *__restrict__ F, pair_t<T> *__restrict__ P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const unsigned base = unit_index(36, blockIdx.y * 9, begin + i);
    pair_t<T> f[9], p[9];
#pragma unroll
    for (int e = 0; e < 9; e++) {
        f[e] = __ldg(F + base + e * CHUNK);
        p[e] = P[base + e * CHUNK];
    }
#pragma unroll
    for (int e = 0; e < 9; e++) {
        p[e].x = fma_(eps, f[e].x, p[e].x);
        p[e].y = fma_(eps, f[e].y, p[e].y);
        P[base + e * CHUNK] = p[e];
    }
}

// threads per block N_t: the tuner's database entry or the default
static int tuned_threads(const qcd_lattice *lat, int prec, int subset, int kernel, int dflt) {
    TuneCfg cfg;
    return tune_lookup(lat, prec, subset, kernel, cfg) && cfg.threads ? cfg.threads : dflt;
}

template <typename T>
static int launch_link_update_t(const qcd_lattice *lat, int subset, double eps, const void *P, void *U, int mode,
                                cudaStream_t st) {
    int begin, count;
    subset_range(lat->p, subset, begin, count);
    const int threads = tuned_threads(lat, sizeof(T) == 8 ? QCD_F64 : QCD_F32, subset, QCD_KERNEL_LINK_UPDATE, 128);
    const dim3 grid((count + threads - 1) / threads, 4);
    const pair_t<T> *p = (const pair_t<T> *)P;
    pair_t<T> *u = (pair_t<T> *)U;
    if (mode == 0) link_update_kernel<T, 0><<<grid, threads, 0, st>>>(lat->p.V, begin, count, (T)eps, p, u);
    else if (mode == 1) link_update_kernel<T, 1><<<grid, threads, 0, st>>>(lat->p.V, begin, count, (T)eps, p, u);
    else link_update_kernel<T, 2><<<grid, threads, 0, st>>>(lat->p.V, begin, count, (T)eps, p, u);
    return check_launch(mode == 2 ? "reunit" : "link_update");
}

int launch_link_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *P, void *U, int mode,
                       cudaStream_t st) {
    return prec == QCD_F64 ? launch_link_update_t<double>(lat, subset, eps, P, U, mode, st)
                           : launch_link_update_t<float>(lat, subset, eps, P, U, mode, st);
}

template <typename T>
static int launch_link_update_push_t(const qcd_lattice *lat, double eps, const void *P, void *U, int reunit,
                                     const qcd_lattice *lo, void *lo_U, const qcd_lattice *hi, void *hi_U,
                                     cudaStream_t st) {
    const int threads = 128;
    const dim3 grid((lat->p.V + threads - 1) / threads, 4);
    const LatP &pl = lo ? lo->p : lat->p, &ph = hi ? hi->p : lat->p;
    if (reunit)
        link_update_push_kernel<T, 1><<<grid, threads, 0, st>>>(lat->p, (T)eps, (const pair_t<T> *)P, (pair_t<T> *)U, pl,
                                                                (pair_t<T> *)lo_U, ph, (pair_t<T> *)hi_U);
    else
        link_update_push_kernel<T, 0><<<grid, threads, 0, st>>>(lat->p, (T)eps, (const pair_t<T> *)P, (pair_t<T> *)U, pl,
                                                                (pair_t<T> *)lo_U, ph, (pair_t<T> *)hi_U);
    return check_launch("link_update_push");
}

int launch_link_update_push(const qcd_lattice *lat, int prec, double eps, const void *P, void *U, int reunit,
                            const qcd_lattice *lo, void *lo_U, const qcd_lattice *hi, void *hi_U, cudaStream_t st) {
    return prec == QCD_F64 ? launch_link_update_push_t<double>(lat, eps, P, U, reunit, lo, lo_U, hi, hi_U, st)
                           : launch_link_update_push_t<float>(lat, eps, P, U, reunit, lo, lo_U, hi, hi_U, st);
}

template <typename T>
static int launch_mom_update_t(const qcd_lattice *lat, int subset, double eps, const void *F, void *P,
                               cudaStream_t st) {
    int begin, count;
    subset_range(lat->p, subset, begin, count);
    const int threads = tuned_threads(lat, sizeof(T) == 8 ? QCD_F64 : QCD_F32, subset, QCD_KERNEL_MOM_UPDATE, 256);
    const dim3 grid((count + threads - 1) / threads, 4);
    mom_update_kernel<T><<<grid, threads, 0, st>>>(lat->p.V, begin, count, (T)eps, (const pair_t<T> *)F,
                                                   (pair_t<T> *)P);
    return check_launch("mom_update");
}

int launch_mom_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *F, void *P,
                      cudaStream_t st) {
    return prec == QCD_F64 ? launch_mom_update_t<double>(lat, subset, eps, F, P, st)
                           : launch_mom_update_t<float>(lat, subset, eps, F, P, st);
}

}  // namespace qcd
