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
