// random.cu — Gaussian momentum refresh (O4), hot start (O5), perturbation noise and raw generator
// blocks, all from the counter-based generator of rng.cuh ("a random number generator").
// One thread per link; the counter is keyed on the LEXICOGRAPHIC site, so the output does not depend
// on layout, subset, block shape or any later domain decomposition.
#include "qcd_internal.h"
#include "rng.cuh"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

// KIND 0: P = sum p_a T_a (purpose 1).  KIND 1: U = exp(i sigma Q) (purpose 0).
template <typename T, int KIND>
__global__ void __launch_bounds__(128) gauss_field_kernel(const LatP lat, const int begin, const int count,
                                                          const uint64_t seed, const uint32_t stream_id,
                                                          const double sigma, pair_t<T> *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const int cb = begin + i;
    const int mu = blockIdx.y;
    const Site st = site_of_cb(lat, cb);
    double q[8];
    gauss8(seed, global_site(lat, st.s), mu, stream_id, KIND == 0 ? 1u : 0u, q);
    if (KIND == 0) {
        M3<T> P;
        herm_from_coeffs(P, q);
        store_link(P, out, lat.V, mu, cb);
    } else {
#pragma unroll
        for (int a = 0; a < 8; a++) q[a] *= sigma;
        // exponentiate in double, round once for fp32 fields
        M3<double> Q, E;
        herm_from_coeffs(Q, q);
        expi_herm(E, Q);
        M3<T> R;
#pragma unroll
        for (int e = 0; e < 9; e++) {
            R.re[e] = (T)E.re[e];
            R.im[e] = (T)E.im[e];
        }
        store_link(R, out, lat.V, mu, cb);
    }
}

// U += sigma N, entry e = 3*row+col gets (g0, g1) of block j = e (purpose 2)
template <typename T>
__global__ void __launch_bounds__(128) perturb_kernel(const LatP lat, const uint64_t seed, const double sigma,
                                                      pair_t<T> *__restrict__ U) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= lat.V) return;
    const int mu = blockIdx.y;
    const Site st = site_of_cb(lat, cb);
    pair_t<T> *p = U + unit_index(36, mu * 9, cb);
#pragma unroll 1
    for (int e = 0; e < 9; e++) {
        uint32_t w[4];
        double u[2], g[2];
        rng_block(seed, global_site(lat, st.s), (uint32_t)(mu * 16 + e), 0u, 2u, w, u, g);
        pair_t<T> v = p[e * CHUNK];
        v.x = (T)((double)v.x + sigma * g[0]);
        v.y = (T)((double)v.y + sigma * g[1]);
        p[e * CHUNK] = v;
    }
}

// O15: spin-colour Gaussian fill, component k = blockIdx.y: eta_k(x) = (g0 + i g1)/sqrt(2) of generator block
// (site, 64 + k, stream_id, purpose 4); pair layout with 12 units per site: component k of site cb at unit_index(12, k, cb)
template <typename T>
__global__ void __launch_bounds__(128) spinor_gauss_kernel(const LatP lat, const int begin, const int count,
                                                           const uint64_t seed, const uint32_t stream_id,
                                                           pair_t<T> *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const int cb = begin + i;
    const int k = blockIdx.y;
    const Site st = site_of_cb(lat, cb);
    uint32_t w[4];
    double u[2], g[2];
    rng_block(seed, global_site(lat, st.s), (uint32_t)(64 + k), stream_id, 4u, w, u, g);
    const double isq2 = 0.70710678118654752440;
    pair_t<T> v;
    v.x = (T)(g[0] * isq2);
    v.y = (T)(g[1] * isq2);
    out[unit_index(12, k, cb)] = v;
}

int launch_spinor_gaussian(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *eta,
                           cudaStream_t st) {
    int begin, count;
    subset_range(lat->p, subset, begin, count);
    const int threads = 128;
    const dim3 grid((count + threads - 1) / threads, 12);
    if (prec == QCD_F64) spinor_gauss_kernel<double><<<grid, threads, 0, st>>>(lat->p, begin, count, seed, stream_id, (double2 *)eta);
    else spinor_gauss_kernel<float><<<grid, threads, 0, st>>>(lat->p, begin, count, seed, stream_id, (float2 *)eta);
    return check_launch("spinor_gaussian");
}

__global__ void rng_blocks_kernel(const uint64_t seed, const uint32_t stream_id, const uint32_t purpose, const int n,
                                  const uint32_t *__restrict__ site, const uint32_t *__restrict__ mu_j,
                                  uint32_t *__restrict__ words, double *__restrict__ uniforms,
                                  double *__restrict__ gauss) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t w[4];
    double u[2], g[2];
    rng_block(seed, site[i], mu_j[i], stream_id, purpose, w, u, g);
    if (words)
        for (int k = 0; k < 4; k++) words[4 * i + k] = w[k];
    if (uniforms) {
        uniforms[2 * i] = u[0];
        uniforms[2 * i + 1] = u[1];
    }
    if (gauss) {
        gauss[2 * i] = g[0];
        gauss[2 * i + 1] = g[1];
    }
}

int launch_mom_refresh(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *P,
                       cudaStream_t st) {
    int begin, count;
    subset_range(lat->p, subset, begin, count);
    const int threads = 128;
    const dim3 grid((count + threads - 1) / threads, 4);
    if (prec == QCD_F64)
        gauss_field_kernel<double, 0><<<grid, threads, 0, st>>>(lat->p, begin, count, seed, stream_id, 1.0, (double2 *)P);
    else
        gauss_field_kernel<float, 0><<<grid, threads, 0, st>>>(lat->p, begin, count, seed, stream_id, 1.0, (float2 *)P);
    return check_launch("mom_refresh");
}

int launch_hot_start(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, cudaStream_t st) {
    const int threads = 128;
    const dim3 grid((lat->p.V + threads - 1) / threads, 4);
    if (prec == QCD_F64)
        gauss_field_kernel<double, 1><<<grid, threads, 0, st>>>(lat->p, 0, lat->p.V, seed, 0u, sigma, (double2 *)U);
    else
        gauss_field_kernel<float, 1><<<grid, threads, 0, st>>>(lat->p, 0, lat->p.V, seed, 0u, sigma, (float2 *)U);
    return check_launch("hot_start");
}

int launch_perturb(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, cudaStream_t st) {
    const int threads = 128;
    const dim3 grid((lat->p.V + threads - 1) / threads, 4);
    if (prec == QCD_F64) perturb_kernel<double><<<grid, threads, 0, st>>>(lat->p, seed, sigma, (double2 *)U);
    else perturb_kernel<float><<<grid, threads, 0, st>>>(lat->p, seed, sigma, (float2 *)U);
    return check_launch("perturb");
}

int launch_rng_blocks(uint64_t seed, uint32_t stream_id, uint32_t purpose, int n, const uint32_t *site,
                      const uint32_t *mu_j, uint32_t *words, double *uniforms, double *gauss, cudaStream_t st) {
    if (n == 0) return QCD_OK;
    rng_blocks_kernel<<<(n + 127) / 128, 128, 0, st>>>(seed, stream_id, purpose, n, site, mu_j, words, uniforms, gauss);
    return check_launch("rng_blocks");
}

}  // namespace qcd
