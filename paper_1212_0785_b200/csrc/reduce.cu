// reduce.cu — plaquette (O6) and the global / per-subset sums (O12; "sum, sumMulti").
//
// Deterministic two-pass reductions: the lattice is cut into (timeslice, parity) segments, each a
// contiguous range of checkerboard indices, and every segment into fixed chunks of RED_CHUNK sites.
// Pass 1: one block per chunk, fixed per-thread order, fixed shuffle/shared tree -> one partial.
// Pass 2: one block per result sums the partials in a fixed order.  The geometry depends only on
// the lattice, never on tuning, so results are bit-identical from run to run.
#include <mutex>

#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

// fixed-order block sum; result valid in thread 0
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double warp_part[RED_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) warp_part[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) {
        for (int k = 0; k < (int)blockDim.x / 32; k++) r += warp_part[k];
    }
    __syncthreads();
    return r;
}

// ---- per-site values -----------------------------------------------------------------------

// sum_{mu<nu} Re tr P_mu_nu(x), P_mu_nu(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger
// which: 0 = all six planes, 1 = the three space-space planes, 2 = the three space-time planes (R19)
template <typename T>
__device__ __forceinline__ double site_plaquette(const LatP &lat, const pair_t<T> *__restrict__ U, int cb,
                                                 int which = 0) {
    const Site st = site_of_cb(lat, cb);
    const int V = lat.V;
    int cbf[4];
#pragma unroll
    for (int d = 0; d < 4; d++) cbf[d] = cb_of(lat, st.s + dfwd(lat, st, d), st.par ^ 1);
    T acc = T(0);
    // fp32: four blocks per SM at 128 registers pay (-10 %), so U_mu(x) is loaded again for every plane (an L1 hit)
    // instead of being held; fp64: three blocks at 168 registers with U_mu(x) held are faster (0.48 against 0.52 ms)
    constexpr bool RELOAD = sizeof(T) == 4;
#pragma unroll
    for (int mu = 0; mu < 3; mu++) {
        M3<T> Um;
        if (!RELOAD) load_link(Um, U, V, mu, cb);
#pragma unroll
        for (int nu = mu + 1; nu < 4; nu++) {
            if ((which == 1 && nu == 3) || (which == 2 && nu != 3)) continue;
            if (RELOAD) load_link(Um, U, V, mu, cb);
            // Re tr{[U_mu(x) U_nu(x+mu)] U_mu(x+nu)^dag U_nu(x)^dag}, left to right: three matrices besides U_mu(x) are
            // live at a time (the two-bracket form needs four and spilled at 168 registers)
            M3<T> A, X, Z;
            load_link(A, U, V, nu, cbf[mu]);
            mul<false, false, false>(X, Um, A);
            load_link(A, U, V, mu, cbf[nu]);
            mul<false, true, false>(Z, X, A);
            load_link(A, U, V, nu, cb);
            acc += retr_mul_dag(Z, A);
        }
    }
    return (double)acc;
}

// QCD_SUM_INNER (kind 3, internal): comp 0 / 1 = Re / Im of sum_k conj(a_k) b_k over the ncomp/2 complex
// components of two pair-layout fields (O16)
constexpr int SUM_INNER = 3;

template <typename T>
__device__ __forceinline__ double site_value(int kind, int ncomp, int comp, int V, const T *__restrict__ f, int cb,
                                             const T *__restrict__ f2 = nullptr) {
    if (kind == QCD_SUM_SCALAR) return (double)__ldg(f + unit_index(ncomp, comp, cb));
    const unsigned b0 = unit_index(ncomp / 2, 0, cb);  // pair fields: ncomp/2 complex units per site
    double acc = 0.0;
    if (kind == SUM_INNER) {
        const pair_t<T> *a = (const pair_t<T> *)f, *b = (const pair_t<T> *)f2;
        for (int k = 0; k < ncomp / 2; k++) {
            const pair_t<T> x = __ldg(a + b0 + k * CHUNK), y = __ldg(b + b0 + k * CHUNK);
            if (comp == 0) acc = fma((double)x.x, (double)y.x, fma((double)x.y, (double)y.y, acc));
            else  // both products rounded before the difference (no FMA contraction): Im <a,a> is exactly 0
                acc += __dsub_rn(__dmul_rn((double)x.x, (double)y.y), __dmul_rn((double)x.y, (double)y.x));
        }
        return acc;
    }
    if (kind == QCD_SUM_NORM2) {
        const pair_t<T> *p = (const pair_t<T> *)f;
        for (int k = 0; k < ncomp / 2; k++) {
            const pair_t<T> v = __ldg(p + b0 + k * CHUNK);
            acc = fma((double)v.x, (double)v.x, acc);
            acc = fma((double)v.y, (double)v.y, acc);
        }
    } else {
        const pair_t<T> *p = (const pair_t<T> *)f;
        for (int m = 0; m < ncomp / 18; m++) {
            acc += (double)__ldg(p + b0 + (m * 9 + 0) * CHUNK).x;
            acc += (double)__ldg(p + b0 + (m * 9 + 4) * CHUNK).x;
            acc += (double)__ldg(p + b0 + (m * 9 + 8) * CHUNK).x;
        }
    }
    return acc;
}

// ---- pass 1 --------------------------------------------------------------------------------

// grid (chunks_per_seg, nseg, ncomp_out).
// partial[(comp*nseg + seg)*cps + chunk], seg = 2*t + parity
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) reduce_pass1(const LatP lat, const int kind, const int ncomp,
                                                            const void *__restrict__ field, double *__restrict__ partial,
                                                            const void *__restrict__ field2 = nullptr,
                                                            const int par_only = -1) {
    // par_only = 0 / 1: a parity subset — only that parity's segments are visited (grid.y = Lt), the partial
    // array keeps its full (2 Lt segment) indexing so the second pass is the same
    const int cps = gridDim.x, nseg = par_only < 0 ? gridDim.y : 2 * gridDim.y;
    const int seg = par_only < 0 ? blockIdx.y : 2 * blockIdx.y + par_only, comp = blockIdx.z;
    const int Vsh = lat.Vh / lat.L[3];
    const int seg_begin = (seg & 1) * lat.Vh + (seg >> 1) * Vsh;
    double acc = 0.0;
#pragma unroll 1
    for (int k = 0; k < RED_CHUNK / RED_THREADS; k++) {
        const int i = blockIdx.x * RED_CHUNK + k * RED_THREADS + threadIdx.x;
        if (i < Vsh) {
            const int cb = seg_begin + i;
            acc += site_value<T>(kind, ncomp, comp, lat.V, (const T *)field, cb, (const T *)field2);
        }
    }
    const double r = block_sum(acc);
    if (threadIdx.x == 0) partial[((size_t)comp * nseg + seg) * cps + blockIdx.x] = r;
}

// plaquette pass 1, same chunk geometry and partial layout as reduce_pass1 (grid (cps, nseg, ncomp_out)) but in
// PLAQ_THREADS-thread blocks, several resident per SM: the stencil kernel wants warps, not wide blocks
// (profiles/r02_per_kernel.md).  which0: 0 = all planes; 1 = comp 0 space-space, comp 1 space-time.
constexpr int PLAQ_THREADS = 128;
template <typename T>
__global__ void __launch_bounds__(PLAQ_THREADS, sizeof(T) == 8 ? 3 : 4) plaquette_pass1(const LatP lat, const int which0,
                                                                   const pair_t<T> *__restrict__ U,
                                                                   double *__restrict__ partial) {
    const int cps = gridDim.x, nseg = gridDim.y;
    const int seg = blockIdx.y, comp = blockIdx.z;
    const int Vsh = lat.Vh / lat.L[3];
    const int seg_begin = (seg & 1) * lat.Vh + (seg >> 1) * Vsh;
    double acc = 0.0;
#pragma unroll 1
    for (int k = 0; k < RED_CHUNK / PLAQ_THREADS; k++) {
        const int i = blockIdx.x * RED_CHUNK + k * PLAQ_THREADS + threadIdx.x;
        if (i < Vsh) acc += site_plaquette<T>(lat, U, seg_begin + i, which0 ? 1 + comp : 0);
    }
    const double r = block_sum(acc);
    if (threadIdx.x == 0) partial[((size_t)comp * nseg + seg) * cps + blockIdx.x] = r;
}

// subset_id path: grid (RED_GENERIC_CHUNKS, nsub, ncomp_out); partial[(comp*nsub + k)*RED_GENERIC_CHUNKS + chunk]
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) reduce_pass1_ids(const LatP lat, const int kind, const int ncomp,
                                                                const void *__restrict__ field,
                                                                const int32_t *__restrict__ ids,
                                                                double *__restrict__ partial) {
    const int k = blockIdx.y, comp = blockIdx.z, nsub = gridDim.y;
    const int csize = (lat.V + RED_GENERIC_CHUNKS - 1) / RED_GENERIC_CHUNKS;
    const int begin = blockIdx.x * csize;
    const int end = min(begin + csize, lat.V);
    double acc = 0.0;
    for (int cb = begin + threadIdx.x; cb < end; cb += RED_THREADS)
        if (__ldg(ids + cb) == k) acc += site_value<T>(kind, ncomp, comp, lat.V, (const T *)field, cb);
    const double r = block_sum(acc);
    if (threadIdx.x == 0) partial[((size_t)comp * nsub + k) * RED_GENERIC_CHUNKS + blockIdx.x] = r;
}

// ---- pass 2 --------------------------------------------------------------------------------

// out[blockIdx.x * out_stride + comp] = scale * sum of `count` partials starting at
// partial[(comp*ngroups + blockIdx.x) * count], taking every `step`-th group member if step > 1 ...
// Written generally: group g = blockIdx.x covers partial indices base(g) + i*stride_i, i < count.
__global__ void __launch_bounds__(RED_THREADS) reduce_pass2(const double *__restrict__ partial, const int ngroups,
                                                            const int count, const double scale,
                                                            double *__restrict__ out, const int out_stride) {
    const int g = blockIdx.x, comp = blockIdx.y;
    const double *p = partial + ((size_t)comp * ngroups + g) * count;
    double acc = 0.0;
    for (int i = threadIdx.x; i < count; i += RED_THREADS) acc += p[i];
    const double r = block_sum(acc);
    if (threadIdx.x == 0) out[(size_t)g * out_stride + comp] = scale * r;
}

// global sum over the segments of one parity set: segments seg with (seg&1)==par if par<2, all if par==2
__global__ void __launch_bounds__(RED_THREADS) reduce_pass2_global(const double *__restrict__ partial, const int nseg,
                                                                   const int cps, const int par, const double scale,
                                                                   double *__restrict__ out) {
    const int comp = blockIdx.x;
    const double *p = partial + (size_t)comp * nseg * cps;
    double acc = 0.0;
    if (par == 2) {
        for (int i = threadIdx.x; i < nseg * cps; i += RED_THREADS) acc += p[i];
    } else {
        const int n = (nseg / 2) * cps;
        for (int i = threadIdx.x; i < n; i += RED_THREADS) {
            const int t = i / cps, c = i - t * cps;
            acc += p[(size_t)(2 * t + par) * cps + c];
        }
    }
    const double r = block_sum(acc);
    if (threadIdx.x == 0) out[comp] = scale * r;
}

// ---- launchers -----------------------------------------------------------------------------

template <typename T>
static int plaquette_t(const qcd_lattice *lat, const void *U, double *out_avg, double *out_per_t, double *ws,
                       cudaStream_t st) {
    const LatP &p = lat->p;
    const int cps = lat->red_chunks_per_seg, nseg = lat->red_nseg;
    plaquette_pass1<T><<<dim3(cps, nseg, 1), PLAQ_THREADS, 0, st>>>(p, 0, (const pair_t<T> *)U, ws);
    const int Lt = p.L[3];
    const double Vs = (double)(p.V / Lt);
    if (out_per_t)  // segments 2t, 2t+1 are adjacent: one group of 2*cps partials per timeslice
        reduce_pass2<<<dim3(Lt, 1), RED_THREADS, 0, st>>>(ws, Lt, 2 * cps, 1.0 / (18.0 * Vs), out_per_t, 1);
    reduce_pass2_global<<<1, RED_THREADS, 0, st>>>(ws, nseg, cps, 2, 1.0 / (18.0 * (double)p.V), out_avg);
    return check_launch("plaquette");
}

int launch_plaquette(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t, double *ws,
                     cudaStream_t st) {
    return prec == QCD_F64 ? plaquette_t<double>(lat, U, out_avg, out_per_t, ws, st)
                           : plaquette_t<float>(lat, U, out_avg, out_per_t, ws, st);
}

// ---- qcd_plaquette_noalloc: the same two passes with the partial sums in memory the library brings along ----
//
// Some callers of this library cannot hand it a workspace because they have no way to get device memory: code
// that runs inside an application whose own memory manager has claimed the whole device (the setting of
// PAPER.md:71,83, where every package's allocations are redirected to one pool that such a caller holds no
// handle to), and measurement code inside a running trajectory, where a cudaMalloc / cudaFree pair would
// stall every stream of the device.  For them the first-pass partials live in this file-scope array.  It is
// part of the library image: every GPU on which the library is loaded carries its 256 KiB until the process
// exits, whether or not the call is ever made.
//
// g_noalloc_partials names the array in DEVICE code.  In host code the same identifier is only a handle for the
// runtime's symbol calls — it is not a device address, and a kernel handed `g_noalloc_partials` from the host
// would write somewhere else entirely — so the launcher below asks the runtime for the array's address on the
// current device, once per device, and passes that pointer to the kernels.
static __device__ __align__(256) double g_noalloc_partials[NOALLOC_MAX_PARTIALS];

constexpr int NOALLOC_MAX_DEVICES = 64;
static double *g_noalloc_addr[NOALLOC_MAX_DEVICES];  // device address of g_noalloc_partials on device i; NULL = not asked yet
static std::mutex g_noalloc_mutex;

// the array's address on the CURRENT device (set-up on the first call per device: one cudaGetSymbolAddress)
static int noalloc_partials(double **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        set_error("qcd_plaquette_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
        return QCD_ECUDA;
    }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) {
        set_error("qcd_plaquette_noalloc: device ordinal %d outside the %d this call keeps an address for", dev,
                  NOALLOC_MAX_DEVICES);
        return QCD_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_partials);
        if (e != cudaSuccess || !p) {
            set_error("qcd_plaquette_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return QCD_ECUDA;
        }
        g_noalloc_addr[dev] = (double *)p;
    }
    *out = g_noalloc_addr[dev];
    return QCD_OK;
}

// Nothing in the array has to start at zero: pass 1 stores one partial per block into every slot pass 2 reads
// (slots [0, nseg*cps)), so what an earlier call left behind is overwritten before it is looked at.
int launch_plaquette_noalloc(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                             cudaStream_t st) {
    double *ws = nullptr;
    const int rc = noalloc_partials(&ws);
    if (rc != QCD_OK) return rc;
    return launch_plaquette(lat, prec, U, out_avg, out_per_t, ws, st);
}

// out[g] = scale * sum of the `count` per-block partials partial[g*count .. (g+1)*count), g < ngroups, fixed
// order (second pass of kernels that reduce as a by-product, e.g. the force kernel with SUMS)
int launch_sum_partials(const double *partial, int ngroups, int count, double scale, double *out, cudaStream_t st) {
    reduce_pass2<<<dim3(ngroups, 1), RED_THREADS, 0, st>>>(partial, ngroups, count, scale, out, 1);
    return check_launch("sum_partials");
}

template <typename T>
static int plaquette_st_t(const qcd_lattice *lat, const void *U, double *out_avg, double *out_per_t, double *ws,
                          cudaStream_t st) {
    const LatP &p = lat->p;
    const int cps = lat->red_chunks_per_seg, nseg = lat->red_nseg;
    plaquette_pass1<T><<<dim3(cps, nseg, 2), PLAQ_THREADS, 0, st>>>(p, 1, (const pair_t<T> *)U, ws);
    const int Lt = p.L[3];
    const double Vs = (double)(p.V / Lt);
    if (out_per_t)  // out_per_t[t*2 + comp]
        reduce_pass2<<<dim3(Lt, 2), RED_THREADS, 0, st>>>(ws, Lt, 2 * cps, 1.0 / (9.0 * Vs), out_per_t, 2);
    reduce_pass2_global<<<2, RED_THREADS, 0, st>>>(ws, nseg, cps, 2, 1.0 / (9.0 * (double)p.V), out_avg);
    return check_launch("plaquette_st");
}

int launch_plaquette_st(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                        double *ws, cudaStream_t st) {
    return prec == QCD_F64 ? plaquette_st_t<double>(lat, U, out_avg, out_per_t, ws, st)
                           : plaquette_st_t<float>(lat, U, out_avg, out_per_t, ws, st);
}

template <typename T>
static int sum_t(const qcd_lattice *lat, int subset, int kind, int ncomp, const void *field, double *out, double *ws,
                 cudaStream_t st) {
    const int cps = lat->red_chunks_per_seg, nseg = lat->red_nseg;
    const int nout = kind == QCD_SUM_SCALAR ? ncomp : 1;
    const int par = subset == QCD_ALL ? 2 : subset == QCD_EVEN ? 0 : 1;
    if (par == 2) reduce_pass1<T><<<dim3(cps, nseg, nout), RED_THREADS, 0, st>>>(lat->p, kind, ncomp, field, ws);
    else reduce_pass1<T><<<dim3(cps, nseg / 2, nout), RED_THREADS, 0, st>>>(lat->p, kind, ncomp, field, ws, nullptr, par);
    reduce_pass2_global<<<nout, RED_THREADS, 0, st>>>(ws, nseg, cps, par, 1.0, out);
    return check_launch("sum");
}

int launch_sum(const qcd_lattice *lat, int prec, int subset, int kind, int ncomp, const void *field, double *out,
               double *ws, cudaStream_t st) {
    return prec == QCD_F64 ? sum_t<double>(lat, subset, kind, ncomp, field, out, ws, st)
                           : sum_t<float>(lat, subset, kind, ncomp, field, out, ws, st);
}

// O16: out[0], out[1] = Re, Im of <a, b> over the subset; per_t = true: out[t*2 + {0,1}] per timeslice
template <typename T>
static int inner_t(const qcd_lattice *lat, int subset, int nc, const void *a, const void *b, bool per_t, double *out,
                   double *ws, cudaStream_t st) {
    const int cps = lat->red_chunks_per_seg, nseg = lat->red_nseg;
    const int par = subset == QCD_ALL ? 2 : subset == QCD_EVEN ? 0 : 1;
    if (par == 2 || per_t) reduce_pass1<T><<<dim3(cps, nseg, 2), RED_THREADS, 0, st>>>(lat->p, SUM_INNER, 2 * nc, a, ws, b);
    else reduce_pass1<T><<<dim3(cps, nseg / 2, 2), RED_THREADS, 0, st>>>(lat->p, SUM_INNER, 2 * nc, a, ws, b, par);
    if (per_t) {
        const int Lt = lat->p.L[3];
        reduce_pass2<<<dim3(Lt, 2), RED_THREADS, 0, st>>>(ws, Lt, 2 * cps, 1.0, out, 2);
    } else {
        reduce_pass2_global<<<2, RED_THREADS, 0, st>>>(ws, nseg, cps, par, 1.0, out);
    }
    return check_launch("inner_product");
}

int launch_inner_product(const qcd_lattice *lat, int prec, int subset, int nc, const void *a, const void *b,
                         bool per_t, double *out, double *ws, cudaStream_t st) {
    return prec == QCD_F64 ? inner_t<double>(lat, subset, nc, a, b, per_t, out, ws, st)
                           : inner_t<float>(lat, subset, nc, a, b, per_t, out, ws, st);
}

template <typename T>
static int sum_multi_t(const qcd_lattice *lat, int kind, int ncomp, const void *field, const int32_t *ids, int nsub,
                       double *out, double *ws, cudaStream_t st) {
    const int nout = kind == QCD_SUM_SCALAR ? ncomp : 1;
    if (!ids) {
        const int cps = lat->red_chunks_per_seg, nseg = lat->red_nseg;
        reduce_pass1<T><<<dim3(cps, nseg, nout), RED_THREADS, 0, st>>>(lat->p, kind, ncomp, field, ws);
        reduce_pass2<<<dim3(nsub, nout), RED_THREADS, 0, st>>>(ws, nsub, 2 * cps, 1.0, out, nout);
    } else {
        reduce_pass1_ids<T><<<dim3(RED_GENERIC_CHUNKS, nsub, nout), RED_THREADS, 0, st>>>(lat->p, kind, ncomp, field,
                                                                                          ids, ws);
        reduce_pass2<<<dim3(nsub, nout), RED_THREADS, 0, st>>>(ws, nsub, RED_GENERIC_CHUNKS, 1.0, out, nout);
    }
    return check_launch("sum_multi");
}

int launch_sum_multi(const qcd_lattice *lat, int prec, int kind, int ncomp, const void *field,
                     const int32_t *subset_id, int nsub, double *out, double *ws, cudaStream_t st) {
    return prec == QCD_F64 ? sum_multi_t<double>(lat, kind, ncomp, field, subset_id, nsub, out, ws, st)
                           : sum_multi_t<float>(lat, kind, ncomp, field, subset_id, nsub, out, ws, st);
}

}  // namespace qcd
