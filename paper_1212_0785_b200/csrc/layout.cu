// layout.cu — helpers off the hot path: canonical lexicographic AoS <-> device layout, index maps (O1).
#include "qcd_internal.h"
#include "site.cuh"
#include "su3.cuh"

namespace qcd {

// Device index of real c of site cb (su3.cuh: chunks of 32 sites).  Pair fields (ncomp a multiple of 18 or 24):
// unit = complex pair, ncomp/2 units per site, real index 2*unit_index(ncomp/2, c>>1, cb) + (c&1).
// Real fields: unit = real, ncomp units per site, index unit_index(ncomp, c, cb).
template <typename T, bool UNPACK>
__global__ void __launch_bounds__(256) pack_kernel(const LatP lat, const int ncomp, const bool matrix,
                                                   const T *__restrict__ src, T *__restrict__ dst) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= lat.V) return;
    const Site st = site_of_cb(lat, cb);
    const size_t aos = (size_t)st.s * ncomp;
    for (int c = blockIdx.y; c < ncomp; c += gridDim.y) {
        const size_t soa = matrix ? 2 * (size_t)unit_index(ncomp / 2, c >> 1, cb) + (c & 1) : (size_t)unit_index(ncomp, c, cb);
        if (UNPACK) dst[aos + c] = src[soa];
        else dst[soa] = src[aos + c];
    }
}

// Same maps through a shared-memory transpose, so that both sides are coalesced: a block takes PK_SITES
// consecutive lexicographic sites (one contiguous chunk of the canonical array, both parities) and the
// matching PK_SITES/2 consecutive checkerboard indices of each parity (pair h = s>>1 holds one even and one
// odd site because Lx is even).  Site stride in shared memory is ncomp+2 reals (bank spread).
constexpr int PK_SITES = 64;

// site0, site_end: the lexicographic range handled (whole lattice, or whole timeslices of it); the canonical array
// starts at site0.
template <typename T, bool UNPACK>
__global__ void __launch_bounds__(256) pack_tr_kernel(const LatP lat, const int ncomp, const bool matrix,
                                                      const T *__restrict__ src, T *__restrict__ dst,
                                                      const int site0, const int site_end) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *sm = reinterpret_cast<T *>(smem_raw);
    const int ss = ncomp + 2;
    const int s0 = site0 + blockIdx.x * PK_SITES;
    const int ns = min(PK_SITES, site_end - s0);  // the range and s0 are even: ns is even
    const int nh = ns >> 1;
    const int h0 = s0 >> 1;
    const int nel = ns * ncomp;
    const T *aos_in = UNPACK ? nullptr : src + (size_t)(s0 - site0) * ncomp;
    T *aos_out = UNPACK ? dst + (size_t)(s0 - site0) * ncomp : nullptr;
    if (!UNPACK)
        for (int i = threadIdx.x; i < nel; i += blockDim.x) sm[(i / ncomp) * ss + i % ncomp] = aos_in[i];
    else {
        // checkerboard side -> shared
        for (int i = threadIdx.x; i < nel; i += blockDim.x) {
            // i = ((c2 * 2 + par) * nh + hl) * w + ri, w = 2 reals (matrix) or 1
            const int w = matrix ? 2 : 1;
            const int ri = i % w;
            int r = i / w;
            const int hl = r % nh;
            r /= nh;
            const int par = r & 1;
            const int c = (r >> 1) * w + ri;
            const int h = h0 + hl;
            const int row = (2 * h) / lat.L[0];
            const int y = row % lat.L[1], zt = row / lat.L[1];
            const int odd = (y + zt % lat.L[2] + zt / lat.L[2] + par) & 1;
            const int cb = par * lat.Vh + h;
            const size_t soa = matrix ? 2 * (size_t)unit_index(ncomp / 2, c >> 1, cb) + (c & 1) : (size_t)unit_index(ncomp, c, cb);
            sm[(2 * hl + odd) * ss + c] = src[soa];
        }
    }
    __syncthreads();
    if (UNPACK)
        for (int i = threadIdx.x; i < nel; i += blockDim.x) aos_out[i] = sm[(i / ncomp) * ss + i % ncomp];
    else
        for (int i = threadIdx.x; i < nel; i += blockDim.x) {
            const int w = matrix ? 2 : 1;
            const int ri = i % w;
            int r = i / w;
            const int hl = r % nh;
            r /= nh;
            const int par = r & 1;
            const int c = (r >> 1) * w + ri;
            const int h = h0 + hl;
            const int row = (2 * h) / lat.L[0];
            const int y = row % lat.L[1], zt = row / lat.L[1];
            const int odd = (y + zt % lat.L[2] + zt / lat.L[2] + par) & 1;
            const int cb = par * lat.Vh + h;
            const size_t soa = matrix ? 2 * (size_t)unit_index(ncomp / 2, c >> 1, cb) + (c & 1) : (size_t)unit_index(ncomp, c, cb);
            dst[soa] = sm[(2 * hl + odd) * ss + c];
        }
}

__global__ void map_kernel(const LatP lat, const int which, int32_t *__restrict__ out) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= lat.V) return;
    const Site st = site_of_lex(lat, s);
    const int cb = cb_of(lat, s, st.par);
    if (which == QCD_MAP_CB_OF_LEX) out[s] = cb;
    else if (which == QCD_MAP_LEX_OF_CB) out[cb] = site_of_cb(lat, cb).s;  // decode path of the kernels
    else if (which >= QCD_MAP_NBR_FWD0 && which <= QCD_MAP_NBR_FWD3) out[s] = s + dfwd(lat, st, which - QCD_MAP_NBR_FWD0);
    else if (which >= QCD_MAP_NBR_BWD0 && which <= QCD_MAP_NBR_BWD3) out[s] = s + dbwd(lat, st, which - QCD_MAP_NBR_BWD0);
    else if (which == QCD_MAP_PARITY) out[s] = st.par;
    else out[s] = st.c[3];
}

// the transposing kernel on the lexicographic range [site0, site_end) (both even)
static int launch_pack_range(const qcd_lattice *lat, int prec, int ncomp, bool matrix, const void *src, void *dst,
                             bool unpack, int site0, int site_end, cudaStream_t st) {
    const size_t rb = prec == QCD_F64 ? 8 : 4;
    const size_t shm = (size_t)PK_SITES * (ncomp + 2) * rb;
    const int blocks = (site_end - site0 + PK_SITES - 1) / PK_SITES;
    if (prec == QCD_F64) {
        if (unpack) pack_tr_kernel<double, true><<<blocks, 256, shm, st>>>(lat->p, ncomp, matrix, (const double *)src, (double *)dst, site0, site_end);
        else pack_tr_kernel<double, false><<<blocks, 256, shm, st>>>(lat->p, ncomp, matrix, (const double *)src, (double *)dst, site0, site_end);
    } else {
        if (unpack) pack_tr_kernel<float, true><<<blocks, 256, shm, st>>>(lat->p, ncomp, matrix, (const float *)src, (float *)dst, site0, site_end);
        else pack_tr_kernel<float, false><<<blocks, 256, shm, st>>>(lat->p, ncomp, matrix, (const float *)src, (float *)dst, site0, site_end);
    }
    return check_launch(unpack ? "unpack" : "pack");
}

int launch_pack_slab(const qcd_lattice *lat, int prec, int ncomp, bool pairs, const void *src, void *dst, bool unpack,
                     int t_begin, int nt, cudaStream_t st) {
    const int Vs = lat->p.V / lat->p.L[3];
    return launch_pack_range(lat, prec, ncomp, pairs, src, dst, unpack, t_begin * Vs, (t_begin + nt) * Vs, st);
}

// One thread per site of the `nt` source timeslices: copies the units of the links selected by mu_mask (matrix
// fields) or all nc units from the source field to the same spatial site of the destination timeslices.  The two
// lattices share the spatial extents; each side is addressed with its own checkerboard index (the parity of a site
// depends on its local t).  With a peer pointer as dst this kernel is the NVLink transport of the halo exchange.
template <typename T>
__global__ void __launch_bounds__(256) copy_timeslices_kernel(const LatP src_lat, const pair_t<T> *__restrict__ src,
                                                              const int src_t, const LatP dst_lat,
                                                              pair_t<T> *__restrict__ dst, const int dst_t, const int nt,
                                                              const int nc, const unsigned mu_mask) {
    const int Vsh = src_lat.Vh / src_lat.L[3];  // sites per parity and timeslice
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * nt * Vsh) return;
    const int par = i / (nt * Vsh);
    const int cb = par * src_lat.Vh + src_t * Vsh + (i - par * nt * Vsh);  // consecutive threads: consecutive sites
    const Site st = site_of_cb(src_lat, cb);
    const int dt = dst_t + (st.c[3] - src_t);
    const int ds = st.s + (dt - st.c[3]) * dst_lat.stride[3];
    const int dcb = cb_of(dst_lat, ds, (st.c[0] + st.c[1] + st.c[2] + dt) & 1);
    for (int k = 0; k < nc; k++) {
        if (nc == 36 && !((mu_mask >> (k / 9)) & 1u)) continue;
        dst[unit_index(nc, k, dcb)] = __ldg(src + unit_index(nc, k, cb));
    }
}

int launch_copy_timeslices(const qcd_lattice *src_lat, const void *src, int src_t, const qcd_lattice *dst_lat, void *dst,
                           int dst_t, int nt, int prec, int nc, unsigned mu_mask, cudaStream_t st) {
    const int n = nt * (src_lat->p.V / src_lat->p.L[3]);
    const int blocks = (n + 255) / 256;
    if (prec == QCD_F64)
        copy_timeslices_kernel<double><<<blocks, 256, 0, st>>>(src_lat->p, (const double2 *)src, src_t, dst_lat->p,
                                                               (double2 *)dst, dst_t, nt, nc, mu_mask);
    else
        copy_timeslices_kernel<float><<<blocks, 256, 0, st>>>(src_lat->p, (const float2 *)src, src_t, dst_lat->p,
                                                              (float2 *)dst, dst_t, nt, nc, mu_mask);
    return check_launch("copy_timeslices");
}

int launch_pack(const qcd_lattice *lat, int prec, int ncomp, bool pairs, const void *src, void *dst, bool unpack,
                cudaStream_t st) {
    const bool matrix = pairs;  // complex-pair layout (colour matrices, spin-colour vectors) or real layout
    const size_t rb = prec == QCD_F64 ? 8 : 4;
    const size_t shm = (size_t)PK_SITES * (ncomp + 2) * rb;
    if (shm <= 48 * 1024)  // transpose through shared memory; larger ncomp falls back to the direct kernel
        return launch_pack_range(lat, prec, ncomp, matrix, src, dst, unpack, 0, lat->p.V, st);
    const dim3 grid((lat->p.V + 255) / 256, ncomp < 72 ? ncomp : 72);
    if (prec == QCD_F64) {
        if (unpack) pack_kernel<double, true><<<grid, 256, 0, st>>>(lat->p, ncomp, matrix, (const double *)src, (double *)dst);
        else pack_kernel<double, false><<<grid, 256, 0, st>>>(lat->p, ncomp, matrix, (const double *)src, (double *)dst);
    } else {
        if (unpack) pack_kernel<float, true><<<grid, 256, 0, st>>>(lat->p, ncomp, matrix, (const float *)src, (float *)dst);
        else pack_kernel<float, false><<<grid, 256, 0, st>>>(lat->p, ncomp, matrix, (const float *)src, (float *)dst);
    }
    return check_launch(unpack ? "unpack" : "pack");
}

int launch_get_map(const qcd_lattice *lat, int which, int32_t *out, cudaStream_t st) {
    map_kernel<<<(lat->p.V + 255) / 256, 256, 0, st>>>(lat->p, which, out);
    return check_launch("get_map");
}

}  // namespace qcd
