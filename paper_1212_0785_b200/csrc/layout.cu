// layout.cu — helpers off the hot path: canonical lexicographic AoS <-> device layout, index maps (O1).
#include "qcd_internal.h"
#include "site.cuh"

namespace qcd {

// MATRIX layout (ncomp % 18 == 0): real r = 2k+ri of site cb at real index 2*(k*V + cb) + ri.
// REAL layout: component c of site cb at c*V + cb.
template <typename T, bool UNPACK>
__global__ void __launch_bounds__(256) pack_kernel(const LatP lat, const int ncomp, const bool matrix,
                                                   const T *__restrict__ src, T *__restrict__ dst) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= lat.V) return;
    const Site st = site_of_cb(lat, cb);
    const size_t aos = (size_t)st.s * ncomp;
    for (int c = blockIdx.y; c < ncomp; c += gridDim.y) {
        const size_t soa = matrix ? 2 * ((size_t)(c >> 1) * lat.V + cb) + (c & 1) : (size_t)c * lat.V + cb;
        if (UNPACK) dst[aos + c] = src[soa];
        else dst[soa] = src[aos + c];
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

int launch_pack(const qcd_lattice *lat, int prec, int ncomp, const void *src, void *dst, bool unpack,
                cudaStream_t st) {
    const bool matrix = ncomp % 18 == 0;
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
