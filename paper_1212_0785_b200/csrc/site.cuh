// site.cuh — index arithmetic (O1): lexicographic <-> checkerboard, neighbours.
#pragma once

#include "qcd_internal.h"

namespace qcd {

struct Site {
    int c[4];  // coordinates x,y,z,t
    int s;     // lexicographic index
    int par;   // (x+y+z+t)&1
};

__device__ __forceinline__ int cb_of(const LatP &lat, int s, int par) { return par * lat.Vh + (s >> 1); }

// checkerboard index -> site.  s>>1 = h fixes (x&~1, y, z, t); the parity bit fixes x&1.
__device__ __forceinline__ Site site_of_cb(const LatP &lat, int cb) {
    Site st;
    st.par = cb >= lat.Vh ? 1 : 0;
    const int s2 = 2 * (cb - st.par * lat.Vh);
    int r = s2 / lat.L[0];
    const int x2 = s2 - r * lat.L[0];
    st.c[1] = r % lat.L[1];
    r /= lat.L[1];
    st.c[2] = r % lat.L[2];
    st.c[3] = r / lat.L[2];
    const int odd = (st.c[1] + st.c[2] + st.c[3] + st.par) & 1;
    st.c[0] = x2 + odd;
    st.s = s2 + odd;
    return st;
}

__device__ __forceinline__ Site site_of_lex(const LatP &lat, int s) {
    Site st;
    st.s = s;
    int r = s / lat.L[0];
    st.c[0] = s - r * lat.L[0];
    st.c[1] = r % lat.L[1];
    r /= lat.L[1];
    st.c[2] = r % lat.L[2];
    st.c[3] = r / lat.L[2];
    st.par = (st.c[0] + st.c[1] + st.c[2] + st.c[3]) & 1;
    return st;
}

// the generator's site counter: the GLOBAL lexicographic index (slab lattices carry an offset)
__device__ __forceinline__ uint32_t global_site(const LatP &lat, int s) {
    return (uint32_t)(((unsigned long long)s + (unsigned long long)lat.site_off) % (unsigned long long)lat.gV);
}

// lexicographic index change for one periodic hop in +mu / -mu
__device__ __forceinline__ int dfwd(const LatP &lat, const Site &st, int mu) {
    return st.c[mu] == lat.L[mu] - 1 ? -(lat.L[mu] - 1) * lat.stride[mu] : lat.stride[mu];
}
__device__ __forceinline__ int dbwd(const LatP &lat, const Site &st, int mu) {
    return st.c[mu] == 0 ? (lat.L[mu] - 1) * lat.stride[mu] : -lat.stride[mu];
}

// cb range [begin, begin+count) of a subset
__host__ __device__ inline void subset_range(const LatP &lat, int subset, int &begin, int &count) {
    begin = subset == QCD_ODD ? lat.Vh : 0;
    count = subset == QCD_ALL ? lat.V : lat.Vh;
}

}  // namespace qcd
