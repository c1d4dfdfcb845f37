// rng.cuh — counter-based generator (O3): Philox4x32-10, key = seed, counter =
// (lexicographic site, mu*16+j, stream_id, purpose); two exact 52-bit uniforms and one
// Box-Muller pair per block.  Gaussians are always produced in double.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace qcd {

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t w[4]) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// u = (2k+1) 2^-53 with k the 52 bits (wa>>6, wb>>6): exact, strictly inside (0,1)
__device__ __forceinline__ double uniform52(uint32_t wa, uint32_t wb) {
    const unsigned long long k = ((unsigned long long)(wa >> 6) << 26) | (unsigned long long)(wb >> 6);
    return (double)(2ull * k + 1ull) * 0x1p-53;
}

__device__ __forceinline__ void rng_block(uint64_t seed, uint32_t s, uint32_t mu_j, uint32_t stream_id,
                                          uint32_t purpose, uint32_t w[4], double u[2], double g[2]) {
    philox4x32_10(s, mu_j, stream_id, purpose, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), w);
    u[0] = uniform52(w[0], w[1]);
    u[1] = uniform52(w[2], w[3]);
    const double r = sqrt(-2.0 * log(u[0]));
    double sn, cs;
    sincos(2.0 * 3.14159265358979323846264338327950288 * u[1], &sn, &cs);
    g[0] = r * cs;
    g[1] = r * sn;
}

// the eight N(0,1) coefficients of link (s,mu): q[2j], q[2j+1] from block j
__device__ __forceinline__ void gauss8(uint64_t seed, uint32_t s, int mu, uint32_t stream_id, uint32_t purpose,
                                       double q[8]) {
#pragma unroll
    for (int j = 0; j < 4; j++) {
        uint32_t w[4];
        double u[2];
        rng_block(seed, s, (uint32_t)(mu * 16 + j), stream_id, purpose, w, u, q + 2 * j);
    }
}

}  // namespace qcd
