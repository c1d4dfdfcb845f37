// tmem.cuh — Tensor Memory (sm_100a: 512 columns x 128 lanes x 32 bit per SM) used as per-thread scratch.
//
// The stencil kernels are register-bound (an fp64 3x3 complex matrix is 36 registers) and every kilobyte of
// shared memory they take is a kilobyte less L1 for the neighbour links.  Tensor Memory is otherwise idle in
// these kernels (no tensor-core work: 3x3 complex algebra is not a dense contraction), is private per lane,
// and is read / written with tcgen05.ld / tcgen05.st without touching the L1 / shared-memory pipe.  With the
// 32x32b shape warp w of a block owns lanes 32 (w % 4) .. +31, and thread i of the warp the columns of lane i:
// a block of 4 warps that allocates C columns gives every thread C 32-bit words.
#pragma once

#include <stdint.h>

namespace qcd {

// one warp of the block (all 32 lanes): allocate NCOLS columns (power of two >= 32), base address -> *slot (shared)
template <int NCOLS>
__device__ __forceinline__ void tmem_alloc(uint32_t *slot) {
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(slot);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(s), "n"(NCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t base) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(base), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }

// N consecutive columns of this thread's lane
__device__ __forceinline__ void tmem_ld1(uint32_t a, uint32_t *w) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];\n" : "=r"(w[0]) : "r"(a));
}
__device__ __forceinline__ void tmem_ld2(uint32_t a, uint32_t *w) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];\n" : "=r"(w[0]), "=r"(w[1]) : "r"(a));
}
__device__ __forceinline__ void tmem_ld8(uint32_t a, uint32_t *w) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
                 : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7])
                 : "r"(a));
}
__device__ __forceinline__ void tmem_ld16(uint32_t a, uint32_t *w) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]), "=r"(w[8]),
          "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15])
        : "r"(a));
}
__device__ __forceinline__ void tmem_st1(uint32_t a, const uint32_t *w) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};\n" ::"r"(a), "r"(w[0]) : "memory");
}
__device__ __forceinline__ void tmem_st2(uint32_t a, const uint32_t *w) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};\n" ::"r"(a), "r"(w[0]), "r"(w[1]) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t a, const uint32_t *w) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};\n" ::"r"(a), "r"(w[0]),
                 "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t a, const uint32_t *w) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};\n" ::"r"(a),
        "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]), "r"(w[8]), "r"(w[9]),
        "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15])
        : "memory");
}

// nine reals (the TA part of one direction, force.cu) at column `col` of this thread's lane
__device__ __forceinline__ void tmem_load9(uint32_t a, double *v) {
    uint32_t w[18];
    tmem_ld16(a, w);
    tmem_ld2(a + 16, w + 16);
    tmem_wait_ld();
#pragma unroll
    for (int k = 0; k < 9; k++) v[k] = __hiloint2double((int)w[2 * k + 1], (int)w[2 * k]);
}
__device__ __forceinline__ void tmem_store9(uint32_t a, const double *v) {
    uint32_t w[18];
#pragma unroll
    for (int k = 0; k < 9; k++) {
        w[2 * k] = (uint32_t)__double2loint(v[k]);
        w[2 * k + 1] = (uint32_t)__double2hiint(v[k]);
    }
    tmem_st16(a, w);
    tmem_st2(a + 16, w + 16);
}
__device__ __forceinline__ void tmem_load9(uint32_t a, float *v) {
    uint32_t w[9];
    tmem_ld8(a, w);
    tmem_ld1(a + 8, w + 8);
    tmem_wait_ld();
#pragma unroll
    for (int k = 0; k < 9; k++) v[k] = __uint_as_float(w[k]);
}
__device__ __forceinline__ void tmem_store9(uint32_t a, const float *v) {
    uint32_t w[9];
#pragma unroll
    for (int k = 0; k < 9; k++) w[k] = __float_as_uint(v[k]);
    tmem_st8(a, w);
    tmem_st1(a + 8, w + 8);
}

}  // namespace qcd
