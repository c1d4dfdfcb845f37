// probe.cu — the denominators the roofline fractions are quoted against ("Measure DFMA/FFMA peaks
// with a probe"; MEASURED_PEAKS.json has only the HBM copy and the bf16 GEMM).  Each probe is one kernel launch
// that bench.py times with CUDA events like any other call (the library never synchronises):
//   FMA   chains of 3x3 complex products held in registers, no memory: the plain-ALU FMA rate the staple
//         arithmetic can reach (the same mul<> the force kernel uses)
//   L1    every block re-reads its own 64 kB with 128-bit loads: L1-resident load bandwidth
//   LDS   the same from shared memory
//   L2    all blocks stream one 48 MB buffer: L2-resident bandwidth as the SMs see it
#include "qcd_internal.h"
#include "su3.cuh"

namespace qcd {

constexpr int PROBE_THREADS = 512;
constexpr int PROBE_BLOCKS_PER_SM = 2;
constexpr size_t PROBE_L1_BYTES = 64 * 1024;         // per block (two blocks per SM: 128 kB, L1-resident)
constexpr size_t PROBE_LDS_BYTES = 64 * 1024;        // per block
constexpr size_t PROBE_L2_BYTES = 48ull << 20;       // whole buffer

template <typename T>
__global__ void __launch_bounds__(256) probe_fma_kernel(const int reps, const T seed, T *out) {
    M3<T> A, B, C;
#pragma unroll
    for (int e = 0; e < 9; e++) {
        A.re[e] = seed + e * T(0.01) + threadIdx.x * T(1e-4);
        A.im[e] = seed - e * T(0.02);
        B.re[e] = seed * e * T(0.1);
        B.im[e] = T(0.3) - seed;
    }
    for (int r = 0; r < reps; r++) {
        mul<false, true, false>(C, A, B);
        mul<false, false, false>(A, C, B);
    }
    T s = 0;
#pragma unroll
    for (int e = 0; e < 9; e++) s += A.re[e] + A.im[e];
    if (s == T(1.2345)) out[0] = s;  // never true: keeps the chain alive
}

// eight independent 128-bit loads in flight per thread and iteration (a single dependent load per iteration
// measures latency, not the data path: 84 instead of 117 B/clk/SM)
__global__ void probe_l1_kernel(const double2 *__restrict__ p, const size_t n_per_block, const int reps, double2 *out) {
    const double2 *q = p + (size_t)blockIdx.x * n_per_block;
    double2 acc = {0, 0};
    const size_t bd = blockDim.x;
    for (int r = 0; r < reps; r++)
        for (size_t i = threadIdx.x; i + 7 * bd < n_per_block; i += 8 * bd) {
            double2 v[8];
#pragma unroll
            for (int u = 0; u < 8; u++) v[u] = __ldg(q + i + u * bd);
#pragma unroll
            for (int u = 0; u < 8; u++) {
                acc.x += v[u].x;
                acc.y += v[u].y;
            }
        }
    if (acc.x == 1.2345) out[0] = acc;
}

__global__ void probe_l2_kernel(const double2 *__restrict__ p, const size_t n, const int reps, double2 *out) {
    double2 acc = {0, 0};
    const size_t start = ((size_t)blockIdx.x * 7919 * 1024) % n;
    const size_t bd = blockDim.x;
    for (int r = 0; r < reps; r++)
        for (size_t i = threadIdx.x; i + 3 * bd < n / 8; i += 4 * bd) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
                size_t j = start + i + u * bd;
                if (j >= n) j -= n;
                v[u] = __ldg(p + j);
            }
#pragma unroll
            for (int u = 0; u < 4; u++) {
                acc.x += v[u].x;
                acc.y += v[u].y;
            }
        }
    if (acc.x == 1.2345) out[0] = acc;
}

__global__ void probe_lds_kernel(const int reps, double2 *out) {
    extern __shared__ double2 s[];
    constexpr int N = (int)(PROBE_LDS_BYTES / 16);
    for (int i = threadIdx.x; i < N; i += blockDim.x) s[i] = make_double2(i, 1);
    __syncthreads();
    double2 acc = {0, 0};
    for (int r = 0; r < reps; r++)
#pragma unroll 8
        for (int i = threadIdx.x; i < N; i += blockDim.x) {
            const double2 v = s[i];
            acc.x += v.x;
            acc.y += v.y;
        }
    if (acc.x == 1.2345) out[0] = acc;
}

static int sm_count() {
    int dev = 0, n = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    return n;
}

double probe_work(int what, int prec, int reps) {
    const double nb = (double)sm_count() * PROBE_BLOCKS_PER_SM;
    switch (what) {
        case QCD_PROBE_FMA: return nb * 2 * 256.0 * reps * 2 * 108;  // 4 blocks of 256 per SM, two products per rep
        case QCD_PROBE_L1: return nb * (double)PROBE_L1_BYTES * reps;
        case QCD_PROBE_LDS: return nb * (double)PROBE_LDS_BYTES * reps;
        case QCD_PROBE_L2: return nb * (double)(PROBE_L2_BYTES / 8) * reps;
    }
    (void)prec;
    return 0.0;
}

size_t probe_scratch_bytes(int what) {
    const size_t nb = (size_t)sm_count() * PROBE_BLOCKS_PER_SM;
    if (what == QCD_PROBE_L1) return nb * PROBE_L1_BYTES + 64;
    if (what == QCD_PROBE_L2) return PROBE_L2_BYTES + 64;
    return 64;
}

int launch_probe(int what, int prec, int reps, void *scratch, cudaStream_t st) {
    const int nb = sm_count() * PROBE_BLOCKS_PER_SM;
    double2 *buf = (double2 *)scratch;
    switch (what) {
        case QCD_PROBE_FMA:
            if (prec == QCD_F64) probe_fma_kernel<double><<<2 * nb, 256, 0, st>>>(reps, 0.5, (double *)scratch);
            else probe_fma_kernel<float><<<2 * nb, 256, 0, st>>>(reps, 0.5f, (float *)scratch);
            break;
        case QCD_PROBE_L1:
            probe_l1_kernel<<<nb, PROBE_THREADS, 0, st>>>(buf + 4, PROBE_L1_BYTES / 16, reps, buf);
            break;
        case QCD_PROBE_LDS:
            cudaFuncSetAttribute(probe_lds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PROBE_LDS_BYTES);
            probe_lds_kernel<<<nb, PROBE_THREADS, PROBE_LDS_BYTES, st>>>(reps, buf);
            break;
        case QCD_PROBE_L2:
            probe_l2_kernel<<<nb, PROBE_THREADS, 0, st>>>(buf + 4, PROBE_L2_BYTES / 16, reps, buf);
            break;
    }
    return check_launch("probe");
}

}  // namespace qcd
