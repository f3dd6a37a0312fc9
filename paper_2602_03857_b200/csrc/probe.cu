// probe.cu -- FP64 issue microbenchmark behind grav_fp64_mix_probe (include/grav.h): how much of the FP64 pipe a
// warp scheduler of this GPU sustains when K independent DFMA chains per warp are interleaved with NI integer
// (LOP3) instructions per group of K DFMAs, at W warps per scheduler.  It is the measurement the instruction mix
// of csrc/psi2.cuh was designed from (profiles/r1_fp64_issue_microbench.md) and holds none of the
// method's arithmetic.
#include <cuda_runtime.h>

#include "../../include/grav.h"

namespace {

template <int K, int NI>
__global__ void mix_probe_kernel(double* out, int iters, double a, double b, int seed) {
    double x[K];
    // thread-dependent values, so that the fillers are vector LOP3s like the integer work of the kernels (with uniform
    // values ptxas moves them to the uniform datapath as ULOP3)
    const int tid = (int)threadIdx.x;
    int iv[4] = {seed + tid, seed * 3 + tid, seed * 5 - tid, seed * 7 ^ tid};
#pragma unroll
    for (int j = 0; j < K; ++j) x[j] = a * (j + 1) + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int j = 0; j < K; ++j) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[j]) : "d"(a), "d"(b));
#pragma unroll
            for (int n = 0; n < NI; ++n)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xe8;" : "+r"(iv[n & 3]) : "r"(tid), "r"(iv[(n + 1) & 3]));
        }
    }
    double s = 0;
#pragma unroll
    for (int j = 0; j < K; ++j) s += x[j];
    s += iv[0] + iv[1] + iv[2] + iv[3];
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

template <int K, int NI>
cudaError_t run(int sms, int warps_per_smsp, int iters, float* ms) {
    int tpb = warps_per_smsp * 4 * 32, grid = sms;
    while (tpb > 1024) { tpb /= 2; grid *= 2; }
    double* out = nullptr;
    cudaError_t e = cudaMalloc(&out, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    mix_probe_kernel<K, NI><<<grid, tpb>>>(out, iters / 10 + 1, 1.0000001, 1e-9, 3);
    cudaEventRecord(e0);
    mix_probe_kernel<K, NI><<<grid, tpb>>>(out, iters, 1.0000001, 1e-9, 3);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return e;
}

}  // namespace

extern "C" grav_status grav_fp64_mix_probe(int device, int chains, int others, int warps_per_smsp, int iters,
                                           double* dfma_warp_inst_per_smsp, double* ms_out) {
    if (!dfma_warp_inst_per_smsp || !ms_out || iters <= 0 || warps_per_smsp < 1 || warps_per_smsp > 16)
        return GRAV_EINVAL;
    int prev = 0;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return GRAV_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return GRAV_ECUDA;
    const int sms = prop.multiProcessorCount;
    float ms = 0.f;
    cudaError_t e = cudaErrorInvalidValue;
#define GRAV_PROBE_CASE(K, NI) \
    if (chains == K && others == NI) e = run<K, NI>(sms, warps_per_smsp, iters, &ms);
    GRAV_PROBE_CASE(1, 0) GRAV_PROBE_CASE(2, 0) GRAV_PROBE_CASE(4, 0) GRAV_PROBE_CASE(8, 0)
    GRAV_PROBE_CASE(2, 1) GRAV_PROBE_CASE(2, 2) GRAV_PROBE_CASE(4, 1) GRAV_PROBE_CASE(4, 2) GRAV_PROBE_CASE(4, 4)
    GRAV_PROBE_CASE(8, 2) GRAV_PROBE_CASE(8, 4) GRAV_PROBE_CASE(8, 8)
#undef GRAV_PROBE_CASE
    cudaSetDevice(prev);
    if (e == cudaErrorInvalidValue) return GRAV_EINVAL;
    if (e != cudaSuccess) return GRAV_ECUDA;
    *dfma_warp_inst_per_smsp = (double)iters * 16.0 * chains * warps_per_smsp;
    *ms_out = ms;
    return GRAV_OK;
}
