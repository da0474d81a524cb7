// probe.cu -- throughput micro-benchmarks behind the roofline denominators (include/ants_recon.h,
// ants_probe_throughput).  The reconstruction is bound by the plain FP32 pipes, for which
// MEASURED_PEAKS.json has no entry: the derived peak (SMs x 128 lanes x 2 x clock) is cross-checked here by
// dependent-free instruction streams of the kinds the kernels issue (FFMA, packed FFMA2, MUFU, DFMA).
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ants_recon.h"
#include "recon_common.cuh"

namespace ants {

constexpr int kChains = 8;       // independent accumulators per thread (latency 4 cycles is covered many times over)
constexpr int kUnroll = 16;      // instructions per chain per loop trip

// kind 0: FFMA with one register operand reused (acc = acc * x + y, x and y loop-invariant)
// kind 4: FFMA with three distinct, changing register operands (acc_j = acc_j * acc_{j+1} + acc_{j+2})
template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(float x, float y, int iters, float *sink) {
    float acc[kChains];
    f32x2 acc2[kChains];
    double accd[kChains];
#pragma unroll
    for (int j = 0; j < kChains; ++j) {
        acc[j] = x + (float)(threadIdx.x + j);
        acc2[j] = pk(acc[j], acc[j] + 1.f);
        accd[j] = (double)acc[j];
    }
    const f32x2 x2 = pk1(x), y2 = pk1(y);
    const double xd = (double)x, yd = (double)y;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
#pragma unroll
            for (int j = 0; j < kChains; ++j) {
                if (KIND == 0) acc[j] = fmaf(acc[j], x, y);
                else if (KIND == 1) acc2[j] = fma2(acc2[j], x2, y2);
                else if (KIND == 2) acc[j] = lg2_approx(acc[j]);
                else if (KIND == 3) accd[j] = fma(accd[j], xd, yd);
                else acc[j] = fmaf(acc[j], acc[(j + 1) % kChains], acc[(j + 2) % kChains]);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s += acc[j] + hsum2(acc2[j]) + (float)accd[j];
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace ants

extern "C" int ants_probe_throughput(int32_t kind, int32_t iters, double *lane_ops_per_second_out,
                                     double *milliseconds_out) {
    using namespace ants;
    if (kind < 0 || kind > 4 || iters < 1 || !lane_ops_per_second_out) return ANTS_ERR_INVALID;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    const void *k = kind == 0 ? (const void *)probe_kernel<0> : kind == 1 ? (const void *)probe_kernel<1>
                  : kind == 2 ? (const void *)probe_kernel<2> : kind == 3 ? (const void *)probe_kernel<3>
                                                                           : (const void *)probe_kernel<4>;
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, 256, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    const int grid = sms * occ;
    float *sink = nullptr;
    if (cudaMalloc(&sink, (size_t)grid * 256 * sizeof(float)) != cudaSuccess) { cudaGetLastError(); return ANTS_ERR_NOMEM; }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float x = 0.999f, y = 0.001f;
    int it = iters;
    void *args[] = {&x, &y, &it, &sink};
    bool ok = cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess;
    int warm = iters / 8 + 1;
    void *wargs[] = {&x, &y, &warm, &sink};
    ok = ok && cudaLaunchKernel(k, dim3(grid), dim3(256), wargs, 0, nullptr) == cudaSuccess;
    ok = ok && cudaEventRecord(e0, nullptr) == cudaSuccess;
    ok = ok && cudaLaunchKernel(k, dim3(grid), dim3(256), args, 0, nullptr) == cudaSuccess;
    ok = ok && cudaEventRecord(e1, nullptr) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess;
    float ms = 0.f;
    ok = ok && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    if (!ok || !(ms > 0.f)) { cudaGetLastError(); return ANTS_ERR_CUDA; }
    // one lane-op = one scalar result: FFMA2 produces two per thread-instruction
    const double per_thread = (double)iters * kUnroll * kChains * (kind == 1 ? 2.0 : 1.0);
    *lane_ops_per_second_out = per_thread * 256.0 * grid / (ms * 1e-3);
    if (milliseconds_out) *milliseconds_out = ms;
    return ANTS_OK;
}
