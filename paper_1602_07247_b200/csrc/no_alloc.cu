// no_alloc.cu -- ants_lrf_fit_gains_static (include/ants_recon.h): the gain evaluation of ants_lrf_fit_gains
// (section 6.3, reading R24) for callers that must not allocate -- code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc.  The scratch the kernel needs (the FP64 sums, the pair
// counters, the device copies of the sensor positions and of the profile) lives in ONE file-scope device array of a
// fixed, modest size; every GPU that loads the library holds it until the process exits.  Nothing here calls
// cudaMalloc, cudaFree or an allocating library routine, and the host side uses no heap memory either.
//
// The array's name is, in host code, a host-side stand-in and NOT a device address: the address is asked once per
// device, with that device current, from cudaGetSymbolAddress, and handed to the kernel as a pointer.
#include <cmath>
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/ants_recon.h"

namespace {

constexpr int kMaxSensors = ANTS_STATIC_MAX_SENSORS;     // 128: a lane owns the sensors lane + 32 c, c < 4
constexpr int kMaxCoeffs = ANTS_STATIC_MAX_COEFFS;       // 1024 = n_int_r + 3 at most
constexpr int kMaxDevices = 64;

// layout of the scratch, in bytes from its start
constexpr size_t kOffAcc = 0;                                                  // double [kMaxSensors][2] {sum y s, sum s^2}
constexpr size_t kOffUsed = kOffAcc + sizeof(double) * 2 * kMaxSensors;        // unsigned long long [kMaxSensors]
constexpr size_t kOffXY = kOffUsed + sizeof(unsigned long long) * kMaxSensors; // float [kMaxSensors][2]
constexpr size_t kOffCoef = kOffXY + sizeof(float) * 2 * kMaxSensors;          // float [kMaxCoeffs]
constexpr size_t kScratchBytes = kOffCoef + sizeof(float) * kMaxCoeffs;        // 8192
constexpr size_t kZeroBytes = kOffXY;                                          // what must start at zero: sums, counters
static_assert(kScratchBytes == ANTS_STATIC_SCRATCH_BYTES, "header and layout disagree");

static __device__ __align__(256) unsigned char g_gain_scratch[kScratchBytes];

// Variant of lrf_gain_kernel (lrf_fit.cuh) with every device buffer inside `scratch`.  One warp per event, lanes over
// sensors; a lane keeps the two sums of the sensors it owns in registers for all the events its warp sees and adds
// them to the FP64 accumulators once at the end.
__global__ void __launch_bounds__(256) lrf_gain_static_kernel(unsigned char *scratch, const float *signals,
                                                              const float *xyzA, long long n_events, int N, int n_int,
                                                              double lo, double hi, double h) {
    __shared__ double coef_s[kMaxCoeffs];              // the profile's coefficients in double
    double *acc = reinterpret_cast<double *>(scratch + kOffAcc);
    unsigned long long *n_used = reinterpret_cast<unsigned long long *>(scratch + kOffUsed);
    const float *sens_xy = reinterpret_cast<const float *>(scratch + kOffXY);
    const float *coeffs = reinterpret_cast<const float *>(scratch + kOffCoef);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    for (int j = threadIdx.x; j < n_int + 3; j += blockDim.x) coef_s[j] = (double)coeffs[j];
    __syncthreads();
    double num[4] = {0, 0, 0, 0}, den[4] = {0, 0, 0, 0};
    unsigned long long cnt[4] = {0, 0, 0, 0};
    double sx[4], sy[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = lane + 32 * c;
        sx[c] = i < N ? (double)sens_xy[2 * i] : 0.0;
        sy[c] = i < N ? (double)sens_xy[2 * i + 1] : 0.0;
    }
    for (long long e = (long long)blockIdx.x * warps + warp; e < n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;    // R22
        const float *sig = signals + e * N;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int i = lane + 32 * c;
            if (i >= N) continue;
            const double dx = x - sx[c], dy = y - sy[c];
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r >= lo && r <= hi)) continue;
            const double t = (r - lo) / h;
            const int k = min((int)floor(t), n_int - 1);
            const double u = t - (double)k, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
            const double s = coef_s[k] * (o * o * o / 6.0) + coef_s[k + 1] * ((3.0 * u3 - 6.0 * u2 + 4.0) / 6.0) +
                             coef_s[k + 2] * ((-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) / 6.0) + coef_s[k + 3] * (u3 / 6.0);
            const double yv = (double)__ldg(sig + i) / A;
            num[c] += yv * s;
            den[c] += s * s;
            ++cnt[c];
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = lane + 32 * c;
        if (i < N && cnt[c]) {
            atomicAdd(acc + 2 * i, num[c]);
            atomicAdd(acc + 2 * i + 1, den[c]);
            atomicAdd(n_used + i, cnt[c]);
        }
    }
}

// the scratch's device address on every device that has asked for it, and the lock that serialises the calls of
// this process (they all share the one array)
std::mutex g_mu;
unsigned char *g_scratch_ptr[kMaxDevices] = {};
int g_sms[kMaxDevices] = {};

}  // namespace

extern "C" int ants_lrf_fit_gains_static(const float *sensor_xy, const float *knots, const float *coeffs, int32_t N,
                                         int32_t n_int, const float *signals, const float *xyzA, int64_t n_events,
                                         float *gains_out, double *n_used_out, void *cuda_stream) {
    if (!sensor_xy || !knots || !coeffs || !gains_out || N < 1 || n_int < 1 || n_events < 0) return ANTS_ERR_INVALID;
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    // beyond the fixed scratch: refused, nothing is truncated
    if (N > kMaxSensors || n_int + 3 > kMaxCoeffs) return ANTS_ERR_UNSUPPORTED;
    const double lo = (double)knots[0], hi = (double)knots[1];
    if (!std::isfinite(lo) || !std::isfinite(hi) || !(lo >= 0.0) || !(hi > lo)) return ANTS_ERR_INVALID;
    for (int j = 0; j < n_int + 3; ++j)
        if (!std::isfinite(coeffs[j])) return ANTS_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return ANTS_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) return ANTS_ERR_UNSUPPORTED;

    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        // set-up, once per device, with that device current: the array's device address and the SM count
        unsigned char *ptr = nullptr;
        int sms = 0;
        if (cudaGetSymbolAddress((void **)&ptr, g_gain_scratch) != cudaSuccess || !ptr ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            cudaGetLastError();
            return ANTS_ERR_CUDA;
        }
        g_scratch_ptr[dev] = ptr;
        g_sms[dev] = sms;
    }
    unsigned char *scratch = g_scratch_ptr[dev];

    // the array keeps the previous call's contents: sums and counters are cleared, positions and profile overwritten
    bool ok = cudaMemsetAsync(scratch, 0, kZeroBytes, st) == cudaSuccess &&
              cudaMemcpyAsync(scratch + kOffXY, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(scratch + kOffCoef, coeffs, (size_t)(n_int + 3) * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess;
    if (ok && n_events > 0) {
        const int warps = 8;
        const long long want = (n_events + warps - 1) / warps;
        long long grid = (long long)g_sms[dev] * 4;          // 256 threads, 8 KB of static shared memory: 4+ CTAs per SM
        if (grid > want) grid = want;
        lrf_gain_static_kernel<<<(unsigned)grid, warps * 32, 0, st>>>(scratch, signals, xyzA, (long long)n_events, N, n_int,
                                                                     lo, hi, (hi - lo) / n_int);
        ok = cudaGetLastError() == cudaSuccess;
    }
    double acc[2 * kMaxSensors];
    unsigned long long used[kMaxSensors];
    ok = ok && cudaMemcpyAsync(acc, scratch + kOffAcc, (size_t)N * 2 * sizeof(double), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaMemcpyAsync(used, scratch + kOffUsed, (size_t)N * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaStreamSynchronize(st) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        cudaStreamSynchronize(st);      // nothing of this call is left in flight on the shared array
        return ANTS_ERR_CUDA;
    }
    for (int i = 0; i < N; ++i) {
        if (n_used_out) n_used_out[i] = (double)used[i];
        gains_out[i] = acc[2 * i + 1] > 0.0 ? (float)(acc[2 * i] / acc[2 * i + 1]) : std::nanf("");
    }
    return ANTS_OK;
}
