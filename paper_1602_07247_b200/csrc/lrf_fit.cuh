// lrf_fit.cuh -- LRF calculation for axial LRFs: least-squares B-spline fit from event positions and
// sensor signals (section 6 "The LRF module calculates these functions from datasets
// containing photosensor signals and the corresponding event positions"; PAPER.md:400-414 grouping,
// positions reconstructed or true).  Readings R21-R23: unweighted least squares of
// y = S / (A g) against the uniform cubic B-spline at r = |p - P_i|; events need finite x, y, A and
// A > 0; pairs need r_lo <= r <= r_hi.
//
// The kernel accumulates the normal equations M = sum B^T B (symmetric, half-bandwidth 3) and
// b = sum B^T y in FP64: one warp per event, lanes over sensors, every pair adds 10 band entries and
// 4 right-hand-side entries with shared-memory FP64 atomics into the CTA's copy (one copy per warp for a
// shared profile, where all sensors hit the same table), which is flushed once to the global
// accumulators.  All arithmetic is double: the path is bound by the atomics and by the signal stream,
// not by FP64 throughput.  The host solves the banded systems (ants_recon.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ants {

struct FitParams {
    const float *sens_xy;        // device [N][2]
    const float *gains;          // device [N] (all 1 when the caller passed none)
    const int *group;            // device [N] table index per sensor (R28), or nullptr: 0 (n_lrf = 1) / i (n_lrf = N)
    const float *signals;        // device [E][N]
    const float *xyzA;           // device [E][4]
    long long n_events;
    int N, n_lrf, n_int, nc;     // nc = n_int + 3 coefficients
    double lo, hi, h;            // h = (hi - lo) / n_int
    double *acc;                 // device [n_lrf][nc][5]: {M[j][j], M[j][j+1], M[j][j+2], M[j][j+3], b[j]}
    unsigned long long *n_used;  // device [n_lrf]
    int copies;                  // shared-memory copies of the accumulators per CTA (1, or warps * lane_split)
    int lane_split;              // copies per warp (contention on the FP64 atomics falls with it)
};

__global__ void __launch_bounds__(256) lrf_fit_kernel(const FitParams p) {
    extern __shared__ double fit_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int per_copy = p.n_lrf * p.nc * 5;
    for (int i = threadIdx.x; i < per_copy * p.copies; i += blockDim.x) fit_smem[i] = 0.0;
    if (p.n_lrf > 1)
        for (int i = threadIdx.x; i < p.n_lrf; i += blockDim.x)
            reinterpret_cast<unsigned long long *>(fit_smem + (size_t)per_copy * p.copies)[i] = 0ULL;
    __syncthreads();
    // shared profile: copies = warps * lane_split private copies, lanes of a warp spread over lane_split of them
    double *mine = fit_smem + (p.copies > 1 ? (size_t)(warp * p.lane_split + (lane % p.lane_split)) * per_copy : 0);
    // pairs used: a register count for a shared profile, shared-memory counters for per-sensor tables
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(fit_smem + (size_t)per_copy * p.copies);
    unsigned long long used = 0ULL;

    for (long long e = (long long)blockIdx.x * warps + warp; e < p.n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        // R22: finite x, y, A and A > 0 (NaN fails every comparison)
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;
        const float *sig = p.signals + e * p.N;
        for (int i = lane; i < p.N; i += 32) {
            const double dx = x - (double)p.sens_xy[2 * i], dy = y - (double)p.sens_xy[2 * i + 1];
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r >= p.lo && r <= p.hi)) continue;                                   // R22
            const int tabi = p.group ? p.group[i] : (p.n_lrf == 1 ? 0 : i);
            const double g = (p.group || p.n_lrf == 1) ? (double)p.gains[i] : 1.0;
            const double yv = (double)__ldg(sig + i) / (A * g);                         // R21, R23
            const double t = (r - p.lo) / p.h;
            const int k = min((int)floor(t), p.n_int - 1);
            const double u = t - (double)k, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
            const double b4[4] = {o * o * o / 6.0, (3.0 * u3 - 6.0 * u2 + 4.0) / 6.0,
                                  (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) / 6.0, u3 / 6.0};
            double *tab = mine + (size_t)tabi * p.nc * 5;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                double *row = tab + (size_t)(k + a) * 5;
                atomicAdd(row + 4, b4[a] * yv);
#pragma unroll
                for (int c = a; c < 4; ++c) atomicAdd(row + (c - a), b4[a] * b4[c]);
            }
            if (p.n_lrf == 1) ++used;
            else atomicAdd(cnt + tabi, 1ULL);
        }
    }
    if (p.n_lrf == 1) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
        if (lane == 0 && used) atomicAdd(p.n_used, used);
    }
    __syncthreads();
    if (p.n_lrf > 1)
        for (int i = threadIdx.x; i < p.n_lrf; i += blockDim.x)
            if (cnt[i]) atomicAdd(p.n_used + i, cnt[i]);
    for (int i = threadIdx.x; i < per_copy; i += blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < p.copies; ++c) s += fit_smem[c * per_copy + i];
        if (s != 0.0) atomicAdd(p.acc + i, s);
    }
}

// ---- relative gains for a fixed shared profile (R24): g_i = sum y s / sum s^2 --------
// One warp per event, lanes over sensors; every lane keeps the two sums of the sensors it owns
// (i = lane + 32 c, c < 4: N <= 128) in registers for all the events its warp sees -- no atomics in the
// loop -- and adds them to the global FP64 accumulators once at the end.
struct GainParams {
    const float *sens_xy;        // device [N][2]
    const float *coeffs;         // device [n_int + 3]
    const float *signals;        // device [E][N]
    const float *xyzA;           // device [E][4]
    long long n_events;
    int N, n_int;
    double lo, hi, h;
    double *acc;                 // device [N][2]: {sum y s, sum s^2}
    unsigned long long *n_used;  // device [N]
};

__global__ void __launch_bounds__(256) lrf_gain_kernel(const GainParams p) {
    extern __shared__ double gain_smem[];      // the profile's coefficients in double
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    for (int j = threadIdx.x; j < p.n_int + 3; j += blockDim.x) gain_smem[j] = (double)p.coeffs[j];
    __syncthreads();
    double num[4] = {0, 0, 0, 0}, den[4] = {0, 0, 0, 0};
    unsigned long long cnt[4] = {0, 0, 0, 0};
    double sx[4], sy[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = lane + 32 * c;
        sx[c] = i < p.N ? (double)p.sens_xy[2 * i] : 0.0;
        sy[c] = i < p.N ? (double)p.sens_xy[2 * i + 1] : 0.0;
    }
    for (long long e = (long long)blockIdx.x * warps + warp; e < p.n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;    // R22
        const float *sig = p.signals + e * p.N;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int i = lane + 32 * c;
            if (i >= p.N) continue;
            const double dx = x - sx[c], dy = y - sy[c];
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r >= p.lo && r <= p.hi)) continue;
            const double t = (r - p.lo) / p.h;
            const int k = min((int)floor(t), p.n_int - 1);
            const double u = t - (double)k, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
            const double s = gain_smem[k] * (o * o * o / 6.0) + gain_smem[k + 1] * ((3.0 * u3 - 6.0 * u2 + 4.0) / 6.0) +
                             gain_smem[k + 2] * ((-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) / 6.0) + gain_smem[k + 3] * (u3 / 6.0);
            const double yv = (double)__ldg(sig + i) / A;
            num[c] += yv * s;
            den[c] += s * s;
            ++cnt[c];
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = lane + 32 * c;
        if (i < p.N && cnt[c]) {
            atomicAdd(p.acc + 2 * i, num[c]);
            atomicAdd(p.acc + 2 * i + 1, den[c]);
            atomicAdd(p.n_used + i, cnt[c]);
        }
    }
}

// ---- axial+z tensor LRF (R25): normal equations of the shared (r, z) spline -----------
// nc = (n_z + 3)(n_r + 3) unknowns; a pair touches 4 x 4 of them.  The CTA keeps, per row j1, the 4 x 7
// block of entries M[j1][j1 + dz ncr + dr], dz = 0..3, dr = -3..3 (the upper triangle in linear order) and
// the right-hand side: 29 doubles per row in shared memory, 136 + 16 FP64 atomics per pair.
struct FitRZParams {
    const float *sens_xy, *gains, *signals, *xyzA;
    long long n_events;
    int N, n_r, n_z, ncr, nc;
    double r_lo, r_hi, hr, z_lo, z_hi, hz;
    double *acc;                 // device [nc][29]: [dz * 7 + dr + 3] for dz = 0..3, then the rhs at [28]
    unsigned long long *n_used;  // device [1]
};

__global__ void __launch_bounds__(256) lrf_fit_rz_kernel(const FitRZParams p) {
    extern __shared__ double rz_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int total = p.nc * 29;
    for (int i = threadIdx.x; i < total; i += blockDim.x) rz_smem[i] = 0.0;
    __syncthreads();
    unsigned long long used = 0ULL;
    for (long long e = (long long)blockIdx.x * warps + warp; e < p.n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, z = (double)pe.z, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308 && z >= p.z_lo && z <= p.z_hi)) continue;
        const double tz = (z - p.z_lo) / p.hz;
        const int kz = min((int)floor(tz), p.n_z - 1);
        const double uz = tz - (double)kz, oz = 1.0 - uz, uz2 = uz * uz, uz3 = uz2 * uz;
        const double bz[4] = {oz * oz * oz / 6.0, (3.0 * uz3 - 6.0 * uz2 + 4.0) / 6.0,
                              (-3.0 * uz3 + 3.0 * uz2 + 3.0 * uz + 1.0) / 6.0, uz3 / 6.0};
        const float *sig = p.signals + e * p.N;
        for (int i = lane; i < p.N; i += 32) {
            const double dx = x - (double)p.sens_xy[2 * i], dy = y - (double)p.sens_xy[2 * i + 1];
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r >= p.r_lo && r <= p.r_hi)) continue;
            const double yv = (double)__ldg(sig + i) / (A * (double)p.gains[i]);
            const double tr = (r - p.r_lo) / p.hr;
            const int kr = min((int)floor(tr), p.n_r - 1);
            const double u = tr - (double)kr, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
            const double br[4] = {o * o * o / 6.0, (3.0 * u3 - 6.0 * u2 + 4.0) / 6.0,
                                  (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) / 6.0, u3 / 6.0};
#pragma unroll
            for (int b1 = 0; b1 < 4; ++b1)
#pragma unroll
                for (int a1 = 0; a1 < 4; ++a1) {
                    const double w1 = bz[b1] * br[a1];
                    double *row = rz_smem + (size_t)((kz + b1) * p.ncr + kr + a1) * 29;
                    atomicAdd(row + 28, w1 * yv);
#pragma unroll
                    for (int b2 = b1; b2 < 4; ++b2)
#pragma unroll
                        for (int a2 = 0; a2 < 4; ++a2) {
                            if (b2 == b1 && a2 < a1) continue;
                            atomicAdd(row + (b2 - b1) * 7 + (a2 - a1) + 3, w1 * bz[b2] * br[a2]);
                        }
                }
            ++used;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
    if (lane == 0 && used) atomicAdd(p.n_used, used);
    __syncthreads();
    for (int i = threadIdx.x; i < total; i += blockDim.x)
        if (rz_smem[i] != 0.0) atomicAdd(p.acc + i, rz_smem[i]);
}

// ---- event filters (section 5.2; R26): rejected rows of xyzA become NaN, in place ------
struct FilterParams {
    float *xyzA;                 // device [E][4], in place
    const float *score;          // device [E]
    long long n_events;
    float score_max, energy_min, energy_max, radius_max;   // NaN = criterion off
    unsigned long long *n_pass;  // device [1]
};

__global__ void __launch_bounds__(256) event_filter_kernel(const FilterParams p) {
    unsigned long long pass = 0ULL;
    const double rm2 = (double)p.radius_max * (double)p.radius_max;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < p.n_events; e += (long long)gridDim.x * blockDim.x) {
        const float4 v = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const float s = p.score[e];
        bool keep = fabsf(v.x) <= 3.402823466e38f && fabsf(v.y) <= 3.402823466e38f && fabsf(v.w) <= 3.402823466e38f &&
                    fabsf(s) <= 3.402823466e38f;
        if (p.score_max == p.score_max) keep = keep && s <= p.score_max;
        if (p.energy_min == p.energy_min) keep = keep && v.w >= p.energy_min;
        if (p.energy_max == p.energy_max) keep = keep && v.w <= p.energy_max;
        if (p.radius_max == p.radius_max) keep = keep && (double)v.x * (double)v.x + (double)v.y * (double)v.y <= rm2;
        if (keep) ++pass;
        else {
            const float q = __int_as_float(0x7fc00000);
            reinterpret_cast<float4 *>(p.xyzA)[e] = make_float4(q, q, q, q);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pass += __shfl_xor_sync(0xffffffffu, pass, o);
    if ((threadIdx.x & 31) == 0 && pass) atomicAdd(p.n_pass, pass);
}

}  // namespace ants

namespace ants {

// ---- XY tables (R35) and the XY component of a Composite LRF: normal equations of
// ONE table's tensor-product spline in the sensor-local coordinates (u, v) = T_i (p - P_i), accumulated exactly as
// lrf_fit_rz_kernel does (per row the 4 x 7 block of the upper triangle + the right-hand side, 29 doubles).  Lanes
// run over the table's member sensors; a Composite fit subtracts the table's axial spline from y first.
struct FitXYParams {
    const float *sens_xy, *gains, *xform;     // device [N][2], [N] (1 for per-sensor tables), [N][4] or nullptr
    const int *members;                        // device [n_members] sensors of this table
    int n_members;
    const float *signals, *xyzA;
    long long n_events;
    int N, nx, ny, ncu, nc;
    double u_lo, u_hi, hu, v_lo, v_hi, hv;
    const float *axial;                        // device [a_n + 3] axial coefficients of this table, or nullptr
    int a_n;
    double a_lo, a_hi;
    double *acc;                               // device [nc][29]
    unsigned long long *n_used;                // device [1]
    // Sliced tables (R36): this launch takes the events between planes `slab` and `slab + 1` and adds
    // one of the three sums the joint normal equations are made of, the pair's basis products weighted by
    // (1-w)^2 (part 0: plane `slab` with itself; right-hand side weighted by 1-w), w^2 (part 1: plane `slab + 1`
    // with itself; right-hand side by w) or (1-w) w (part 2: the two planes with each other; no right-hand side).
    // slab < 0: a plain XY table.
    int slab, part, n_planes;
    double z_lo, z_hi, dz;
};

__global__ void __launch_bounds__(256) lrf_fit_xy_kernel(const FitXYParams p) {
    extern __shared__ double xy_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int total = p.nc * 29;
    for (int i = threadIdx.x; i < total; i += blockDim.x) xy_smem[i] = 0.0;
    __syncthreads();
    unsigned long long used = 0ULL;
    for (long long e = (long long)blockIdx.x * warps + warp; e < p.n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;       // R22
        double wm = 1.0, wy = 1.0;
        if (p.slab >= 0) {
            const double z = (double)pe.z;
            if (!(z >= p.z_lo && z <= p.z_hi)) continue;                                            // R36
            const int pl = max(min((int)floor((z - p.z_lo) / p.dz), p.n_planes - 2), 0);
            if (pl != p.slab) continue;
            const double w = (z - (p.z_lo + (double)pl * p.dz)) / p.dz;
            wm = p.part == 0 ? (1.0 - w) * (1.0 - w) : p.part == 1 ? w * w : (1.0 - w) * w;
            wy = p.part == 0 ? 1.0 - w : p.part == 1 ? w : 0.0;
        }
        const float *sig = p.signals + e * p.N;
        for (int q = lane; q < p.n_members; q += 32) {
            const int i = p.members[q];
            const double dx = x - (double)p.sens_xy[2 * i], dy = y - (double)p.sens_xy[2 * i + 1];
            double u = dx, v = dy;
            if (p.xform) {
                const float4 T = reinterpret_cast<const float4 *>(p.xform)[i];
                u = (double)T.x * dx + (double)T.y * dy;
                v = (double)T.z * dx + (double)T.w * dy;
            }
            if (!(u >= p.u_lo && u <= p.u_hi && v >= p.v_lo && v <= p.v_hi)) continue;              // R35
            double yv = (double)__ldg(sig + i) / (A * (double)p.gains[i]);
            if (p.axial) {
                const double r = fmin(fmax(sqrt(dx * dx + dy * dy), p.a_lo), p.a_hi);
                const double t = (r - p.a_lo) / ((p.a_hi - p.a_lo) / p.a_n);
                const int k = min((int)floor(t), p.a_n - 1);
                const double f = t - (double)k, o = 1.0 - f, f2 = f * f, f3 = f2 * f;
                yv -= (double)p.axial[k] * (o * o * o / 6.0) + (double)p.axial[k + 1] * ((3.0 * f3 - 6.0 * f2 + 4.0) / 6.0) +
                      (double)p.axial[k + 2] * ((-3.0 * f3 + 3.0 * f2 + 3.0 * f + 1.0) / 6.0) + (double)p.axial[k + 3] * (f3 / 6.0);
            }
            const double tu = (u - p.u_lo) / p.hu, tv = (v - p.v_lo) / p.hv;
            const int ku = min((int)floor(tu), p.nx - 1), kv = min((int)floor(tv), p.ny - 1);
            const double fu = tu - (double)ku, ou = 1.0 - fu, fu2 = fu * fu, fu3 = fu2 * fu;
            const double fv = tv - (double)kv, ov = 1.0 - fv, fv2 = fv * fv, fv3 = fv2 * fv;
            const double bu[4] = {ou * ou * ou / 6.0, (3.0 * fu3 - 6.0 * fu2 + 4.0) / 6.0,
                                  (-3.0 * fu3 + 3.0 * fu2 + 3.0 * fu + 1.0) / 6.0, fu3 / 6.0};
            const double bv[4] = {ov * ov * ov / 6.0, (3.0 * fv3 - 6.0 * fv2 + 4.0) / 6.0,
                                  (-3.0 * fv3 + 3.0 * fv2 + 3.0 * fv + 1.0) / 6.0, fv3 / 6.0};
#pragma unroll
            for (int b1 = 0; b1 < 4; ++b1)
#pragma unroll
                for (int a1 = 0; a1 < 4; ++a1) {
                    const double w0 = bv[b1] * bu[a1], w1 = w0 * wm;
                    double *row = xy_smem + (size_t)((kv + b1) * p.ncu + ku + a1) * 29;
                    if (wy != 0.0) atomicAdd(row + 28, w0 * wy * yv);
#pragma unroll
                    for (int b2 = b1; b2 < 4; ++b2)
#pragma unroll
                        for (int a2 = 0; a2 < 4; ++a2) {
                            if (b2 == b1 && a2 < a1) continue;
                            atomicAdd(row + (b2 - b1) * 7 + (a2 - a1) + 3, w1 * bv[b2] * bu[a2]);
                        }
                }
            ++used;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
    if (lane == 0 && used && (p.slab < 0 || p.part == 0)) atomicAdd(p.n_used, used);
    __syncthreads();
    for (int i = threadIdx.x; i < total; i += blockDim.x)
        if (xy_smem[i] != 0.0) atomicAdd(p.acc + i, xy_smem[i]);
}

}  // namespace ants

namespace ants {

// ---- axial LRF calculation, ONE shared profile (n_lrf = 1), without atomics in the loop (round 2) ----------------
// lrf_fit_kernel spends its time in shared-memory FP64 CAS loops (14 per pair, several lanes of a warp hitting the
// same interval).  Here every THREAD owns a private copy of the 5 (n + 3) band entries in shared memory, laid out
// [entry][thread] so that a warp's accesses to one entry are consecutive doubles: the 14 updates of a pair are plain
// load-add-store, free of conflicts and of retries, and the bound becomes the shared-memory bandwidth (224 B per
// pair).  The copies are summed once at the end and added to the global accumulators.
__global__ void __launch_bounds__(128) lrf_fit_shared_kernel(const FitParams p) {
    extern __shared__ double fs_smem[];                 // [nc * 5][blockDim.x]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5, T = blockDim.x;
    const int entries = p.nc * 5;
    for (int i = threadIdx.x; i < entries * T; i += T) fs_smem[i] = 0.0;
    __syncthreads();
    double *mine = fs_smem + threadIdx.x;
    unsigned long long used = 0ULL;
    // a lane keeps the sensors i = lane + 32 c: their constants stay in registers for all events
    double sx[4], sy[4], ginv[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = lane + 32 * c;
        sx[c] = i < p.N ? (double)p.sens_xy[2 * i] : 0.0;
        sy[c] = i < p.N ? (double)p.sens_xy[2 * i + 1] : 0.0;
        ginv[c] = i < p.N ? 1.0 / (double)p.gains[i] : 0.0;
    }
    const double inv_h = 1.0 / p.h;
    // few warps fit beside the private copies, so latency is covered inside the warp: the position rows and the
    // signals of the next two events wait in registers, and the (independent) arithmetic of a lane's four sensors
    // is written side by side before their updates
    const long long stride = (long long)gridDim.x * warps;
    constexpr int kAhead = 2;
    float4 pe_q[kAhead + 1];
    float sg_q[kAhead + 1][4];
    auto fetch = [&](int slot, long long ev) {
        const bool in = ev < p.n_events;
        pe_q[slot] = in ? __ldg(reinterpret_cast<const float4 *>(p.xyzA) + ev) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int i = lane + 32 * c;
            sg_q[slot][c] = (in && i < p.N) ? __ldg(p.signals + ev * p.N + i) : 0.f;
        }
    };
    // one pair's update of this thread's private band: all loads, then the adds, then the stores
    auto update = [&](int k, const double b4[4], double yv) {
        double *row = mine + (size_t)k * 5 * T;
        double v[14];
        int n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            v[n++] = row[(a * 5 + 4) * T];
#pragma unroll
            for (int c = a; c < 4; ++c) v[n++] = row[(a * 5 + c - a) * T];
        }
        n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            v[n++] += b4[a] * yv;
#pragma unroll
            for (int c = a; c < 4; ++c) v[n++] += b4[a] * b4[c];
        }
        n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            row[(a * 5 + 4) * T] = v[n++];
#pragma unroll
            for (int c = a; c < 4; ++c) row[(a * 5 + c - a) * T] = v[n++];
        }
    };
    auto prepare = [&](double x, double y, double sxi, double syi, double sv, double invAg, int &k, double b4[4], double &yv) -> bool {
        const double dx = x - sxi, dy = y - syi;
        const double r = sqrt(dx * dx + dy * dy);
        yv = sv * invAg;                                                                          // R21, R23
        const double t = (r - p.lo) * inv_h;
        k = min(max((int)floor(t), 0), p.n_int - 1);
        const double u = t - (double)k, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
        b4[0] = o * o * o * (1.0 / 6.0);
        b4[1] = (3.0 * u3 - 6.0 * u2 + 4.0) * (1.0 / 6.0);
        b4[2] = (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) * (1.0 / 6.0);
        b4[3] = u3 * (1.0 / 6.0);
        return r >= p.lo && r <= p.hi;                                                            // R22
    };
    const long long e0 = (long long)blockIdx.x * warps + warp;
#pragma unroll
    for (int a = 0; a < kAhead; ++a) fetch(a, e0 + a * stride);
    for (long long e = e0; e < p.n_events; e += stride) {
        fetch(kAhead, e + kAhead * stride);
        const float4 pe = pe_q[0];
        float sg[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) sg[c] = sg_q[0][c];
#pragma unroll
        for (int a = 0; a < kAhead; ++a) {
            pe_q[a] = pe_q[a + 1];
#pragma unroll
            for (int c = 0; c < 4; ++c) sg_q[a][c] = sg_q[a + 1][c];
        }
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;     // R22
        const double invA = 1.0 / A;
        int kk[4];
        double bb[4][4], yy[4];
        bool ok[4];
#pragma unroll
        for (int c = 0; c < 4; ++c)
            ok[c] = prepare(x, y, sx[c], sy[c], (double)sg[c], invA * ginv[c], kk[c], bb[c], yy[c]) && lane + 32 * c < p.N;
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (ok[c]) { update(kk[c], bb[c], yy[c]); ++used; }
        for (int i = lane + 128; i < p.N; i += 32) {                     // arrays of more than 128 sensors
            int k;
            double b4[4], yv;
            if (prepare(x, y, (double)p.sens_xy[2 * i], (double)p.sens_xy[2 * i + 1], (double)__ldg(p.signals + e * p.N + i),
                        invA / (double)p.gains[i], k, b4, yv)) {
                update(k, b4, yv);
                ++used;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
    if (lane == 0 && used) atomicAdd(p.n_used, used);
    __syncthreads();
    for (int i = threadIdx.x; i < entries; i += T) {
        double s = 0.0;
        for (int c = 0; c < T; ++c) s += fs_smem[(size_t)i * T + (c + threadIdx.x) % T];     // staggered: no bank conflicts
        if (s != 0.0) atomicAdd(p.acc + i, s);
    }
}

}  // namespace ants

namespace ants {

// ---- axial LRF calculation, ONE TABLE PER SENSOR (n_lrf = N, no groups), without atomics in the loop -----------------
// lrf_fit_kernel maps a warp to an event and lanes to sensors: several warps of a CTA update the same sensor's table,
// hence its shared-memory FP64 CAS loops.  Here a THREAD owns a sensor: thread t of every CTA takes sensor t of all the
// events its CTA sees, and that sensor's band, 5 (n + 3) entries, sits in column t of a shared-memory array laid out
// [entry][thread] -- the 14 updates of a pair are plain load-add-store, free of conflicts and of retries; the signals
// of an event are one coalesced row read, its position one broadcast load.  The columns are added to the global
// accumulators once at the end.  Needs N <= 128 and 40 (n + 3) N bytes of shared memory (the host checks; else
// lrf_fit_kernel).
__global__ void __launch_bounds__(128) lrf_fit_owned_kernel(const FitParams p) {
    extern __shared__ double fo_smem[];                 // [nc * 5][blockDim.x]
    const int T = blockDim.x, t = threadIdx.x;
    const int entries = p.nc * 5;
    for (int i = t; i < entries * T; i += T) fo_smem[i] = 0.0;
    __syncthreads();
    double *mine = fo_smem + t;
    const bool have = t < p.N;
    const double sx = have ? (double)p.sens_xy[2 * t] : 0.0, sy = have ? (double)p.sens_xy[2 * t + 1] : 0.0;
    const double inv_h = 1.0 / p.h;
    unsigned long long used = 0ULL;
    // the position rows and the signals of the next two events wait in registers (few warps fit beside the tables)
    constexpr int kAhead = 2;
    float4 pe_q[kAhead + 1];
    float sg_q[kAhead + 1];
    auto fetch = [&](int slot, long long ev) {
        const bool in = ev < p.n_events;
        pe_q[slot] = in ? __ldg(reinterpret_cast<const float4 *>(p.xyzA) + ev) : make_float4(0.f, 0.f, 0.f, 0.f);
        sg_q[slot] = (in && have) ? __ldg(p.signals + ev * p.N + t) : 0.f;
    };
    const long long stride = gridDim.x;
#pragma unroll
    for (int a = 0; a < kAhead; ++a) fetch(a, (long long)blockIdx.x + a * stride);
    for (long long e = blockIdx.x; e < p.n_events; e += stride) {
        fetch(kAhead, e + kAhead * stride);
        const float4 pe = pe_q[0];
        const double sv = (double)sg_q[0];
#pragma unroll
        for (int a = 0; a < kAhead; ++a) { pe_q[a] = pe_q[a + 1]; sg_q[a] = sg_q[a + 1]; }
        const double x = (double)pe.x, y = (double)pe.y, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308)) continue;     // R22 (CTA-uniform)
        const double dx = x - sx, dy = y - sy;
        const double r = sqrt(dx * dx + dy * dy);
        if (!(have && r >= p.lo && r <= p.hi)) continue;                                          // R22
        const double yv = sv / A;                                                                  // R21 (own table: no gain)
        const double tt = (r - p.lo) * inv_h;
        const int k = min(max((int)floor(tt), 0), p.n_int - 1);
        const double u = tt - (double)k, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
        const double b4[4] = {o * o * o * (1.0 / 6.0), (3.0 * u3 - 6.0 * u2 + 4.0) * (1.0 / 6.0),
                              (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) * (1.0 / 6.0), u3 * (1.0 / 6.0)};
        double *row = mine + (size_t)k * 5 * T;
        double v[14];
        int n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            v[n++] = row[(a * 5 + 4) * T];
#pragma unroll
            for (int c = a; c < 4; ++c) v[n++] = row[(a * 5 + c - a) * T];
        }
        n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            v[n++] += b4[a] * yv;
#pragma unroll
            for (int c = a; c < 4; ++c) v[n++] += b4[a] * b4[c];
        }
        n = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            row[(a * 5 + 4) * T] = v[n++];
#pragma unroll
            for (int c = a; c < 4; ++c) row[(a * 5 + c - a) * T] = v[n++];
        }
        ++used;
    }
    if (have) {
        if (used) atomicAdd(p.n_used + t, used);
        for (int j = 0; j < entries; ++j) {
            const double s = mine[(size_t)j * T];
            if (s != 0.0) atomicAdd(p.acc + (size_t)t * entries + j, s);
        }
    }
}

}  // namespace ants

namespace ants {

// ---- axial+z tensor LRF calculation, factorised per event (round 2) ------------------------------------------------
// All pairs of one event share the event's z, hence the same four z-basis weights bz: the event's contribution to
// the normal equations is (bz bz^T) (x) (sum_i br_i br_i^T) and to the right-hand side bz (x) (sum_i br_i y_i).  The
// warp therefore first accumulates the event's r-part -- the banded 4-wide matrix and the vector of an axial fit,
// 14 entries per pair -- in a buffer of its own, and then expands it once into the CTA's accumulators: about
// 1,200 conflict-free adds per event instead of 152 per pair (lrf_fit_rz_kernel; 4,500 per event on config 4).
__global__ void __launch_bounds__(256) lrf_fit_rz2_kernel(const FitRZParams p) {
    extern __shared__ double rz2_smem[];                // [nc][29] CTA accumulators, then [warps][ncr][5] r-parts
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int total = p.nc * 29, rlen = p.ncr * 5;
    for (int i = threadIdx.x; i < total + warps * rlen; i += blockDim.x) rz2_smem[i] = 0.0;
    __syncthreads();
    double *Rb = rz2_smem + total + (size_t)warp * rlen;      // [ncr][5]: {R[j][j], R[j][j+1], R[j][j+2], R[j][j+3], rhs[j]}
    unsigned long long used = 0ULL;
    for (long long e = (long long)blockIdx.x * warps + warp; e < p.n_events; e += (long long)gridDim.x * warps) {
        const float4 pe = reinterpret_cast<const float4 *>(p.xyzA)[e];
        const double x = (double)pe.x, y = (double)pe.y, z = (double)pe.z, A = (double)pe.w;
        if (!(fabs(x) <= 1.7e308 && fabs(y) <= 1.7e308 && A > 0.0 && A <= 1.7e308 && z >= p.z_lo && z <= p.z_hi)) continue;
        const double tz = (z - p.z_lo) / p.hz;
        const int kz = min((int)floor(tz), p.n_z - 1);
        const double uz = tz - (double)kz, oz = 1.0 - uz, uz2 = uz * uz, uz3 = uz2 * uz;
        const double bz[4] = {oz * oz * oz / 6.0, (3.0 * uz3 - 6.0 * uz2 + 4.0) / 6.0,
                              (-3.0 * uz3 + 3.0 * uz2 + 3.0 * uz + 1.0) / 6.0, uz3 / 6.0};
        const float *sig = p.signals + e * p.N;
        int k_min = p.ncr, k_max = -1;
        for (int i = lane; i < p.N; i += 32) {
            const double dx = x - (double)p.sens_xy[2 * i], dy = y - (double)p.sens_xy[2 * i + 1];
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r >= p.r_lo && r <= p.r_hi)) continue;
            const double yv = (double)__ldg(sig + i) / (A * (double)p.gains[i]);
            const double tr = (r - p.r_lo) / p.hr;
            const int kr = min((int)floor(tr), p.n_r - 1);
            const double u = tr - (double)kr, o = 1.0 - u, u2 = u * u, u3 = u2 * u;
            const double br[4] = {o * o * o / 6.0, (3.0 * u3 - 6.0 * u2 + 4.0) / 6.0,
                                  (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) / 6.0, u3 / 6.0};
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                double *row = Rb + (size_t)(kr + a) * 5;
                atomicAdd(row + 4, br[a] * yv);
#pragma unroll
                for (int c = a; c < 4; ++c) atomicAdd(row + (c - a), br[a] * br[c]);
            }
            k_min = min(k_min, kr);
            k_max = max(k_max, kr + 3);
            ++used;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            k_min = min(k_min, __shfl_xor_sync(0xffffffffu, k_min, o));
            k_max = max(k_max, __shfl_xor_sync(0xffffffffu, k_max, o));
        }
        __syncwarp();
        // expand: rows (kz + b1) ncr + ja, slots (dz, dr) of the 4 x 7 block and the right-hand side.  A lane takes one
        // (row ja, offset dr) entry of the r-part -- or the row's right-hand side -- and adds it to all (b1, dz) places
        // it belongs to, the z-weights bz[b1] bz[b1 + dz] with compile-time indices (the lanes of a warp hit distinct
        // addresses; only the warps of the CTA meet)
        const int n_rows = k_max - k_min + 1;
        const size_t zrow = (size_t)p.ncr * 29;
        double *zbase = rz2_smem + (size_t)kz * zrow;
        for (int it = lane; it < n_rows * 8; it += 32) {
            const int ja = k_min + (it >> 3), d = it & 7;
            if (d == 7) {
                const double rv = Rb[(size_t)ja * 5 + 4];
                if (rv != 0.0) {
#pragma unroll
                    for (int b1 = 0; b1 < 4; ++b1) atomicAdd(zbase + b1 * zrow + (size_t)ja * 29 + 28, bz[b1] * rv);
                }
            } else {
                const int dr = d - 3, jc = ja + dr;
                if (jc < 0 || jc >= p.ncr) continue;
                const double rv = Rb[(size_t)min(ja, jc) * 5 + (dr < 0 ? -dr : dr)];
                if (rv == 0.0) continue;
                double *q = zbase + (size_t)ja * 29 + d;
#pragma unroll
                for (int b1 = 0; b1 < 4; ++b1) {
                    if (dr >= 0) atomicAdd(q + b1 * zrow, bz[b1] * bz[b1] * rv);                    // dz = 0: upper triangle only
#pragma unroll
                    for (int dz = 1; dz < 4; ++dz)
                        if (b1 + dz <= 3) atomicAdd(q + b1 * zrow + dz * 7, bz[b1] * bz[b1 + dz] * rv);
                }
            }
        }
        __syncwarp();
        for (int it = lane; it < n_rows * 5; it += 32) Rb[(size_t)k_min * 5 + it] = 0.0;
        __syncwarp();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
    if (lane == 0 && used) atomicAdd(p.n_used, used);
    __syncthreads();
    for (int i = threadIdx.x; i < total; i += blockDim.x)
        if (rz2_smem[i] != 0.0) atomicAdd(p.acc + i, rz2_smem[i]);
}

}  // namespace ants
