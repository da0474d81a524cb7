// recon_common.cuh -- device-side parameter blocks and small helpers shared by
// the 2-D and 3-D contracting-grid kernels (section 5.1.2.2).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ants {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kMagic = 12582912.0f;     // 1.5 * 2^23: (t + kMagic) rounds t to the nearest integer
constexpr int kMagicBits = 0x4B400000;    // bit pattern of kMagic; low bits of (t + kMagic) hold round(t)
#define kInf (__int_as_float(0x7f800000))

// LRF model as the kernels see it (device pointers; built once in ants_lrf_create, step a0).
struct ModelDev {
    const float4 *sens;     // [N] {X, Y, gL, 1/g}: gL scales the table into L_i (the relative gain for a shared or
                            //   group profile, 1 for per-sensor tables); 1/g weights the centroid
    const int *grp;         // [N] table index of every sensor (0 for one shared profile, i for per-sensor tables,
                            //   the group index for a grouped model)
    const float4 *poly;     // axial: [n_lrf][n_r + 1] rows {q0,q1,q2,q3}: s = q0 + v(q1 + v(q2 + v q3)),
                            //   v = t - round(t - 0.5) - 0.5 in [-0.5, 0.5], t = (r - r_lo) * sc;
                            //   row n_r is the constant extension s(r_hi).
                            // axial+z: [n_z + 3][n_r + 1] such rows, one r-spline per z coefficient row
    const double *polyd;    // axial: [n_lrf][n_r][4] power basis in u = t - k in [0,1] (final score, FP64)
                            // axial+z: [n_z + 3][n_r][4]
    // XY-type parameterisations (recon_gen.cuh): B-spline coefficients of the XY tables
    // [n_lrf][n_planes or 1][ny + 3][nx + 3] (u fastest) and the sensors' local frames {T00, T01, T10, T11}
    const float *cxy;       // device, or nullptr
    const float4 *xf;       // device [N], or nullptr (identity)
    int lrf_kind;           // 1 Axial, 2 Axial+Z, 3 XY, 4 Composite, 5 Sliced
    int nx, ny, n_planes;
    float u_lo, su, v_lo, sv;   // su = nx / (u_hi - u_lo), sv = ny / (v_hi - v_lo)
    int N, n_lrf, n_r, n_z;
    float r_lo, r_hi, sc, of, tmax;   // sc = n_r/(r_hi - r_lo); of = -r_lo*sc - 0.5; tmax = n_r - 0.5
    float z_lo, z_hi, scz;            // scz = n_z/(z_hi - z_lo)
    // sensor selection (R19): passive[i] != 0 -> sensor left out of everything; signal_min / dist_max
    // (NaN = off) pick the sensors of the statistical part per event; select = any of the three is on
    const unsigned char *passive;     // device [N] or nullptr
    float signal_min, dist_max;
    int select;
};

// an inactive sensor of the current event is flagged by a NaN in SC[i].y
#define ANTS_QNAN (__int_as_float(0x7fc00000))

struct Params {
    ModelDev m;
    const float *signals;   // [E][N]
    long long n_events;
    float *out_xyzA;        // [E][4]
    float *out_score;       // [E]
    uint16_t *out_path;     // [E][K] or nullptr
    int G, K, nodes, dim;   // nodes = G^dim
    int k_diff;             // first iteration scored differentially (K = never)
    int k_series;           // 3-D Poisson: first iteration whose log1p is the series (before: lg2(1 + q))
    int positive;           // every LRF strictly positive on its domain (validity tests can be skipped)
    float h0_xy, h0_z, factor, z_seed;
    int seed_mode;          // 0 centroid, 1 strongest sensor (R20)
    // dynamic event distribution: ctr[0] = next event to hand out, ctr[1] = warps that have finished;
    // the last warp out zeroes both, so the pair is ready for the launch that reuses the slot
    unsigned long long *ctr;
    int total_warps;        // gridDim.x * warps_per_cta
    int warps_per_cta;
    int tile_events;        // events staged per CTA tile (= warps_per_cta)
    int gen_dtab;           // general kernel: a double copy of the XY coefficients sits in shared memory
    int reuse;              // packed 2-D kernel: carry coinciding nodes' scores over from the previous grid
    int lockstep;           // general kernel: the warps of a CTA take their events in rounds behind a barrier (the packed
                            // 2-D kernel has this as a template flag)
};

__device__ __forceinline__ float sqrt_approx(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- packed FP32 pairs (Blackwell FFMA2 / FADD2 / FMUL2: one issue slot, two lanes of work) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f32x2 pk1(float v) { return pk(v, v); }
__device__ __forceinline__ void upk(f32x2 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
// acc += a * b in place (keeps the accumulator in its register pair: no copy at the loop end)
__device__ __forceinline__ void fma2_acc(f32x2 &acc, f32x2 a, f32x2 b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float hsum2(f32x2 v) {
    float a, b;
    upk(v, a, b);
    return a + b;
}

// log2 of two positive, normal, finite numbers to a few ulp (relative, also next to 1, where lg2.approx has only an
// absolute bound), in a third of the instructions of two inlined log2f: x = 2^e m with m in [2/3, 4/3),
// log2 m = (2 / ln 2) atanh(s), s = (m - 1)/(m + 1), |s| <= 0.2, odd series to s^11 (next term 6e-11); the division
// is rcp.approx (1 ulp).  The plain score's term sumS log2(A_ref sumL / sumS) needs the relative accuracy: its
// argument is ~1 at the nodes that compete for the minimum (an absolute error of 2^-22 sumS broke the node-index
// rule on config 1 in round 2).
__device__ __forceinline__ f32x2 log2_pos2(float x0, float x1) {
    const int b0 = __float_as_int(x0), b1 = __float_as_int(x1);
    const int e0 = (b0 - 0x3f2aaaab) >> 23, e1 = (b1 - 0x3f2aaaab) >> 23;
    const f32x2 f = add2(pk(__int_as_float(b0 - (e0 << 23)), __int_as_float(b1 - (e1 << 23))), pk1(-1.f));
    float d0, d1;
    upk(add2(f, pk1(2.f)), d0, d1);
    const f32x2 s = mul2(f, pk(rcp_approx(d0), rcp_approx(d1))), t = mul2(s, s);
    const f32x2 poly = fma2(t, fma2(t, fma2(t, fma2(t, fma2(t, pk1(0.262308189f), pk1(0.320598898f)), pk1(0.412198583f)),
                                            pk1(0.577078016f)), pk1(0.961796694f)), pk1(2.885390082f));
    return fma2(s, poly, pk((float)e0, (float)e1));
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// argmin over the warp of (score, index); ties go to the lower index (R9).  All lanes get the result.
__device__ __forceinline__ void warp_argmin(float &s, int &idx) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        float os = __shfl_xor_sync(kFull, s, o);
        int oi = __shfl_xor_sync(kFull, idx, o);
        bool take = (os < s) || (os == s && oi < idx);
        s = take ? os : s;
        idx = take ? oi : idx;
    }
}

// next event for this warp (lane 0 draws from the launch's counter, all lanes get it)
__device__ __forceinline__ long long grab_event(unsigned long long *ctr, int lane) {
    unsigned long long v = 0ULL;
    if (lane == 0) v = atomicAdd(ctr, 1ULL);
    return (long long)__shfl_sync(kFull, v, 0);
}
// CTA-wide round: one thread takes `warps` consecutive events for the CTA, all threads learn the first (the two
// barriers also keep the CTA's warps in the same phase of the search: see recon2d_pk_kernel.cuh)
__device__ __forceinline__ long long grab_round(unsigned long long *ctr, int warps, long long *slot_s) {
    __syncthreads();
    if (threadIdx.x == 0) *slot_s = (long long)atomicAdd(ctr, (unsigned long long)warps);
    __syncthreads();
    return *slot_s;
}
// a warp is done: count it; the last one re-arms the counters
__device__ __forceinline__ void retire_warp(unsigned long long *ctr, int total_warps, int lane) {
    if (lane == 0) {
        const unsigned long long d = atomicAdd(ctr + 1, 1ULL);
        if (d == (unsigned long long)(total_warps - 1)) {
            ctr[0] = 0ULL;
            ctr[1] = 0ULL;
            __threadfence();
        }
    }
}

// start position = axis of the sensor with the strongest signal (R20): largest prepared signal among
// the sensors not flagged passive (NaN in SC[i].y), lowest index on ties.  Each lane scans the sensors
// it loaded itself (i = lane + 32 c), so no synchronisation is needed before the call.
__device__ __forceinline__ void strongest_sensor(const float2 *SC, const float4 *sens_s, int N, int lane,
                                                 float &cx, float &cy) {
    float key = kInf;            // -S of the lane's best
    int bi = 0x7fffffff;
    for (int i = lane; i < N; i += 32) {
        const float2 sc = SC[i];
        if (sc.y == sc.y && -sc.x < key) { key = -sc.x; bi = i; }
    }
    warp_argmin(key, bi);
    bi = min(bi, N - 1);
    cx = sens_s[bi].x;
    cy = sens_s[bi].y;
}

// ---- step a1 for one event, shared by the kernels that do not prefetch: load the signals (coalesced), prepare
// them (R18), centroid or strongest-sensor start (R20), sensor selection (R19).  SC[i] receives
// {S_i, log2(S_i / gL_i) or 0}, an inactive sensor is flagged by NaN in .y.  Returns false when the event fails
// (its outputs are written here: NaN row, score +inf, path 0xFFFF).
struct Params;
// `pre` (optional): the event's first 128 signals already in registers, pre[c] = signal of sensor lane + 32 c.
template <int METHOD>
__device__ bool prepare_event(const Params &p, const float4 *sens_s, float2 *SC, long long e, int lane,
                              float &sumS, float &cx, float &cy, const float *pre = nullptr);

// same result as warp_argmin through two integer reductions (REDUX): scores mapped to order-preserving
// unsigned keys, then the lowest index among the lanes holding the minimum.  s must not be NaN.
__device__ __forceinline__ void warp_argmin_redux(float &s, int &idx) {
    unsigned b = s == 0.f ? 0u : __float_as_uint(s);   // -0 and +0 tie
    unsigned key = (b & 0x80000000u) ? ~b : (b | 0x80000000u);
    unsigned kmin = __reduce_min_sync(kFull, key);
    int cand = key == kmin ? idx : 0x7fffffff;
    idx = __reduce_min_sync(kFull, cand);
    unsigned bm = (kmin & 0x80000000u) ? (kmin & 0x7fffffffu) : ~kmin;
    s = __uint_as_float(bm);
}

// round-to-nearest interval index k and centred local coordinate v of t in [-0.5, tmax]
__device__ __forceinline__ void split_t(float t, int &k, float &v) {
    float tm = t + kMagic;
    k = __float_as_int(tm) - kMagicBits;
    v = t - (tm - kMagic);
}

// 16-byte shared-memory load from a 32-bit shared address
__device__ __forceinline__ float4 lds128(unsigned addr) {
    float4 v;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// CTA-shared model tables of the axial kernels: sens_s [N] float4, poly_s [rows] float4, grp_s [N] int (padded)
__host__ __device__ inline size_t cta_table_bytes(int N, int rows) {
    return (size_t)(N + rows) * 16 + ((size_t)N * 4 + 15) / 16 * 16;
}

__device__ __forceinline__ float horner(const float4 p, float v) {
    return fmaf(fmaf(fmaf(p.w, v, p.z), v, p.y), v, p.x);
}

template <int METHOD>
__device__ __forceinline__ bool prepare_event(const Params &p, const float4 *sens_s, float2 *SC, long long e, int lane,
                                              float &sumS, float &cx, float &cy, const float *pre) {
    const ModelDev &m = p.m;
    const int N = m.N;
    const float *sig = p.signals + e * N;
    float sw = 0.f, sxw = 0.f, syw = 0.f;
    sumS = 0.f;
    bool finite = true;
#pragma unroll 4
    for (int i = lane, c = 0; i < N; i += 32, ++c) {
        if (m.passive && m.passive[i]) {             // R19: out of everything, signal not looked at
            SC[i] = make_float2(0.f, ANTS_QNAN);
            continue;
        }
        float S;
        if (pre && c < 4) S = c == 0 ? pre[0] : c == 1 ? pre[1] : c == 2 ? pre[2] : pre[3];
        else S = __ldg(sig + i);
        finite = finite && (fabsf(S) <= 3.402823466e38f);
        if (METHOD == 0) S = fmaxf(S, 0.f);          // R18
        const float4 sn = sens_s[i];
        const float wgt = S * sn.w;
        sumS += S;
        sw += wgt;
        sxw = fmaf(sn.x, wgt, sxw);
        syw = fmaf(sn.y, wgt, syw);
        float cs = 0.f;
        // c_i = log2(S_i / g_i) only conditions the plain score (sum_i S_i c_i is the same at every node), so the
        // fast forms do: an error in it shifts all scores of the event alike
        if (METHOD == 0 && S > 0.f) cs = lg2_approx(fmaxf(S * rcp_approx(sn.z), 1e-30f));
        SC[i] = make_float2(S, cs);
    }
    finite = __all_sync(kFull, finite);
    sumS = warp_sum(sumS);
    sw = warp_sum(sw);
    sxw = warp_sum(sxw);
    syw = warp_sum(syw);
    __syncwarp();
    bool ok = finite && (sumS > 0.f) && (p.seed_mode != 0 || sw > 0.f);
    if (ok) {
        cx = sxw / sw;
        cy = syw / sw;
        if (p.seed_mode == 1) strongest_sensor(SC, sens_s, N, lane, cx, cy);    // R20
        if (m.select) {
            // R19: the sensors of the statistical part, fixed for the event: signal threshold and distance
            // from the start position; sum S runs over them
            float s_act = 0.f;
            for (int i = lane; i < N; i += 32) {
                const float2 sc = SC[i];
                if (sc.y == sc.y) {
                    const float4 sn = sens_s[i];
                    const float dx = cx - sn.x, dy = cy - sn.y;
                    const bool keep = !(sc.x < m.signal_min) && !(sqrtf(fmaf(dx, dx, dy * dy)) > m.dist_max);
                    if (keep) s_act += sc.x;
                    else SC[i] = make_float2(0.f, ANTS_QNAN);
                }
            }
            sumS = warp_sum(s_act);
            __syncwarp();
            ok = sumS > 0.f;
        }
    }
    if (!ok) {
        if (lane == 0) {
            reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(ANTS_QNAN, ANTS_QNAN, ANTS_QNAN, ANTS_QNAN);
            p.out_score[e] = kInf;
        }
        if (p.out_path)
            for (int k = lane; k < p.K; k += 32) p.out_path[e * p.K + k] = 0xFFFF;
    }
    return ok;
}

}  // namespace ants
