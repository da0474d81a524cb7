// ants_recon.cu -- C ABI (include/ants_recon.h) and host logic of the B200
// contracting-grid reconstruction: table build (step a0), launch planning,
// kernel dispatch, the streamed host-buffer pipeline.  No CPU fallback: every
// reconstruction step runs in the kernels of recon2d.cuh / recon3d.cuh.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <array>
#include <atomic>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/ants_recon.h"
#include "recon2d.cuh"
#include "recon2d_pk.cuh"
#include "recon3d.cuh"
#include "recon3d_pk.cuh"
#include "recon_gen.cuh"
#include "refine.cuh"
#include "kernels.h"

using namespace ants;

// launches that may be in flight at once on one model (each owns a counter pair until its last warp retires);
// a launch that wraps around the ring waits, on the device, for the previous user of its slot
static const unsigned kCtrSlots = 1024;

// ---------------------------------------------------------------------------
// the opaque handle
// ---------------------------------------------------------------------------
// launch plan of one (grid, method) on one model: computed once, cached in the handle
struct Plan {
    int npt = 0;             // nodes per lane (template instantiation)
    int cpl = 0, gzm = 0;    // axial+z kernel: columns per lane, compiled z-levels
    int lockstep = 0;        // packed 2-D kernel: CTA-wide event rounds behind a barrier
    bool cross = false;      // packed axial+z kernel: top level of an odd grid packed across the lane's two columns
    int family = 0;          // 0 recon2d_pk_kernel, 2 recon3d_kernel, 3 recon_gen_kernel (general), 4 recon3d_pk_kernel
    int warps = 0;           // warps per CTA
    int ctas_per_sm = 0;     // resident CTAs per SM (cudaOccupancyMaxActiveBlocksPerMultiprocessor, capped by the tuning knob)
    size_t smem = 0;         // dynamic shared memory per CTA
    int k_diff = 0;          // first differential iteration (K = never)
    int k_series = 0;        // axial+z Poisson: first iteration with the log1p series
    int gen_dtab = 0;        // general kernel: double copy of the XY coefficients in shared memory
    int reuse = 0;           // packed 2-D kernel: the node-reuse instantiation
    const void *kernel = nullptr;
    bool ready = false;      // cudaFuncSetAttribute + occupancy done (needs the device)
};
struct PlanKey {
    int32_t dim, G, K, method, select;
    float step0_xy, step0_z, factor;
    bool operator==(const PlanKey &o) const {
        return dim == o.dim && G == o.G && K == o.K && method == o.method && select == o.select &&
               step0_xy == o.step0_xy && step0_z == o.step0_z && factor == o.factor;
    }
};

struct ants_lrf {
    ModelDev dev{};          // device pointers + scalars, passed by value to the kernels
    std::mutex plan_mu;      // guards plans
    std::vector<std::pair<PlanKey, Plan>> plans;
    void *d_grp = nullptr, *d_cxy = nullptr, *d_xf = nullptr;
    double knot_xy = 0.0;    // XY-type models: smallest knot spacing of the XY spline, mm
    cudaEvent_t *slot_ev = nullptr;   // [kCtrSlots] lazily created: the launch that last used a counter slot
    int device = 0;
    int sm_count = 0;
    bool positive = false;   // every spline strictly positive on its domain
    double max_dlog = 0.0;   // max |d ln s / dr| over the domain, 1/mm (only if positive)
    double max_dlog_z = 0.0; // axial+z: max |d ln s / dz|, 1/mm
    double knot_r = 0.0, knot_z = 0.0;   // knot spacing, mm
    void *d_sens = nullptr, *d_poly = nullptr, *d_polyd = nullptr, *d_passive = nullptr;
    unsigned long long *d_ctr = nullptr;   // ring of per-launch event counters {next, done}
    std::atomic<unsigned> next_slot{0};
    // scratch of ants_reconstruct_host (lazily allocated, reused, guarded)
    std::mutex host_mu;
    int64_t scratch_events = 0;
    float *d_sig[3] = {nullptr, nullptr, nullptr};
    float *d_xyzA[3] = {nullptr, nullptr, nullptr};
    float *d_score[3] = {nullptr, nullptr, nullptr};
    cudaStream_t streams[3] = {nullptr, nullptr, nullptr};
};

static std::atomic<int64_t> g_launches{0};

// ---------------------------------------------------------------------------
// step a0: B-spline coefficients -> per-interval cubics
// ---------------------------------------------------------------------------
// Uniform cubic B-spline on interval k with local u in [0,1] (R7), power basis:
//   s = p0 + p1 u + p2 u^2 + p3 u^3 from the four coefficients c[k..k+3].
static void interval_power(const float *c, double p[4]) {
    const double c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3];
    p[0] = (c0 + 4.0 * c1 + c2) / 6.0;
    p[1] = (c2 - c0) / 2.0;
    p[2] = (c0 - 2.0 * c1 + c2) / 2.0;
    p[3] = (c3 - c0 + 3.0 * (c1 - c2)) / 6.0;
}

// minimum of the cubic on [0,1] (end points and interior critical points)
static double cubic_min01(const double p[4]) {
    auto f = [&](double u) { return p[0] + u * (p[1] + u * (p[2] + u * p[3])); };
    double mn = std::fmin(f(0.0), f(1.0));
    const double a = 3.0 * p[3], b = 2.0 * p[2], c = p[1];
    if (std::fabs(a) > 0.0) {
        double disc = b * b - 4.0 * a * c;
        if (disc >= 0.0) {
            double sq = std::sqrt(disc);
            for (double u : {(-b + sq) / (2.0 * a), (-b - sq) / (2.0 * a)})
                if (u > 0.0 && u < 1.0) mn = std::fmin(mn, f(u));
        }
    } else if (std::fabs(b) > 0.0) {
        double u = -c / b;
        if (u > 0.0 && u < 1.0) mn = std::fmin(mn, f(u));
    }
    return mn;
}

// one r-spline (n_r + 3 coefficients) -> fp32 centred rows [n_r + 1] and fp64 rows [n_r][4];
// updates positivity and the log-derivative bound
static void build_rows(const float *c, int n_r, double sc_r, float4 *rows32, double *rows64,
                       bool &positive, double &max_dlog) {
    double last[4] = {0, 0, 0, 0};
    for (int k = 0; k < n_r; ++k) {
        double p[4];
        interval_power(c + k, p);
        for (int a = 0; a < 4; ++a) rows64[4 * k + a] = p[a];
        // re-centre to v = u - 1/2
        rows32[k] = make_float4((float)(p[0] + 0.5 * p[1] + 0.25 * p[2] + 0.125 * p[3]),
                                (float)(p[1] + p[2] + 0.75 * p[3]), (float)(p[2] + 1.5 * p[3]), (float)p[3]);
        if (!(cubic_min01(p) > 0.0)) positive = false;
        for (int s = 0; s <= 16; ++s) {
            double u = s / 16.0;
            double f = p[0] + u * (p[1] + u * (p[2] + u * p[3]));
            double d = p[1] + u * (2.0 * p[2] + 3.0 * u * p[3]);
            if (f > 0.0) max_dlog = std::fmax(max_dlog, std::fabs(d) * sc_r / f);
        }
        for (int a = 0; a < 4; ++a) last[a] = p[a];
    }
    // row n_r: constant extension s(r_hi) (R5)
    rows32[n_r] = make_float4((float)(last[0] + last[1] + last[2] + last[3]), 0.f, 0.f, 0.f);
}

// bicubic Bezier patch, positivity by recursive de Casteljau subdivision: positive if every control
// point is > 0 (convex hull); not positive if a corner (a true surface value) is <= 0; otherwise
// split in four.  Depth-limited: undecided counts as not positive (conservative).
struct Patch { double p[4][4]; };
static void split_cubic(const double in[4], double lo[4], double hi[4]) {
    const double m01 = 0.5 * (in[0] + in[1]), m12 = 0.5 * (in[1] + in[2]), m23 = 0.5 * (in[2] + in[3]);
    const double m012 = 0.5 * (m01 + m12), m123 = 0.5 * (m12 + m23), mid = 0.5 * (m012 + m123);
    lo[0] = in[0]; lo[1] = m01; lo[2] = m012; lo[3] = mid;
    hi[0] = mid; hi[1] = m123; hi[2] = m23; hi[3] = in[3];
}
static bool patch_positive(const Patch &P, int depth) {
    double mn = P.p[0][0];
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) mn = std::fmin(mn, P.p[a][b]);
    if (mn > 0.0) return true;
    if (!(P.p[0][0] > 0.0) || !(P.p[0][3] > 0.0) || !(P.p[3][0] > 0.0) || !(P.p[3][3] > 0.0)) return false;
    if (depth >= 10) return false;
    Patch rl, rh;     // split along the second index
    for (int a = 0; a < 4; ++a) split_cubic(P.p[a], rl.p[a], rh.p[a]);
    for (const Patch *half : {&rl, &rh}) {
        Patch zl, zh; // split along the first index
        for (int b = 0; b < 4; ++b) {
            double in[4] = {half->p[0][b], half->p[1][b], half->p[2][b], half->p[3][b]}, lo[4], hi[4];
            split_cubic(in, lo, hi);
            for (int a = 0; a < 4; ++a) { zl.p[a][b] = lo[a]; zh.p[a][b] = hi[a]; }
        }
        if (!patch_positive(zl, depth + 1) || !patch_positive(zh, depth + 1)) return false;
    }
    return true;
}

// axial+z: positivity and log-slopes of the tensor-product spline s(r, z).
// Positivity: Bezier control nets of every bicubic patch, subdivided until decided (patch_positive).
// Slopes: max |ds/dr|/s and |ds/dz|/s on a 9 x 9 sample of every patch (sizes the log1p series range).
static void tensor_analysis(const float *c, const double *rows64, int n_r, int n_z, double sc_r, double sc_z,
                            bool &positive, double &dlog_r, double &dlog_z) {
    static const double M[4][4] = {{1 / 6.0, 4 / 6.0, 1 / 6.0, 0}, {0, 4 / 6.0, 2 / 6.0, 0},
                                   {0, 2 / 6.0, 4 / 6.0, 0}, {0, 1 / 6.0, 4 / 6.0, 1 / 6.0}};
    positive = true;
    dlog_r = dlog_z = 0.0;
    const int nc = n_r + 3;
    for (int kz = 0; kz < n_z; ++kz)
        for (int kr = 0; kr < n_r; ++kr) {
            Patch P;
            for (int a = 0; a < 4; ++a)
                for (int b = 0; b < 4; ++b) {
                    double v = 0.0;
                    for (int i = 0; i < 4; ++i)
                        for (int j = 0; j < 4; ++j) v += M[a][i] * M[b][j] * (double)c[(kz + i) * nc + kr + j];
                    P.p[a][b] = v;
                }
            if (!patch_positive(P, 0)) positive = false;
            for (int iz = 0; iz <= 8; ++iz) {
                const double u = iz / 8.0, o = 1.0 - u;
                const double bz[4] = {o * o * o / 6.0, (3 * u * u * u - 6 * u * u + 4) / 6.0,
                                      (-3 * u * u * u + 3 * u * u + 3 * u + 1) / 6.0, u * u * u / 6.0};
                const double dz[4] = {-o * o / 2.0, (9 * u * u - 12 * u) / 6.0, (-9 * u * u + 6 * u + 3) / 6.0, u * u / 2.0};
                for (int ir = 0; ir <= 8; ++ir) {
                    const double t = ir / 8.0;
                    double sv = 0.0, sr = 0.0, sz = 0.0;
                    for (int b = 0; b < 4; ++b) {
                        const double *q = rows64 + ((size_t)(kz + b) * n_r + kr) * 4;
                        const double f = q[0] + t * (q[1] + t * (q[2] + t * q[3]));
                        const double d = q[1] + t * (2.0 * q[2] + 3.0 * t * q[3]);
                        sv += bz[b] * f;
                        sr += bz[b] * d;
                        sz += dz[b] * f;
                    }
                    if (sv > 0.0) {
                        dlog_r = std::fmax(dlog_r, std::fabs(sr) * sc_r / sv);
                        dlog_z = std::fmax(dlog_z, std::fabs(sz) * sc_z / sv);
                    } else {
                        positive = false;
                    }
                }
            }
        }
}

static bool finite_f(float v) { return std::isfinite(v); }

struct ants_lrf;
// group == nullptr: n_lrf = 1 (all sensors on table 0, L = g s) or n_lrf = N (sensor i on table i, L = s_i)
static int create_impl(const float *sensor_xy, const float *gains, const int32_t *group, const float *knots,
                       const float *coeffs, const ants_lrf_dims_t *dims, ants_lrf_t **out) {
    if (!out) return ANTS_ERR_INVALID;
    *out = nullptr;
    if (!sensor_xy || !knots || !coeffs || !dims) return ANTS_ERR_INVALID;
    const int N = dims->n_sensors, n_lrf = dims->n_lrf, dim = dims->lrf_dim, n_r = dims->n_int_r;
    const int n_z = dim == 2 ? dims->n_int_z : 0;
    if (N < 1 || N > 65535 || (dim != 1 && dim != 2) || n_r < 1 || n_r > 4096) return ANTS_ERR_INVALID;
    if (group) {
        if (n_lrf < 1 || n_lrf > N) return ANTS_ERR_INVALID;
        for (int i = 0; i < N; ++i)
            if (group[i] < 0 || group[i] >= n_lrf) return ANTS_ERR_INVALID;
        if (dim != 1) return ANTS_ERR_UNSUPPORTED;
    } else if (n_lrf != 1 && n_lrf != N) {
        return ANTS_ERR_INVALID;
    }
    if (dim == 2 && (n_z < 1 || n_z > 1024)) return ANTS_ERR_INVALID;
    const float r_lo = knots[0], r_hi = knots[1];
    if (!finite_f(r_lo) || !finite_f(r_hi) || !(r_lo >= 0.f) || !(r_hi > r_lo)) return ANTS_ERR_INVALID;
    float z_lo = 0.f, z_hi = 1.f;
    if (dim == 2) {
        z_lo = knots[2];
        z_hi = knots[3];
        if (!finite_f(z_lo) || !finite_f(z_hi) || !(z_hi > z_lo)) return ANTS_ERR_INVALID;
    }
    for (int i = 0; i < N; ++i) {
        if (!finite_f(sensor_xy[2 * i]) || !finite_f(sensor_xy[2 * i + 1])) return ANTS_ERR_INVALID;
        if (gains && !(gains[i] > 0.f && finite_f(gains[i]))) return ANTS_ERR_INVALID;
    }
    const int n_rows_z = dim == 2 ? n_z + 3 : 1;
    const size_t n_coef = (size_t)n_lrf * n_rows_z * (n_r + 3);
    for (size_t j = 0; j < n_coef; ++j)
        if (!finite_f(coeffs[j])) return ANTS_ERR_INVALID;
    if (dim == 2 && n_lrf != 1) return ANTS_ERR_UNSUPPORTED;

    ants_lrf *h = new (std::nothrow) ants_lrf;
    if (!h) return ANTS_ERR_NOMEM;
    cudaDeviceProp prop;
    if (cudaGetDevice(&h->device) != cudaSuccess ||
        cudaGetDeviceProperties(&prop, h->device) != cudaSuccess) {
        delete h;
        return ANTS_ERR_CUDA;
    }
    h->sm_count = prop.multiProcessorCount;

    const size_t n_spl = (size_t)n_lrf * n_rows_z;   // r-splines in the table
    std::vector<float4> sens(N), rows32(n_spl * (n_r + 1));
    std::vector<double> rows64(n_spl * n_r * 4);
    std::vector<int> grp(N);
    // a shared or group profile is scaled by the relative gain; per-sensor tables are not
    const bool scaled = group != nullptr || n_lrf == 1;
    for (int i = 0; i < N; ++i) {
        float g = gains ? gains[i] : 1.f;
        sens[i] = make_float4(sensor_xy[2 * i], sensor_xy[2 * i + 1], scaled ? g : 1.f, 1.f / g);
        grp[i] = group ? group[i] : (n_lrf == 1 ? 0 : i);
    }
    const double sc_r = (double)n_r / ((double)r_hi - (double)r_lo);
    bool positive = true;
    double max_dlog = 0.0;
    for (size_t s = 0; s < n_spl; ++s)
        build_rows(coeffs + s * (n_r + 3), n_r, sc_r, rows32.data() + s * (n_r + 1),
                   rows64.data() + s * n_r * 4, positive, max_dlog);
    double max_dlog_z = 0.0;
    if (dim == 2) tensor_analysis(coeffs, rows64.data(), n_r, n_z, sc_r, (double)n_z / ((double)z_hi - (double)z_lo),
                                  positive, max_dlog, max_dlog_z);
    h->positive = positive;
    h->max_dlog = max_dlog;
    h->max_dlog_z = max_dlog_z;
    h->knot_r = 1.0 / sc_r;
    h->knot_z = dim == 2 ? ((double)z_hi - (double)z_lo) / n_z : 0.0;

    h->slot_ev = new (std::nothrow) cudaEvent_t[kCtrSlots]();
    if (!h->slot_ev) { delete h; return ANTS_ERR_NOMEM; }
    cudaError_t e0 = cudaMalloc(&h->d_ctr, kCtrSlots * 2 * sizeof(unsigned long long));
    if (e0 == cudaSuccess) e0 = cudaMemset(h->d_ctr, 0, kCtrSlots * 2 * sizeof(unsigned long long));
    cudaError_t e1 = cudaMalloc(&h->d_sens, sens.size() * sizeof(float4));
    cudaError_t e2 = cudaMalloc(&h->d_poly, rows32.size() * sizeof(float4));
    cudaError_t e3 = cudaMalloc(&h->d_polyd, rows64.size() * sizeof(double));
    cudaError_t e4 = cudaMalloc(&h->d_grp, grp.size() * sizeof(int));
    if (e0 != cudaSuccess || e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess) {
        cudaGetLastError();
        ants_destroy(h);
        return (e1 == cudaErrorMemoryAllocation || e2 == cudaErrorMemoryAllocation ||
                e3 == cudaErrorMemoryAllocation || e4 == cudaErrorMemoryAllocation) ? ANTS_ERR_NOMEM : ANTS_ERR_CUDA;
    }
    if (cudaMemcpy(h->d_sens, sens.data(), sens.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->d_poly, rows32.data(), rows32.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->d_polyd, rows64.data(), rows64.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->d_grp, grp.data(), grp.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        ants_destroy(h);
        return ANTS_ERR_CUDA;
    }
    ModelDev &m = h->dev;
    m.sens = (const float4 *)h->d_sens;
    m.grp = (const int *)h->d_grp;
    m.cxy = nullptr;
    m.xf = nullptr;
    m.nx = m.ny = m.n_planes = 0;
    m.u_lo = m.v_lo = 0.f;
    m.su = m.sv = 1.f;
    m.poly = (const float4 *)h->d_poly;
    m.polyd = (const double *)h->d_polyd;
    m.N = N;
    m.n_lrf = n_lrf;
    m.n_r = n_r;
    m.n_z = n_z;
    m.r_lo = r_lo;
    m.r_hi = r_hi;
    m.sc = (float)sc_r;
    m.of = (float)(-(double)r_lo * sc_r - 0.5);
    m.tmax = (float)n_r - 0.5f;
    m.z_lo = z_lo;
    m.z_hi = z_hi;
    m.scz = dim == 2 ? (float)((double)n_z / ((double)z_hi - (double)z_lo)) : 0.f;
    m.passive = nullptr;
    m.signal_min = m.dist_max = std::nanf("");
    m.select = 0;
    m.lrf_kind = dim;
    *out = h;
    return ANTS_OK;
}

static int create_xy_impl(const float *sensor_xy, const float *gains, const float *knots, const float *coeffs,
                          const ants_lrf_dims_t *dims, const ants_lrf_xy_t *xy, ants_lrf_t **out) {
    if (!out) return ANTS_ERR_INVALID;
    *out = nullptr;
    if (!sensor_xy || !dims || !xy || !xy->knots_xy || !xy->coeffs_xy) return ANTS_ERR_INVALID;
    const int N = dims->n_sensors, n_lrf = dims->n_lrf, kind = dims->lrf_dim;
    if (kind != 3 && kind != 4 && kind != 5) return ANTS_ERR_INVALID;
    const int nx = xy->n_int_x, ny = xy->n_int_y, n_planes = kind == 5 ? xy->n_planes : 0;
    if (N < 1 || N > 65535 || nx < 1 || ny < 1 || nx > 1024 || ny > 1024) return ANTS_ERR_INVALID;
    if (kind == 5 && (n_planes < 2 || n_planes > 4096)) return ANTS_ERR_INVALID;
    if (xy->group) {
        if (n_lrf < 1 || n_lrf > N) return ANTS_ERR_INVALID;
        for (int i = 0; i < N; ++i)
            if (xy->group[i] < 0 || xy->group[i] >= n_lrf) return ANTS_ERR_INVALID;
    } else if (n_lrf != 1 && n_lrf != N) {
        return ANTS_ERR_INVALID;
    }
    const float *kx = xy->knots_xy;
    for (int j = 0; j < (kind == 5 ? 6 : 4); ++j)
        if (!finite_f(kx[j])) return ANTS_ERR_INVALID;
    if (!(kx[1] > kx[0]) || !(kx[3] > kx[2]) || (kind == 5 && !(kx[5] > kx[4]))) return ANTS_ERR_INVALID;
    const size_t ncxy = (size_t)n_lrf * (n_planes > 0 ? n_planes : 1) * (nx + 3) * (ny + 3);
    for (size_t j = 0; j < ncxy; ++j)
        if (!finite_f(xy->coeffs_xy[j])) return ANTS_ERR_INVALID;
    for (int i = 0; i < N; ++i) {
        if (!finite_f(sensor_xy[2 * i]) || !finite_f(sensor_xy[2 * i + 1])) return ANTS_ERR_INVALID;
        if (gains && !(gains[i] > 0.f && finite_f(gains[i]))) return ANTS_ERR_INVALID;
        if (xy->xform)
            for (int j = 0; j < 4; ++j)
                if (!finite_f(xy->xform[4 * i + j])) return ANTS_ERR_INVALID;
    }
    // the axial component of a Composite model goes through the axial table builder
    int n_r = 1;
    float r_lo = 0.f, r_hi = 1.f;
    if (kind == 4) {
        if (!knots || !coeffs) return ANTS_ERR_INVALID;
        n_r = dims->n_int_r;
        r_lo = knots[0];
        r_hi = knots[1];
        if (n_r < 1 || n_r > 4096 || !finite_f(r_lo) || !finite_f(r_hi) || !(r_lo >= 0.f) || !(r_hi > r_lo)) return ANTS_ERR_INVALID;
        for (size_t j = 0; j < (size_t)n_lrf * (n_r + 3); ++j)
            if (!finite_f(coeffs[j])) return ANTS_ERR_INVALID;
    }
    ants_lrf *h = new (std::nothrow) ants_lrf;
    if (!h) return ANTS_ERR_NOMEM;
    cudaDeviceProp prop;
    if (cudaGetDevice(&h->device) != cudaSuccess || cudaGetDeviceProperties(&prop, h->device) != cudaSuccess) {
        delete h;
        return ANTS_ERR_CUDA;
    }
    h->sm_count = prop.multiProcessorCount;
    h->slot_ev = new (std::nothrow) cudaEvent_t[kCtrSlots]();
    if (!h->slot_ev) { delete h; return ANTS_ERR_NOMEM; }
    const bool scaled = xy->group != nullptr || n_lrf == 1;
    std::vector<float4> sens(N), xf(N);
    std::vector<int> grp(N);
    for (int i = 0; i < N; ++i) {
        const float g = gains ? gains[i] : 1.f;
        sens[i] = make_float4(sensor_xy[2 * i], sensor_xy[2 * i + 1], scaled ? g : 1.f, 1.f / g);
        grp[i] = xy->group ? xy->group[i] : (n_lrf == 1 ? 0 : i);
        xf[i] = xy->xform ? make_float4(xy->xform[4 * i], xy->xform[4 * i + 1], xy->xform[4 * i + 2], xy->xform[4 * i + 3])
                          : make_float4(1.f, 0.f, 0.f, 1.f);
    }
    std::vector<float4> rows32;
    std::vector<double> rows64;
    const double sc_r = (double)n_r / ((double)r_hi - (double)r_lo);
    if (kind == 4) {
        rows32.resize((size_t)n_lrf * (n_r + 1));
        rows64.resize((size_t)n_lrf * n_r * 4);
        bool pos = true;
        double dl = 0.0;
        for (int t = 0; t < n_lrf; ++t)
            build_rows(coeffs + (size_t)t * (n_r + 3), n_r, sc_r, rows32.data() + (size_t)t * (n_r + 1),
                       rows64.data() + (size_t)t * n_r * 4, pos, dl);
    }
    h->positive = false;             // general kernel: per-pair validity rules
    h->knot_r = kind == 4 ? 1.0 / sc_r : 1e300;
    h->knot_xy = std::fmin(((double)kx[1] - (double)kx[0]) / nx, ((double)kx[3] - (double)kx[2]) / ny);
    bool ok = cudaMalloc(&h->d_ctr, kCtrSlots * 2 * sizeof(unsigned long long)) == cudaSuccess &&
              cudaMemset(h->d_ctr, 0, kCtrSlots * 2 * sizeof(unsigned long long)) == cudaSuccess &&
              cudaMalloc(&h->d_sens, sens.size() * sizeof(float4)) == cudaSuccess &&
              cudaMalloc(&h->d_grp, grp.size() * sizeof(int)) == cudaSuccess &&
              cudaMalloc(&h->d_xf, xf.size() * sizeof(float4)) == cudaSuccess &&
              cudaMalloc(&h->d_cxy, ncxy * sizeof(float)) == cudaSuccess &&
              (rows32.empty() || (cudaMalloc(&h->d_poly, rows32.size() * sizeof(float4)) == cudaSuccess &&
                                  cudaMalloc(&h->d_polyd, rows64.size() * sizeof(double)) == cudaSuccess));
    ok = ok && cudaMemcpy(h->d_sens, sens.data(), sens.size() * sizeof(float4), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h->d_grp, grp.data(), grp.size() * sizeof(int), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h->d_xf, xf.data(), xf.size() * sizeof(float4), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h->d_cxy, xy->coeffs_xy, ncxy * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess &&
         (rows32.empty() ||
          (cudaMemcpy(h->d_poly, rows32.data(), rows32.size() * sizeof(float4), cudaMemcpyHostToDevice) == cudaSuccess &&
           cudaMemcpy(h->d_polyd, rows64.data(), rows64.size() * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess));
    if (!ok) {
        const cudaError_t e = cudaGetLastError();
        ants_destroy(h);
        return e == cudaErrorMemoryAllocation ? ANTS_ERR_NOMEM : ANTS_ERR_CUDA;
    }
    ModelDev &m = h->dev;
    m.sens = (const float4 *)h->d_sens;
    m.grp = (const int *)h->d_grp;
    m.xf = xy->xform ? (const float4 *)h->d_xf : nullptr;
    m.cxy = (const float *)h->d_cxy;
    m.poly = (const float4 *)h->d_poly;
    m.polyd = (const double *)h->d_polyd;
    m.lrf_kind = kind;
    m.nx = nx;
    m.ny = ny;
    m.n_planes = n_planes;
    m.u_lo = kx[0];
    m.su = (float)((double)nx / ((double)kx[1] - (double)kx[0]));
    m.v_lo = kx[2];
    m.sv = (float)((double)ny / ((double)kx[3] - (double)kx[2]));
    m.N = N;
    m.n_lrf = n_lrf;
    m.n_r = kind == 4 ? n_r : 0;
    m.n_z = 0;
    m.r_lo = r_lo;
    m.r_hi = r_hi;
    m.sc = (float)sc_r;
    m.of = (float)(-(double)r_lo * sc_r - 0.5);
    m.tmax = (float)n_r - 0.5f;
    m.z_lo = kind == 5 ? kx[4] : 0.f;
    m.z_hi = kind == 5 ? kx[5] : 1.f;
    m.scz = 0.f;
    m.passive = nullptr;
    m.signal_min = m.dist_max = std::nanf("");
    m.select = 0;
    *out = h;
    return ANTS_OK;
}

extern "C" int ants_lrf_create_xy(const float *sensor_xy, const float *gains, const float *knots, const float *coeffs,
                                  const ants_lrf_dims_t *dims, const ants_lrf_xy_t *xy, ants_lrf_t **out) {
    return create_xy_impl(sensor_xy, gains, knots, coeffs, dims, xy, out);
}

// groups by the rotation / reflection symmetry of the array, with the sensors' frames (R33)
extern "C" int ants_group_by_symmetry(const float *sensor_xy, int32_t n, int32_t n_fold, int32_t reflect, float tol,
                                      int32_t *group_out, float *xform_out, int32_t *n_groups_out) {
    if (!sensor_xy || !group_out || !n_groups_out || n < 1 || n_fold < 1 || !(tol >= 0.f) || !std::isfinite(tol))
        return ANTS_ERR_INVALID;
    for (int i = 0; i < 2 * n; ++i)
        if (!std::isfinite(sensor_xy[i])) return ANTS_ERR_INVALID;
    const double two_pi = 6.283185307179586476925286766559;
    std::vector<std::array<double, 4>> ops;       // Q row-major
    for (int mirror = 0; mirror <= (reflect ? 1 : 0); ++mirror)
        for (int k = 0; k < n_fold; ++k) {
            const double a = two_pi * k / n_fold, c = std::cos(a), s = std::sin(a);
            // R = [[c, -s], [s, c]];  R M with M = diag(1, -1) flips the second column
            ops.push_back(mirror ? std::array<double, 4>{c, s, s, -c} : std::array<double, 4>{c, -s, s, c});
        }
    for (int i = 0; i < n; ++i) group_out[i] = -1;
    int n_groups = 0;
    for (int ref = 0; ref < n; ++ref) {
        if (group_out[ref] >= 0) continue;
        const double px = sensor_xy[2 * ref], py = sensor_xy[2 * ref + 1];
        for (const auto &Q : ops) {
            const double ix = Q[0] * px + Q[1] * py, iy = Q[2] * px + Q[3] * py;
            for (int i = 0; i < n; ++i) {
                if (group_out[i] >= 0) continue;
                const double dx = (double)sensor_xy[2 * i] - ix, dy = (double)sensor_xy[2 * i + 1] - iy;
                if (std::sqrt(dx * dx + dy * dy) <= (double)tol) {
                    group_out[i] = n_groups;
                    if (xform_out) {          // T = Q^T
                        xform_out[4 * i] = (float)Q[0];
                        xform_out[4 * i + 1] = (float)Q[2];
                        xform_out[4 * i + 2] = (float)Q[1];
                        xform_out[4 * i + 3] = (float)Q[3];
                    }
                    break;
                }
            }
        }
        ++n_groups;
    }
    *n_groups_out = n_groups;
    return ANTS_OK;
}

extern "C" int ants_lrf_create(const float *sensor_xy, const float *gains, const float *knots,
                               const float *coeffs, const ants_lrf_dims_t *dims, ants_lrf_t **out) {
    return create_impl(sensor_xy, gains, nullptr, knots, coeffs, dims, out);
}

extern "C" int ants_lrf_create_grouped(const float *sensor_xy, const float *gains, const int32_t *group,
                                       const float *knots, const float *coeffs, const ants_lrf_dims_t *dims,
                                       ants_lrf_t **out) {
    if (out) *out = nullptr;
    if (!group) return ANTS_ERR_INVALID;
    return create_impl(sensor_xy, gains, group, knots, coeffs, dims, out);
}

extern "C" int32_t ants_lrf_n_sensors(const ants_lrf_t *lrf) { return lrf ? lrf->dev.N : 0; }

// groups by the distance from the sensor centre to the detector centre (R28)
extern "C" int ants_group_by_radius(const float *sensor_xy, int32_t n, float tol, int32_t *group_out,
                                    int32_t *n_groups_out) {
    if (!sensor_xy || !group_out || !n_groups_out || n < 1 || !(tol >= 0.f) || !std::isfinite(tol)) return ANTS_ERR_INVALID;
    std::vector<std::pair<double, int>> order;
    try { order.reserve(n); } catch (const std::bad_alloc &) { return ANTS_ERR_NOMEM; }
    for (int i = 0; i < n; ++i) {
        const double x = sensor_xy[2 * i], y = sensor_xy[2 * i + 1];
        if (!std::isfinite(x) || !std::isfinite(y)) return ANTS_ERR_INVALID;
        order.emplace_back(std::sqrt(x * x + y * y), i);
    }
    std::stable_sort(order.begin(), order.end(),
                     [](const std::pair<double, int> &a, const std::pair<double, int> &b) { return a.first < b.first; });
    int current = -1;
    double anchor = -INFINITY;
    for (const auto &o : order) {
        if (o.first - anchor > (double)tol) { ++current; anchor = o.first; }
        group_out[o.second] = current;
    }
    *n_groups_out = current + 1;
    return ANTS_OK;
}

// relative gains carried on at the scale of the previous set (R29)
extern "C" int ants_gains_renormalise(const float *gains_new, const float *gains_prev, int32_t n, float *gains_out) {
    if (!gains_new || !gains_prev || !gains_out || n < 1) return ANTS_ERR_INVALID;
    double sum_prev = 0.0, sum_set = 0.0;
    for (int i = 0; i < n; ++i) {
        if (!(gains_prev[i] > 0.f) || !std::isfinite(gains_prev[i])) return ANTS_ERR_INVALID;
        const bool usable = gains_new[i] > 0.f && std::isfinite(gains_new[i]);
        sum_prev += (double)gains_prev[i];
        sum_set += (double)(usable ? gains_new[i] : gains_prev[i]);
    }
    const double scale = sum_prev / sum_set;     // mean(prev) / mean(set): the counts cancel
    for (int i = 0; i < n; ++i) {
        const bool usable = gains_new[i] > 0.f && std::isfinite(gains_new[i]);
        gains_out[i] = (float)((double)(usable ? gains_new[i] : gains_prev[i]) * scale);
    }
    return ANTS_OK;
}

extern "C" int ants_lrf_set_selection(ants_lrf_t *h, const uint8_t *passive, float signal_min, float dist_max) {
    if (!h) return ANTS_ERR_INVALID;
    ModelDev &m = h->dev;
    if (passive) {
        if (!h->d_passive && cudaMalloc(&h->d_passive, (size_t)m.N) != cudaSuccess) {
            cudaGetLastError();
            return ANTS_ERR_NOMEM;
        }
        std::vector<unsigned char> flags(m.N);
        for (int i = 0; i < m.N; ++i) flags[i] = passive[i] ? 1 : 0;
        if (cudaMemcpy(h->d_passive, flags.data(), (size_t)m.N, cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return ANTS_ERR_CUDA;
        }
        m.passive = (const unsigned char *)h->d_passive;
    } else {
        m.passive = nullptr;
    }
    m.signal_min = signal_min;
    m.dist_max = dist_max;
    m.select = (m.passive || !std::isnan(signal_min) || !std::isnan(dist_max)) ? 1 : 0;
    return ANTS_OK;
}

extern "C" void ants_destroy(ants_lrf_t *h) {
    if (!h) return;
    cudaFree(h->d_sens);
    cudaFree(h->d_poly);
    cudaFree(h->d_polyd);
    cudaFree(h->d_passive);
    cudaFree(h->d_ctr);
    cudaFree(h->d_grp);
    cudaFree(h->d_cxy);
    cudaFree(h->d_xf);
    if (h->slot_ev) {
        for (unsigned s = 0; s < kCtrSlots; ++s)
            if (h->slot_ev[s]) cudaEventDestroy(h->slot_ev[s]);
        delete[] h->slot_ev;
    }
    for (int s = 0; s < 3; ++s) {
        cudaFree(h->d_sig[s]);
        cudaFree(h->d_xyzA[s]);
        cudaFree(h->d_score[s]);
        if (h->streams[s]) cudaStreamDestroy(h->streams[s]);
    }
    cudaGetLastError();
    delete h;
}

extern "C" const char *ants_strerror(int status) {
    switch (status) {
        case ANTS_OK: return "ok";
        case ANTS_ERR_INVALID: return "invalid argument";
        case ANTS_ERR_UNSUPPORTED: return "unsupported combination or size";
        case ANTS_ERR_CUDA: return "CUDA runtime error";
        case ANTS_ERR_NOMEM: return "out of memory";
        case ANTS_ERR_SINGULAR: return "underdetermined fit (an interval without data)";
        default: return "unknown status";
    }
}

extern "C" int64_t ants_launch_count(void) { return g_launches.load(); }

// ---------------------------------------------------------------------------
// launch planning
// ---------------------------------------------------------------------------
// kernel look-ups: the instantiations live in k2d_pk_m*.cu, k2d_gen_m*.cu, k3d_m*.cu (kernels.h)
namespace ants {
const void *kernel_2d_pk_m0(int, int), *kernel_2d_pk_m1(int, int), *kernel_2d_pk_m2(int, int);
const void *kernel_gen_m0(int), *kernel_gen_m1(int), *kernel_gen_m2(int);
const void *kernel_3d_m0(int, int), *kernel_3d_m1(int, int);
const void *kernel_refine(int);
const void *kernel_3d_pk_m0(int, int, int), *kernel_3d_pk_m1(int, int, int);
const void *kernel_3d_pk(int method, int cpl, int gzp, int cross) {
    return method == 0 ? kernel_3d_pk_m0(cpl, gzp, cross) : method == 1 ? kernel_3d_pk_m1(cpl, gzp, cross) : nullptr;
}
const void *kernel_2d_pk(int method, int npt, int reuse) {
    return method == 0 ? kernel_2d_pk_m0(npt, reuse) : method == 1 ? kernel_2d_pk_m1(npt, reuse)
         : method == 2 ? kernel_2d_pk_m2(npt, reuse) : nullptr;
}
const void *kernel_gen(int method, int lrf_kind) {
    return method == 0 ? kernel_gen_m0(lrf_kind) : method == 1 ? kernel_gen_m1(lrf_kind) : method == 2 ? kernel_gen_m2(lrf_kind) : nullptr;
}
const void *kernel_3d(int method, int cpl, int gzm) {
    return method == 0 ? kernel_3d_m0(cpl, gzm) : method == 1 ? kernel_3d_m1(cpl, gzm) : nullptr;
}
}  // namespace ants

static const int kNpt2D[] = {1, 2, 3, 4, 8};
static const double kQSeries = 0.1;   // |dL/L0| bound under which the degree-6 log1p series is used

// tuning knobs, read once per process (experiments only; not needed in production)
static int env_knob(const char *name) {
    const char *e = std::getenv(name);
    return e ? std::atoi(e) : 0;
}
static int knob_warps_per_cta() { static const int v = env_knob("ANTS_WARPS_PER_CTA"); return v; }
static int env_knob_force_reuse() { static const int v = env_knob("ANTS_FORCE_NODE_REUSE"); return v; }
static int knob_no_reuse() { static const int v = env_knob("ANTS_NO_NODE_REUSE"); return v; }
static int knob_max_ctas_per_sm() { static const int v = env_knob("ANTS_MAX_CTAS_PER_SM"); return v; }
static int knob_no_cross() { static const int v = env_knob("ANTS_NO_CROSS_LEVEL"); return v; }

static int validate_grid(const ants_lrf *h, const ants_grid_params_t *g, int32_t method) {
    if (!h || !g) return ANTS_ERR_INVALID;
    if (method != ANTS_POISSON_ML && method != ANTS_CHI_SQUARE && method != ANTS_CHI_SQUARE_SUMRATIO) return ANTS_ERR_INVALID;
    if (g->dim != 2 && g->dim != 3) return ANTS_ERR_INVALID;
    if (g->nodes_per_axis < 2 || g->n_iter < 1 || g->n_iter > 4096) return ANTS_ERR_INVALID;
    if (!(g->factor > 0.f && g->factor < 1.f)) return ANTS_ERR_INVALID;
    if (!(g->step0_xy > 0.f) || !std::isfinite(g->step0_xy)) return ANTS_ERR_INVALID;
    if (g->seed_mode != 0 && g->seed_mode != 1) return ANTS_ERR_INVALID;
    const bool lrf3 = h->dev.n_z > 0 || h->dev.lrf_kind == 5;     // the LRF depends on z
    if (g->dim == 3) {
        if (!lrf3) return ANTS_ERR_INVALID;
        if (!(g->step0_z > 0.f) || !std::isfinite(g->step0_z)) return ANTS_ERR_INVALID;
    }
    if (lrf3 && !std::isnan(g->z_seed) && !std::isfinite(g->z_seed)) return ANTS_ERR_INVALID;
    return ANTS_OK;
}

// first iteration k whose grid is small enough for the differential score: every node within one knot interval
// of the centre (at most one knot crossed per axis); k_series (Poisson): the first of those on which
// |dL/L0| <= exp(max|dlnL/dr| reach) - 1 <= kQSeries, where log1p runs as a series (lg2(1 + q) before)
static void first_diff_iter(const ants_lrf *h, const ants_grid_params_t *g, int32_t method, int &k_diff, int &k_series) {
    k_diff = k_series = g->n_iter;
    if (!h->positive) return;
    const double half = 0.5 * (g->nodes_per_axis - 1);
    double hxy = g->step0_xy;
    for (int k = 0; k < g->n_iter; ++k, hxy *= (double)g->factor) {
        const double reach = std::sqrt(2.0) * half * hxy * 1.001;
        if (!(reach <= 0.9 * h->knot_r)) continue;
        // (tried in round 2: differential grids before the series is valid, with lg2(1 + q): most sensors then sit
        // on the general list with four MUFU per pair, slower than the plain form -- so both switch together)
        if (method != ANTS_POISSON_ML || std::expm1(h->max_dlog * reach) <= kQSeries) { k_diff = k_series = k; break; }
    }
}

// CTA shape: the warps-per-CTA in {8, 4, 2, 1} that lets the most warps share an SM's shared memory
// (each CTA carries its own copy of the model tables; 1 KB per CTA is reserved by the driver).
// ANTS_WARPS_PER_CTA in the environment overrides the choice.
static void pick_cta_shape(size_t tables, size_t per_warp, Plan &pl) {
    const size_t budget = 227 * 1024;
    int best = 1, best_total = 0;
    for (int wp : {8, 4, 2, 1}) {
        const size_t smem = tables + wp * per_warp;
        if (smem > budget) continue;
        int ctas = (int)std::min<size_t>(budget / (smem + 1024), (size_t)(64 / wp));
        ctas = std::min(ctas, 32);
        if (ctas * wp > best_total) { best_total = ctas * wp; best = wp; }
    }
    const int v = knob_warps_per_cta();
    if (v == 1 || v == 2 || v == 4 || v == 8) best = v;
    pl.warps = best;
    pl.smem = tables + best * per_warp;
}

// axial+z LRF: search over (x, y, z) or over (x, y) at fixed z
static int make_plan3d(const ants_lrf *h, const ants_grid_params_t *g, int32_t method, Plan &pl) {
    const ModelDev &m = h->dev;
    const int G = g->nodes_per_axis, Gz = g->dim == 3 ? G : 1;
    int cpl = 0, gzm = 1;
    if (g->dim == 3) {
        if (G > 8) return ANTS_ERR_UNSUPPORTED;           // 512 nodes
        cpl = G * G <= 32 ? 1 : 2;
        gzm = G <= 4 ? 4 : 8;
    } else {
        if (G * G > 256) return ANTS_ERR_UNSUPPORTED;
        const int need = (G * G + 31) / 32;
        for (int c : kNpt2D)
            if (c >= need) { cpl = c; break; }
    }
    // a 3-D search runs the kernel packed over pairs of z-levels; a 2-D search at fixed z the scalar one
    const bool packed = g->dim == 3;
    const int LP = (Gz + 1) / 2;
    if (packed) gzm = LP;                                 // the kernel is compiled for the grid's level pairs
    pl.family = packed ? 4 : 2;
    pl.cpl = cpl;
    pl.gzm = gzm;
    pl.npt = cpl * Gz;
    // an odd grid with two columns per lane packs its top level across the columns (recon3d_pk.cuh, CROSS)
    pl.cross = packed && cpl == 2 && (Gz & 1) && !knob_no_cross();
    pl.kernel = packed ? kernel_3d_pk(method, cpl, gzm, pl.cross) : kernel_3d(method, cpl, gzm);
    if (!pl.kernel) return ANTS_ERR_UNSUPPORTED;
    // differential from the first grid that stays within one knot interval of the centre (r and z);
    // Poisson log1p by series once |dL/L0| <= kQSeries on the whole grid
    pl.k_diff = pl.k_series = g->n_iter;
    if (h->positive) {
        const double half = 0.5 * (G - 1);
        double hxy = g->step0_xy, hz = g->dim == 3 ? g->step0_z : 0.0;
        for (int k = 0; k < g->n_iter; ++k, hxy *= (double)g->factor, hz *= (double)g->factor) {
            const double reach = std::sqrt(2.0) * half * hxy * 1.001, reach_z = half * hz * 1.001;
            const bool ok = reach <= 0.9 * h->knot_r && reach_z <= 0.9 * h->knot_z;
            if (ok && pl.k_diff == g->n_iter) pl.k_diff = k;
            if (ok && std::expm1(h->max_dlog * reach + h->max_dlog_z * reach_z) <= kQSeries) { pl.k_series = k; break; }
        }
        if (pl.k_series < pl.k_diff) pl.k_series = pl.k_diff;
    }
    const size_t tables = (size_t)(m.N + (m.n_z + 3) * (m.n_r + 1)) * 16;
    const size_t per_warp = packed ? warp_smem_bytes_3dpk(m.N, LP, m.n_r + 1, method) : warp_smem_bytes_3d(m.N, Gz, m.n_r + 1);
    pick_cta_shape(tables, per_warp, pl);
    if (pl.smem > 227 * 1024) return ANTS_ERR_UNSUPPORTED;
    return ANTS_OK;
}

// the general kernel: XY-type parameterisations, and axial LRFs that are not positive everywhere
static int make_plan_gen(const ants_lrf *h, const ants_grid_params_t *g, int32_t method, Plan &pl) {
    const ModelDev &m = h->dev;
    const int G = g->nodes_per_axis;
    const long long nodes = g->dim == 3 ? (long long)G * G * G : (long long)G * G;
    if (nodes > 65535) return ANTS_ERR_UNSUPPORTED;
    pl.family = 3;
    // CTA-wide event rounds: measured +15 % on the 19-sensor Composite config 8, nothing on configs 6 and 7 (64 and 37
    // sensors); ANTS_FORCE_NODE_REUSE=2 / ANTS_NO_NODE_REUSE=1 force it on / off for experiments
    pl.lockstep = (m.N <= 32 || env_knob_force_reuse() == 2) && !knob_no_reuse() ? 1 : 0;
    pl.npt = (int)((nodes + 31) / 32);
    pl.kernel = kernel_gen(method, m.lrf_kind);
    if (!pl.kernel) return ANTS_ERR_UNSUPPORTED;
    // FP64 scores from the first grid whose reach is a small fraction of a knot interval of every spline axis:
    // 0.225 for Poisson (with a contraction of 0.5, two iterations after the grids the packed kernels start to
    // score differentially), 0.1 for the chi-square forms, whose FP32 residual form keeps resolving neighbouring
    // nodes much longer.  Measured in round 2 on configs 6 and 8 (6,007 events each): with FP32 two iterations
    // beyond these switch points the oracle's best-to-second gap at a diverging node stays below 2.5e-5
    // (Poisson) and 6e-7 (chi-square, FP32 to the last iteration) against the 1e-4 the index rule allows.
    const double frac = method == ANTS_POISSON_ML ? 0.225 : 0.1;
    pl.k_diff = g->n_iter;
    const double half = 0.5 * (G - 1);
    double knot = std::fmin(h->knot_r > 0.0 ? h->knot_r : 1e300, h->knot_xy > 0.0 ? h->knot_xy : 1e300);
    const double plane = m.lrf_kind == 5 ? ((double)m.z_hi - (double)m.z_lo) / (m.n_planes - 1) : 1e300;
    double hxy = g->step0_xy, hz = g->dim == 3 ? g->step0_z : 0.0;
    for (int k = 0; k < g->n_iter; ++k, hxy *= (double)g->factor, hz *= (double)g->factor)
        if (std::sqrt(2.0) * half * hxy * 1.001 <= frac * knot && half * hz * 1.001 <= frac * plane) { pl.k_diff = k; break; }
    if (const char *e = std::getenv("ANTS_GEN_KFINE")) pl.k_diff = std::min(g->n_iter, std::max(0, std::atoi(e)));   // experiment knob
    pl.k_series = pl.k_diff;
    const int rows = (m.lrf_kind == 1 || m.lrf_kind == 4) ? m.n_lrf * (m.n_r + 1) : 0;
    const int ncxy = m.lrf_kind >= 3 ? m.n_lrf * std::max(m.n_planes, 1) * (m.nx + 3) * (m.ny + 3) : 0;
    // the double copy of the XY coefficients when the CTA's tables stay below 100 KB with it
    pl.gen_dtab = ncxy > 0 && cta_smem_bytes_gen(m.N, rows, ncxy, 1) <= 100 * 1024 ? 1 : 0;
    pick_cta_shape(cta_smem_bytes_gen(m.N, rows, ncxy, pl.gen_dtab), warp_smem_bytes_gen(m.N), pl);
    if (pl.smem > 227 * 1024) return ANTS_ERR_UNSUPPORTED;
    return ANTS_OK;
}

// host-only part of the plan (no CUDA call): kernel variant, score switch-over, shared-memory carve-up
static int make_plan(const ants_lrf *h, const ants_grid_params_t *g, int32_t method, Plan &pl) {
    int rc = validate_grid(h, g, method);
    if (rc != ANTS_OK) return rc;
    const ModelDev &m = h->dev;
    if (m.lrf_kind >= 3 || (m.lrf_kind == 1 && !h->positive)) return make_plan_gen(h, g, method, pl);
    if (m.n_z > 0) {
        if (method == ANTS_CHI_SQUARE_SUMRATIO) return ANTS_ERR_UNSUPPORTED;   // axial LRFs only (R27)
        return make_plan3d(h, g, method, pl);
    }
    const long long nodes = (long long)g->nodes_per_axis * g->nodes_per_axis;
    if (nodes > 256) return ANTS_ERR_UNSUPPORTED;
    int need = (int)((nodes + 31) / 32);
    pl.npt = 0;
    for (int c : kNpt2D)
        if (c >= need) { pl.npt = c; break; }
    if (!pl.npt) return ANTS_ERR_UNSUPPORTED;
    // strictly positive axial LRFs (the normal case): the sensor-pair-packed kernel
    pl.family = 0;
    // node reuse (recon2d_pk_kernel.cuh): contraction 1/2 and odd G; pl.reuse = 2 adds the CTA-wide event rounds
    // (LOCKSTEP).  Measured on every combination (profiles/r02_lockstep.md): node reuse alone gains on the Poisson kernel
    // with up to three nodes per lane and on large arrays (config 5 +20 %), and loses with four nodes per lane on smaller
    // arrays and in the least-squares kernels (instruction fetch); with the rounds it gains everywhere (config 3 +10 %,
    // config 2 +2 % on top of reuse) except on large Poisson arrays, where the events of a CTA differ in cost (the clamped
    // sensors are dropped per event) and the barrier makes the warps wait for the slowest (config 5 -4 %)
    const bool can = g->factor == 0.5f && (g->nodes_per_axis & 1);
    pl.reuse = method == ANTS_POISSON_ML && m.N >= 96 ? 1 : 2;
    if (!can || knob_no_reuse()) pl.reuse = 0;
    if (can && env_knob_force_reuse()) pl.reuse = method == ANTS_POISSON_ML ? env_knob_force_reuse() : 2;
    pl.lockstep = pl.reuse == 2;
    pl.kernel = kernel_2d_pk(method, pl.npt, pl.reuse);
    if (!pl.kernel) return ANTS_ERR_UNSUPPORTED;
    first_diff_iter(h, g, method, pl.k_diff, pl.k_series);
    const size_t tables = (cta_smem_bytes_pk(m.N, m.n_lrf * (m.n_r + 1), pl.npt) + 15) / 16 * 16;
    const size_t per_warp = warp_smem_bytes_pk(m.N, method, (int)nodes);
    pick_cta_shape(tables, per_warp, pl);
    if (pl.smem > 227 * 1024) return ANTS_ERR_UNSUPPORTED;
    return ANTS_OK;
}

// the cached plan of (grid, method): planned on first use; with `need_device` the kernel's shared-memory
// attribute is set and the resident CTAs per SM are asked from the runtime (once per plan)
static int get_plan(const ants_lrf *hc, const ants_grid_params_t *g, int32_t method, bool need_device, Plan &out) {
    if (!hc || !g) return ANTS_ERR_INVALID;
    ants_lrf *h = const_cast<ants_lrf *>(hc);
    const PlanKey key{g->dim, g->nodes_per_axis, g->n_iter, method, h->dev.select, g->step0_xy,
                      g->dim == 3 ? g->step0_z : 0.f, g->factor};
    std::lock_guard<std::mutex> lock(h->plan_mu);
    Plan *pl = nullptr;
    for (auto &kv : h->plans)
        if (kv.first == key) { pl = &kv.second; break; }
    if (!pl) {
        Plan fresh;
        int rc = make_plan(h, g, method, fresh);
        if (rc != ANTS_OK) return rc;
        if (h->plans.size() >= 64) h->plans.erase(h->plans.begin());
        h->plans.emplace_back(key, fresh);
        pl = &h->plans.back().second;
    } else {
        // grid values outside the key (seed mode, z seed) still need checking
        int rc = validate_grid(h, g, method);
        if (rc != ANTS_OK) return rc;
    }
    if (need_device && !pl->ready) {
        if (cudaFuncSetAttribute(pl->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem) != cudaSuccess) {
            cudaGetLastError();
            return ANTS_ERR_CUDA;
        }
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pl->kernel, pl->warps * 32, pl->smem) != cudaSuccess ||
            occ < 1) {
            cudaGetLastError();
            return ANTS_ERR_CUDA;
        }
        const int cap = knob_max_ctas_per_sm();       // tuning knob: fewer resident CTAs
        if (cap >= 1 && cap < occ) occ = cap;
        pl->ctas_per_sm = occ;
        pl->ready = true;
    }
    out = *pl;
    return ANTS_OK;
}

static void kernel_name(const Plan &pl, int32_t method, int lrf_kind, char *buf, size_t n) {
    if (pl.family == 0) std::snprintf(buf, n, "ants::recon2d_pk_kernel<%d,%d,%s%s>", pl.npt, (int)method, pl.reuse ? "true" : "false", pl.lockstep ? ",true" : "");
    else if (pl.family == 3) std::snprintf(buf, n, "ants::recon_gen_kernel<%d,%d>", (int)method, lrf_kind);
    else if (pl.family == 4)
        std::snprintf(buf, n, "ants::recon3d_pk_kernel<%d,%d,%d%s>", pl.cpl, pl.gzm, (int)method, pl.cross ? ",true" : "");
    else std::snprintf(buf, n, "ants::recon3d_kernel<%d,%d,%d>", pl.cpl, pl.gzm, (int)method);
}

extern "C" int ants_plan_info(const ants_lrf_t *lrf, const ants_grid_params_t *grid, int32_t method,
                              int32_t *first_diff, int32_t *nodes_per_lane, int32_t *warps_per_cta,
                              int32_t *ctas_per_sm, int32_t *smem_bytes) {
    Plan pl;
    int rc = get_plan(lrf, grid, method, true, pl);
    if (rc == ANTS_ERR_CUDA) rc = get_plan(lrf, grid, method, false, pl);
    if (rc != ANTS_OK) return rc;
    if (first_diff) *first_diff = pl.k_diff;
    if (nodes_per_lane) *nodes_per_lane = pl.npt;
    if (warps_per_cta) *warps_per_cta = pl.warps;
    if (ctas_per_sm) *ctas_per_sm = pl.ready ? pl.ctas_per_sm : 0;
    if (smem_bytes) *smem_bytes = (int32_t)pl.smem;
    return ANTS_OK;
}

extern "C" int ants_plan_kernel_name(const ants_lrf_t *lrf, const ants_grid_params_t *grid, int32_t method,
                                     char *name_out, int32_t name_cap) {
    if (!name_out || name_cap < 1) return ANTS_ERR_INVALID;
    Plan pl;
    int rc = get_plan(lrf, grid, method, false, pl);
    if (rc != ANTS_OK) return rc;
    kernel_name(pl, method, lrf->dev.lrf_kind, name_out, (size_t)name_cap);
    return ANTS_OK;
}

// ---------------------------------------------------------------------------
// dispatch: one kernel launch per call
// ---------------------------------------------------------------------------
static int launch(const ants_lrf *h, const float *signals, int64_t n_events, const ants_grid_params_t *g,
                  int32_t method, float *out_xyzA, float *out_score, uint16_t *out_path, cudaStream_t stream) {
    if (!h || !g) return ANTS_ERR_INVALID;
    if (n_events < 0) return ANTS_ERR_INVALID;
    if (n_events == 0) {
        Plan probe;
        return get_plan(h, g, method, false, probe);     // arguments are still checked
    }
    if (!signals || !out_xyzA || !out_score) {
        Plan probe;
        const int rc = get_plan(h, g, method, false, probe);
        return rc != ANTS_OK ? rc : ANTS_ERR_INVALID;
    }
    int dev_now = -1;
    if (cudaGetDevice(&dev_now) != cudaSuccess) { cudaGetLastError(); return ANTS_ERR_CUDA; }
    if (dev_now != h->device) return ANTS_ERR_INVALID;   // the model lives on the device it was created on
    Plan pl;
    int rc = get_plan(h, g, method, true, pl);
    if (rc != ANTS_OK) return rc;
    if (g->n_iter > 65535) return ANTS_ERR_INVALID;

    Params p{};
    p.m = h->dev;
    p.signals = signals;
    p.n_events = n_events;
    p.out_xyzA = out_xyzA;
    p.out_score = out_score;
    p.out_path = out_path;
    p.G = g->nodes_per_axis;
    p.K = g->n_iter;
    p.nodes = g->dim == 3 ? p.G * p.G * p.G : p.G * p.G;
    p.k_diff = pl.k_diff;
    p.k_series = pl.k_series;
    p.positive = h->positive ? 1 : 0;
    p.h0_xy = g->step0_xy;
    p.h0_z = g->dim == 3 ? g->step0_z : 0.f;
    p.factor = g->factor;
    p.z_seed = g->z_seed;
    p.dim = g->dim;
    p.seed_mode = g->seed_mode;
    p.warps_per_cta = pl.warps;
    p.tile_events = pl.warps;
    p.gen_dtab = pl.gen_dtab;
    p.reuse = pl.reuse;
    p.lockstep = pl.lockstep;

    long long want = (n_events + pl.warps - 1) / pl.warps;
    long long cap = (long long)h->sm_count * pl.ctas_per_sm;
    int grid = (int)std::min(want, cap);
    // counter slot: a launch that reuses a slot (1024 launches later) first waits, on the device, for the
    // slot's previous launch; the event recorded after this launch is what a later user waits for
    ants_lrf *hm = const_cast<ants_lrf *>(h);
    const unsigned ticket = hm->next_slot.fetch_add(1);
    const unsigned slot = ticket % kCtrSlots;
    if (ticket >= kCtrSlots && hm->slot_ev[slot] &&
        cudaStreamWaitEvent(stream, hm->slot_ev[slot], 0) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    p.ctr = h->d_ctr + 2 * slot;
    p.total_warps = grid * pl.warps;
    void *args[] = {&p};
    if (cudaLaunchKernel(pl.kernel, dim3(grid), dim3(pl.warps * 32), args, pl.smem, stream) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    if (!hm->slot_ev[slot] && cudaEventCreateWithFlags(&hm->slot_ev[slot], cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        hm->slot_ev[slot] = nullptr;
        cudaStreamSynchronize(stream);                  // no event to order a later user of the slot: drain now
    } else if (cudaEventRecord(hm->slot_ev[slot], stream) != cudaSuccess) {
        cudaGetLastError();
        cudaStreamSynchronize(stream);
    }
    g_launches.fetch_add(1);
    return ANTS_OK;
}

extern "C" int ants_reconstruct(const ants_lrf_t *lrf, const float *signals, int64_t n_events,
                                const ants_grid_params_t *grid, int32_t method, float *out_xyzA,
                                float *out_score, void *cuda_stream) {
    return launch(lrf, signals, n_events, grid, method, out_xyzA, out_score, nullptr, (cudaStream_t)cuda_stream);
}

extern "C" int ants_reconstruct_trace(const ants_lrf_t *lrf, const float *signals, int64_t n_events,
                                      const ants_grid_params_t *grid, int32_t method, float *out_xyzA,
                                      float *out_score, uint16_t *out_path, void *cuda_stream) {
    if (n_events > 0 && !out_path) return ANTS_ERR_INVALID;
    return launch(lrf, signals, n_events, grid, method, out_xyzA, out_score, out_path, (cudaStream_t)cuda_stream);
}

// ---------------------------------------------------------------------------
// host-buffer pipeline: chunks on a ring of three streams (H2D, kernel, D2H overlap)
// ---------------------------------------------------------------------------
static int ensure_scratch(ants_lrf *h, int64_t chunk) {
    if (h->scratch_events >= chunk) return ANTS_OK;
    const int N = h->dev.N;
    for (int s = 0; s < 3; ++s) {
        cudaFree(h->d_sig[s]);
        cudaFree(h->d_xyzA[s]);
        cudaFree(h->d_score[s]);
        h->d_sig[s] = h->d_xyzA[s] = h->d_score[s] = nullptr;
    }
    h->scratch_events = 0;
    for (int s = 0; s < 3; ++s) {
        if (!h->streams[s] && cudaStreamCreateWithFlags(&h->streams[s], cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError();
            return ANTS_ERR_CUDA;
        }
        if (cudaMalloc(&h->d_sig[s], (size_t)chunk * N * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&h->d_xyzA[s], (size_t)chunk * 4 * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&h->d_score[s], (size_t)chunk * sizeof(float)) != cudaSuccess) {
            cudaGetLastError();
            return ANTS_ERR_NOMEM;
        }
    }
    h->scratch_events = chunk;
    return ANTS_OK;
}

extern "C" int ants_reconstruct_host(const ants_lrf_t *lrf, const float *signals_host, int64_t n_events,
                                     const ants_grid_params_t *grid, int32_t method, float *out_xyzA_host,
                                     float *out_score_host, int64_t chunk_events) {
    Plan pl;
    int rc = get_plan(lrf, grid, method, false, pl);
    if (rc != ANTS_OK) return rc;
    if (n_events < 0) return ANTS_ERR_INVALID;
    if (n_events == 0) return ANTS_OK;
    if (!signals_host || !out_xyzA_host || !out_score_host) return ANTS_ERR_INVALID;
    ants_lrf *h = const_cast<ants_lrf *>(lrf);
    std::lock_guard<std::mutex> lock(h->host_mu);
    int64_t chunk = chunk_events > 0 ? chunk_events : (int64_t)1 << 20;
    chunk = std::min(chunk, n_events);
    rc = ensure_scratch(h, chunk);
    if (rc != ANTS_OK) return rc;
    const int N = h->dev.N;
    int slot = 0;
    for (int64_t a = 0; a < n_events && rc == ANTS_OK; a += chunk, slot = (slot + 1) % 3) {
        const int64_t n = std::min(chunk, n_events - a);
        cudaStream_t st = h->streams[slot];
        // the stream order makes the slot's buffers safe to reuse: the previous
        // occupant's D2H copy is ahead of this H2D copy on the same stream
        if (cudaMemcpyAsync(h->d_sig[slot], signals_host + a * N, (size_t)n * N * sizeof(float),
                            cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaGetLastError(); rc = ANTS_ERR_CUDA; break; }
        rc = launch(h, h->d_sig[slot], n, grid, method, h->d_xyzA[slot], h->d_score[slot], nullptr, st);
        if (rc != ANTS_OK) break;
        if (cudaMemcpyAsync(out_xyzA_host + a * 4, h->d_xyzA[slot], (size_t)n * 4 * sizeof(float),
                            cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaMemcpyAsync(out_score_host + a, h->d_score[slot], (size_t)n * sizeof(float),
                            cudaMemcpyDeviceToHost, st) != cudaSuccess) { cudaGetLastError(); rc = ANTS_ERR_CUDA; }
    }
    // also on an error: no copy that touches the caller's buffers may still be in flight on return
    for (int s = 0; s < 3; ++s)
        if (cudaStreamSynchronize(h->streams[s]) != cudaSuccess) { cudaGetLastError(); if (rc == ANTS_OK) rc = ANTS_ERR_CUDA; }
    return rc;
}

// ---------------------------------------------------------------------------
// continuous refinement (refine.cuh): one launch, FP64, lanes over sensors
// ---------------------------------------------------------------------------
extern "C" int ants_refine(const ants_lrf_t *lrf, const float *signals, int64_t n_events, int32_t method,
                           int32_t dim, int32_t seed_mode, int32_t n_steps, float *xyzA, float *score,
                           void *cuda_stream) {
    if (!lrf) return ANTS_ERR_INVALID;
    if (method != ANTS_POISSON_ML && method != ANTS_CHI_SQUARE && method != ANTS_CHI_SQUARE_SUMRATIO) return ANTS_ERR_INVALID;
    if ((dim != 2 && dim != 3) || (seed_mode != 0 && seed_mode != 1) || n_steps < 0 || n_steps > 10000 || n_events < 0)
        return ANTS_ERR_INVALID;
    const ModelDev &m = lrf->dev;
    const bool zdep = m.lrf_kind == 2 || m.lrf_kind == 5;
    if (dim == 3 && !zdep) return ANTS_ERR_INVALID;
    if (n_events == 0) return ANTS_OK;
    if (!signals || !xyzA || !score) return ANTS_ERR_INVALID;
    int dev_now = -1;
    if (cudaGetDevice(&dev_now) != cudaSuccess) { cudaGetLastError(); return ANTS_ERR_CUDA; }
    if (dev_now != lrf->device) return ANTS_ERR_INVALID;
    const void *kernel = kernel_refine(method);
    const int warps = 8;
    const int ncxy = m.lrf_kind >= 3 ? m.n_lrf * std::max(m.n_planes, 1) * (m.nx + 3) * (m.ny + 3) : 0;
    const int dtab = ncxy > 0 && cta_smem_bytes_gen(m.N, 0, ncxy, 1) <= 100 * 1024 ? 1 : 0;
    const size_t smem = cta_smem_bytes_gen(m.N, 0, ncxy, dtab) + (size_t)warps * ((size_t)m.N * 40 + 8);
    if (smem > 227 * 1024) return ANTS_ERR_UNSUPPORTED;
    int occ = 0;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, warps * 32, smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    RefineParams rp{};
    rp.m = m;
    rp.signals = signals;
    rp.n_events = n_events;
    rp.xyzA = xyzA;
    rp.score = score;
    rp.dim = dim;
    rp.seed_mode = seed_mode;
    rp.n_steps = n_steps;
    rp.dtab = dtab;
    const long long want = (n_events + warps - 1) / warps;
    const int grid = (int)std::min<long long>(want, (long long)lrf->sm_count * occ);
    void *args[] = {&rp};
    if (cudaLaunchKernel(kernel, dim3(grid), dim3(warps * 32), args, smem, (cudaStream_t)cuda_stream) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    g_launches.fetch_add(1);
    return ANTS_OK;
}

// ---------------------------------------------------------------------------
// scratch of the LRF-calculation calls: one device arena per process, grown on demand and kept, so that a call
// costs no cudaMalloc / cudaFree (round 1: four or five of each per call).  The calls are serialised by its mutex;
// each waits for its stream before it returns, so the next one may reuse the memory.
// ---------------------------------------------------------------------------
struct FitArena {
    std::mutex mu;
    unsigned char *buf = nullptr;
    size_t cap = 0, used = 0;
    int device = -1;
    // reset for a new call that needs `bytes` in total
    bool begin(size_t bytes) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return false; }
        bytes += 4096;
        if (dev != device || bytes > cap) {
            if (buf) { cudaSetDevice(device); cudaFree(buf); cudaSetDevice(dev); }
            buf = nullptr;
            cap = 0;
            const size_t want = std::max<size_t>(bytes, (size_t)1 << 20);
            if (cudaMalloc(&buf, want) != cudaSuccess) { cudaGetLastError(); buf = nullptr; return false; }
            cap = want;
            device = dev;
        }
        used = 0;
        return true;
    }
    template <typename T>
    T *take(size_t count) {
        used = (used + 255) / 256 * 256;
        T *ptr = reinterpret_cast<T *>(buf + used);
        used += count * sizeof(T);
        return used <= cap ? ptr : nullptr;
    }
};
static FitArena g_fit_arena;

// ---------------------------------------------------------------------------
// LRF calculation: normal equations on the GPU (lrf_fit.cuh), banded solve here
// ---------------------------------------------------------------------------
#include "lrf_fit.cuh"

// solve the symmetric positive definite system with half-bandwidth 3 stored as rows {d0, d1, d2, d3, rhs};
// returns false when a pivot is not positive (underdetermined table)
static bool solve_band3(const double *rows, int nc, double *x) {
    std::vector<double> L((size_t)nc * 4, 0.0);      // L[j][d] = L(j + d, j), d = 0..3 (banded Cholesky)
    for (int j = 0; j < nc; ++j) {
        for (int d = 0; d < 4 && j + d < nc; ++d) {
            double s = rows[(size_t)j * 5 + d];      // M(j + d, j)
            for (int k = std::max(0, j + d - 3); k < j; ++k) s -= L[(size_t)k * 4 + (j + d - k)] * L[(size_t)k * 4 + (j - k)];
            if (d == 0) {
                if (!(s > 0.0) || !std::isfinite(s)) return false;
                L[(size_t)j * 4] = std::sqrt(s);
            } else {
                L[(size_t)j * 4 + d] = s / L[(size_t)j * 4];
            }
        }
    }
    std::vector<double> y(nc);
    for (int i = 0; i < nc; ++i) {
        double s = rows[(size_t)i * 5 + 4];
        for (int k = std::max(0, i - 3); k < i; ++k) s -= L[(size_t)k * 4 + (i - k)] * y[k];
        y[i] = s / L[(size_t)i * 4];
    }
    for (int i = nc - 1; i >= 0; --i) {
        double s = y[i];
        for (int k = i + 1; k < std::min(nc, i + 4); ++k) s -= L[(size_t)i * 4 + (k - i)] * x[k];
        x[i] = s / L[(size_t)i * 4];
    }
    return true;
}

static int fit_axial_impl(const float *sensor_xy, const float *gains, const int32_t *group, const float *knots, int32_t N,
                          int32_t n_lrf, int32_t n_int, const float *signals, const float *xyzA,
                          int64_t n_events, float *coeffs_out, double *n_used_out, void *cuda_stream) {
    if (!sensor_xy || !knots || !coeffs_out || N < 1 || n_int < 1 || n_int > 4096 || n_events < 0) return ANTS_ERR_INVALID;
    if (group) {
        if (n_lrf < 1 || n_lrf > N) return ANTS_ERR_INVALID;
        for (int i = 0; i < N; ++i)
            if (group[i] < 0 || group[i] >= n_lrf) return ANTS_ERR_INVALID;
    } else if (n_lrf != 1 && n_lrf != N) {
        return ANTS_ERR_INVALID;
    }
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    const double lo = (double)knots[0], hi = (double)knots[1];
    if (!std::isfinite(lo) || !std::isfinite(hi) || !(lo >= 0.0) || !(hi > lo)) return ANTS_ERR_INVALID;
    for (int i = 0; i < N; ++i)
        if (gains && !(gains[i] > 0.f && std::isfinite(gains[i]))) return ANTS_ERR_INVALID;
    const int nc = n_int + 3;
    const size_t per_copy = (size_t)n_lrf * nc * 5;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    const int warps = 8;
    // shared profile: as many private copies per warp as fit in ~64 KB (fewer lanes per copy, less contention)
    int lane_split = 1;
    if (n_lrf == 1) {
        lane_split = 4;      // measured on B200: 4 is the best of 1..16 (more copies cost resident CTAs)
        while (lane_split > 1 && per_copy * warps * lane_split * sizeof(double) > 32 * 1024) lane_split >>= 1;
    }
    int *d_group = nullptr;
    if (const char *e = std::getenv("ANTS_FIT_LANE_SPLIT")) { const int v = std::atoi(e); if (v >= 1 && v <= 32 && n_lrf == 1) lane_split = v; }
    const int copies = n_lrf == 1 ? warps * lane_split : 1;
    const size_t smem = (per_copy * copies + (size_t)n_lrf) * sizeof(double);
    if (smem > 227 * 1024) return ANTS_ERR_UNSUPPORTED;

    std::vector<float> g(N, 1.f);
    if (gains) std::copy(gains, gains + N, g.begin());
    float *d_xy = nullptr, *d_g = nullptr;
    double *d_acc = nullptr;
    unsigned long long *d_used = nullptr;
    auto cleanup = [&]() { cudaGetLastError(); };
    std::lock_guard<std::mutex> arena_lock(g_fit_arena.mu);
    if (!g_fit_arena.begin((size_t)N * 16 + per_copy * sizeof(double) + (size_t)n_lrf * 8 + 2048)) return ANTS_ERR_NOMEM;
    d_xy = g_fit_arena.take<float>((size_t)N * 2);
    d_g = g_fit_arena.take<float>(N);
    if (group) d_group = g_fit_arena.take<int>(N);
    d_acc = g_fit_arena.take<double>(per_copy);
    d_used = g_fit_arena.take<unsigned long long>(n_lrf);
    if (!d_xy || !d_g || !d_acc || !d_used || (group && !d_group)) return ANTS_ERR_NOMEM;
    bool ok = cudaMemcpyAsync(d_xy, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(d_g, g.data(), (size_t)N * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              (!group || cudaMemcpyAsync(d_group, group, (size_t)N * sizeof(int), cudaMemcpyHostToDevice, st) == cudaSuccess) &&
              cudaMemsetAsync(d_acc, 0, per_copy * sizeof(double), st) == cudaSuccess &&
              cudaMemsetAsync(d_used, 0, (size_t)n_lrf * sizeof(unsigned long long), st) == cudaSuccess;
    // one shared profile whose band fits once per thread: the kernel without atomics in the loop
    const size_t per_thread = (size_t)nc * 5 * sizeof(double);
    int priv_threads = 0;
    if (n_lrf == 1 && !std::getenv("ANTS_FIT_ATOMIC")) {
        priv_threads = (int)std::min<size_t>(128, (113 * 1024 / per_thread) / 32 * 32);     // two CTAs per SM
        if (priv_threads < 64) priv_threads = (int)std::min<size_t>(128, (226 * 1024 / per_thread) / 32 * 32);
        if (priv_threads < 32) priv_threads = 0;
    }
    // one table per sensor (no groups) on an array of up to 128 sensors whose tables fit in shared memory: a thread
    // owns a sensor (lrf_fit_owned_kernel), no atomics in the loop either
    const int own_threads = (N + 31) / 32 * 32;
    const bool owned = n_lrf == N && N > 1 && !group && N <= 128 && per_thread * own_threads <= 226 * 1024 &&
                       !std::getenv("ANTS_FIT_ATOMIC");
    if (ok && n_events > 0 && owned) {
        FitParams p{};
        p.sens_xy = d_xy; p.gains = d_g; p.group = nullptr; p.signals = signals; p.xyzA = xyzA; p.n_events = n_events;
        p.N = N; p.n_lrf = n_lrf; p.n_int = n_int; p.nc = nc;
        p.lo = lo; p.hi = hi; p.h = (hi - lo) / n_int;
        p.acc = d_acc; p.n_used = d_used; p.copies = own_threads; p.lane_split = 1;
        const size_t osmem = per_thread * own_threads;
        int occ = 0;
        ok = cudaFuncSetAttribute((const void *)lrf_fit_owned_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)osmem) == cudaSuccess &&
             cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_fit_owned_kernel, own_threads, osmem) == cudaSuccess && occ >= 1;
        if (ok) {
            const int grid = (int)std::min<long long>(n_events, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel((const void *)lrf_fit_owned_kernel, dim3(grid), dim3(own_threads), args, osmem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
    } else if (ok && n_events > 0 && priv_threads > 0) {
        FitParams p{};
        p.sens_xy = d_xy; p.gains = d_g; p.group = nullptr; p.signals = signals; p.xyzA = xyzA; p.n_events = n_events;
        p.N = N; p.n_lrf = 1; p.n_int = n_int; p.nc = nc;
        p.lo = lo; p.hi = hi; p.h = (hi - lo) / n_int;
        p.acc = d_acc; p.n_used = d_used; p.copies = priv_threads; p.lane_split = 1;
        const size_t psmem = per_thread * priv_threads;
        const int pw = priv_threads / 32;
        int occ = 0;
        ok = cudaFuncSetAttribute((const void *)lrf_fit_shared_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psmem) == cudaSuccess &&
             cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_fit_shared_kernel, priv_threads, psmem) == cudaSuccess && occ >= 1;
        if (ok) {
            const long long want = (n_events + pw - 1) / pw;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel((const void *)lrf_fit_shared_kernel, dim3(grid), dim3(priv_threads), args, psmem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
    } else if (ok && n_events > 0) {
        FitParams p{};
        p.sens_xy = d_xy; p.gains = d_g; p.group = d_group; p.signals = signals; p.xyzA = xyzA; p.n_events = n_events;
        p.N = N; p.n_lrf = n_lrf; p.n_int = n_int; p.nc = nc;
        p.lo = lo; p.hi = hi; p.h = (hi - lo) / n_int;
        p.acc = d_acc; p.n_used = d_used; p.copies = copies; p.lane_split = lane_split;
        ok = cudaFuncSetAttribute((const void *)lrf_fit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess;
        int occ = 0;
        ok = ok && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_fit_kernel, warps * 32, smem) == cudaSuccess && occ >= 1;
        if (ok) {
            const long long want = (n_events + warps - 1) / warps;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel((const void *)lrf_fit_kernel, dim3(grid), dim3(warps * 32), args, smem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
    }
    std::vector<double> acc(per_copy);
    std::vector<unsigned long long> used(n_lrf);
    ok = ok && cudaMemcpyAsync(acc.data(), d_acc, per_copy * sizeof(double), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaMemcpyAsync(used.data(), d_used, (size_t)n_lrf * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaStreamSynchronize(st) == cudaSuccess;
    cleanup();
    if (!ok) return ANTS_ERR_CUDA;
    std::vector<double> x(nc);
    for (int m = 0; m < n_lrf; ++m) {
        if (n_used_out) n_used_out[m] = (double)used[m];
        if (!solve_band3(acc.data() + (size_t)m * nc * 5, nc, x.data())) return ANTS_ERR_SINGULAR;
        for (int j = 0; j < nc; ++j) coeffs_out[(size_t)m * nc + j] = (float)x[j];
    }
    return ANTS_OK;
}

extern "C" int ants_lrf_fit_axial(const float *sensor_xy, const float *gains, const float *knots, int32_t N,
                                  int32_t n_lrf, int32_t n_int, const float *signals, const float *xyzA,
                                  int64_t n_events, float *coeffs_out, double *n_used_out, void *cuda_stream) {
    return fit_axial_impl(sensor_xy, gains, nullptr, knots, N, n_lrf, n_int, signals, xyzA, n_events, coeffs_out,
                          n_used_out, cuda_stream);
}

extern "C" int ants_lrf_fit_axial_grouped(const float *sensor_xy, const float *gains, const int32_t *group,
                                          const float *knots, int32_t N, int32_t n_groups, int32_t n_int,
                                          const float *signals, const float *xyzA, int64_t n_events,
                                          float *coeffs_out, double *n_used_out, void *cuda_stream) {
    if (!group) return ANTS_ERR_INVALID;
    return fit_axial_impl(sensor_xy, gains, group, knots, N, n_groups, n_int, signals, xyzA, n_events, coeffs_out,
                          n_used_out, cuda_stream);
}

extern "C" int ants_lrf_fit_gains(const float *sensor_xy, const float *knots, const float *coeffs, int32_t N,
                                  int32_t n_int, const float *signals, const float *xyzA, int64_t n_events,
                                  float *gains_out, double *n_used_out, void *cuda_stream) {
    if (!sensor_xy || !knots || !coeffs || !gains_out || N < 1 || n_int < 1 || n_int > 4096 || n_events < 0)
        return ANTS_ERR_INVALID;
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    if (N > 128) return ANTS_ERR_UNSUPPORTED;
    const double lo = (double)knots[0], hi = (double)knots[1];
    if (!std::isfinite(lo) || !std::isfinite(hi) || !(lo >= 0.0) || !(hi > lo)) return ANTS_ERR_INVALID;
    for (int j = 0; j < n_int + 3; ++j)
        if (!std::isfinite(coeffs[j])) return ANTS_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    float *d_xy = nullptr, *d_c = nullptr;
    double *d_acc = nullptr;
    unsigned long long *d_used = nullptr;
    auto cleanup = [&]() { cudaGetLastError(); };
    std::lock_guard<std::mutex> arena_lock(g_fit_arena.mu);
    if (!g_fit_arena.begin((size_t)N * 32 + (size_t)(n_int + 3) * 4 + 2048)) return ANTS_ERR_NOMEM;
    d_xy = g_fit_arena.take<float>((size_t)N * 2);
    d_c = g_fit_arena.take<float>(n_int + 3);
    d_acc = g_fit_arena.take<double>((size_t)N * 2);
    d_used = g_fit_arena.take<unsigned long long>(N);
    if (!d_xy || !d_c || !d_acc || !d_used) return ANTS_ERR_NOMEM;
    bool ok = cudaMemcpyAsync(d_xy, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(d_c, coeffs, (size_t)(n_int + 3) * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemsetAsync(d_acc, 0, (size_t)N * 2 * sizeof(double), st) == cudaSuccess &&
              cudaMemsetAsync(d_used, 0, (size_t)N * sizeof(unsigned long long), st) == cudaSuccess;
    if (ok && n_events > 0) {
        GainParams p{};
        p.sens_xy = d_xy; p.coeffs = d_c; p.signals = signals; p.xyzA = xyzA; p.n_events = n_events;
        p.N = N; p.n_int = n_int; p.lo = lo; p.hi = hi; p.h = (hi - lo) / n_int;
        p.acc = d_acc; p.n_used = d_used;
        const int warps = 8;
        const size_t smem = (size_t)(n_int + 3) * sizeof(double);
        int occ = 0;
        ok = cudaFuncSetAttribute((const void *)lrf_gain_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
             cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_gain_kernel, warps * 32, smem) == cudaSuccess && occ >= 1;
        if (ok) {
            const long long want = (n_events + warps - 1) / warps;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel((const void *)lrf_gain_kernel, dim3(grid), dim3(warps * 32), args, smem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
    }
    std::vector<double> acc((size_t)N * 2);
    std::vector<unsigned long long> used(N);
    ok = ok && cudaMemcpyAsync(acc.data(), d_acc, acc.size() * sizeof(double), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaMemcpyAsync(used.data(), d_used, used.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaStreamSynchronize(st) == cudaSuccess;
    cleanup();
    if (!ok) return ANTS_ERR_CUDA;
    for (int i = 0; i < N; ++i) {
        if (n_used_out) n_used_out[i] = (double)used[i];
        gains_out[i] = acc[2 * i + 1] > 0.0 ? (float)(acc[2 * i] / acc[2 * i + 1]) : std::nanf("");
    }
    return ANTS_OK;
}

// dense Cholesky solve (row-major symmetric positive definite M [n][n], overwritten), false if not PD
static bool solve_dense_spd(std::vector<double> &M, std::vector<double> &b, int n) {
    for (int j = 0; j < n; ++j) {
        double s = M[(size_t)j * n + j];
        for (int k = 0; k < j; ++k) s -= M[(size_t)j * n + k] * M[(size_t)j * n + k];
        if (!(s > 0.0) || !std::isfinite(s)) return false;
        const double d = std::sqrt(s);
        M[(size_t)j * n + j] = d;
        for (int i = j + 1; i < n; ++i) {
            double t = M[(size_t)i * n + j];
            for (int k = 0; k < j; ++k) t -= M[(size_t)i * n + k] * M[(size_t)j * n + k];
            M[(size_t)i * n + j] = t / d;
        }
    }
    for (int i = 0; i < n; ++i) {
        double s = b[i];
        for (int k = 0; k < i; ++k) s -= M[(size_t)i * n + k] * b[k];
        b[i] = s / M[(size_t)i * n + i];
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = b[i];
        for (int k = i + 1; k < n; ++k) s -= M[(size_t)k * n + i] * b[k];
        b[i] = s / M[(size_t)i * n + i];
    }
    return true;
}

extern "C" int ants_lrf_fit_axial_z(const float *sensor_xy, const float *gains, const float *knots, int32_t N,
                                    int32_t n_r, int32_t n_z, const float *signals, const float *xyzA,
                                    int64_t n_events, float *coeffs_out, double *n_used_out, void *cuda_stream) {
    if (!sensor_xy || !knots || !coeffs_out || N < 1 || n_r < 1 || n_z < 1 || n_events < 0) return ANTS_ERR_INVALID;
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    const double r_lo = knots[0], r_hi = knots[1], z_lo = knots[2], z_hi = knots[3];
    if (!std::isfinite(r_lo) || !std::isfinite(r_hi) || !(r_lo >= 0.0) || !(r_hi > r_lo) || !std::isfinite(z_lo) ||
        !std::isfinite(z_hi) || !(z_hi > z_lo))
        return ANTS_ERR_INVALID;
    for (int i = 0; i < N; ++i)
        if (gains && !(gains[i] > 0.f && std::isfinite(gains[i]))) return ANTS_ERR_INVALID;
    const int ncr = n_r + 3, nc = ncr * (n_z + 3);
    if (nc > 768) return ANTS_ERR_UNSUPPORTED;
    const size_t total = (size_t)nc * 29, smem = total * sizeof(double);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    std::vector<float> g(N, 1.f);
    if (gains) std::copy(gains, gains + N, g.begin());
    float *d_xy = nullptr, *d_g = nullptr;
    double *d_acc = nullptr;
    unsigned long long *d_used = nullptr;
    auto cleanup = [&]() { cudaGetLastError(); };
    std::lock_guard<std::mutex> arena_lock(g_fit_arena.mu);
    if (!g_fit_arena.begin((size_t)N * 12 + smem + 2048)) return ANTS_ERR_NOMEM;
    d_xy = g_fit_arena.take<float>((size_t)N * 2);
    d_g = g_fit_arena.take<float>(N);
    d_acc = g_fit_arena.take<double>(total);
    d_used = g_fit_arena.take<unsigned long long>(1);
    if (!d_xy || !d_g || !d_acc || !d_used) return ANTS_ERR_NOMEM;
    bool ok = cudaMemcpyAsync(d_xy, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(d_g, g.data(), (size_t)N * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemsetAsync(d_acc, 0, smem, st) == cudaSuccess &&
              cudaMemsetAsync(d_used, 0, sizeof(unsigned long long), st) == cudaSuccess;
    if (ok && n_events > 0) {
        FitRZParams p{};
        p.sens_xy = d_xy; p.gains = d_g; p.signals = signals; p.xyzA = xyzA; p.n_events = n_events;
        p.N = N; p.n_r = n_r; p.n_z = n_z; p.ncr = ncr; p.nc = nc;
        p.r_lo = r_lo; p.r_hi = r_hi; p.hr = (r_hi - r_lo) / n_r;
        p.z_lo = z_lo; p.z_hi = z_hi; p.hz = (z_hi - z_lo) / n_z;
        p.acc = d_acc; p.n_used = d_used;
        const int warps = 8;
        int occ = 0;
        // the per-event factorised kernel (r-part per warp, one expansion per event) unless told otherwise
        const bool factorised = !std::getenv("ANTS_FIT_ATOMIC") && smem + (size_t)warps * ncr * 5 * sizeof(double) <= 227 * 1024;
        const void *kern = factorised ? (const void *)lrf_fit_rz2_kernel : (const void *)lrf_fit_rz_kernel;
        const size_t ksmem = factorised ? smem + (size_t)warps * ncr * 5 * sizeof(double) : smem;
        ok = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ksmem) == cudaSuccess &&
             cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, warps * 32, ksmem) == cudaSuccess && occ >= 1;
        if (ok) {
            const long long want = (n_events + warps - 1) / warps;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel(kern, dim3(grid), dim3(warps * 32), args, ksmem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
    }
    std::vector<double> acc(total);
    unsigned long long used = 0;
    ok = ok && cudaMemcpyAsync(acc.data(), d_acc, smem, cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaMemcpyAsync(&used, d_used, sizeof(used), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaStreamSynchronize(st) == cudaSuccess;
    cleanup();
    if (!ok) return ANTS_ERR_CUDA;
    if (n_used_out) *n_used_out = (double)used;
    std::vector<double> M((size_t)nc * nc, 0.0), b(nc);
    for (int j1 = 0; j1 < nc; ++j1) {
        const int jr1 = j1 % ncr;
        b[j1] = acc[(size_t)j1 * 29 + 28];
        for (int dz = 0; dz < 4; ++dz)
            for (int dr = -3; dr <= 3; ++dr) {
                const int jr2 = jr1 + dr, j2 = j1 + dz * ncr + dr;
                if (jr2 < 0 || jr2 >= ncr || j2 >= nc || j2 < j1) continue;
                const double v = acc[(size_t)j1 * 29 + dz * 7 + dr + 3];
                M[(size_t)j1 * nc + j2] = v;
                M[(size_t)j2 * nc + j1] = v;
            }
    }
    if (!solve_dense_spd(M, b, nc)) return ANTS_ERR_SINGULAR;
    for (int j = 0; j < nc; ++j) coeffs_out[j] = (float)b[j];
    return ANTS_OK;
}

extern "C" int ants_filter_events(float *xyzA, const float *score, int64_t n_events, const ants_filter_t *f,
                                  int64_t *n_pass_out, void *cuda_stream) {
    if (!f || n_events < 0 || (n_events > 0 && (!xyzA || !score))) return ANTS_ERR_INVALID;
    if (n_pass_out) *n_pass_out = 0;
    if (n_events == 0) return ANTS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long *d_pass = nullptr;
    if (cudaMalloc(&d_pass, sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); return ANTS_ERR_NOMEM; }
    FilterParams p{xyzA, score, n_events, f->score_max, f->energy_min, f->energy_max, f->radius_max, d_pass};
    const int grid = (int)std::min<long long>((n_events + 255) / 256, 148LL * 8);
    void *args[] = {&p};
    bool ok = cudaMemsetAsync(d_pass, 0, sizeof(unsigned long long), st) == cudaSuccess &&
              cudaLaunchKernel((const void *)event_filter_kernel, dim3(grid), dim3(256), args, 0, st) == cudaSuccess;
    if (ok) g_launches.fetch_add(1);
    unsigned long long pass = 0;
    // the counter lives until the stream has passed this point: wait when a count is wanted, else free in stream order
    if (ok && n_pass_out) {
        ok = cudaMemcpyAsync(&pass, d_pass, sizeof(pass), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
             cudaStreamSynchronize(st) == cudaSuccess;
        *n_pass_out = (int64_t)pass;
        cudaFree(d_pass);
    } else {
        if (cudaFreeAsync(d_pass, st) != cudaSuccess) { cudaGetLastError(); cudaStreamSynchronize(st); cudaFree(d_pass); }
    }
    if (!ok) { cudaGetLastError(); return ANTS_ERR_CUDA; }
    return ANTS_OK;
}

// ---------------------------------------------------------------------------
// LRF calculation for XY tables / the XY component of a Composite LRF (R35): one launch and one dense
// Cholesky solve per table
// ---------------------------------------------------------------------------
extern "C" int ants_lrf_fit_xy(const float *sensor_xy, const float *gains, const int32_t *group, const float *xform,
                               const float *knots_xy, int32_t N, int32_t n_lrf, int32_t nx, int32_t ny,
                               const float *knots_ax, const float *coeffs_ax, int32_t n_int_r, const float *signals,
                               const float *xyzA, int64_t n_events, float *coeffs_out, double *n_used_out,
                               void *cuda_stream) {
    if (!sensor_xy || !knots_xy || !coeffs_out || N < 1 || nx < 1 || ny < 1 || n_events < 0) return ANTS_ERR_INVALID;
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    if (group) {
        if (n_lrf < 1 || n_lrf > N) return ANTS_ERR_INVALID;
        for (int i = 0; i < N; ++i)
            if (group[i] < 0 || group[i] >= n_lrf) return ANTS_ERR_INVALID;
    } else if (n_lrf != 1 && n_lrf != N) {
        return ANTS_ERR_INVALID;
    }
    const double u_lo = knots_xy[0], u_hi = knots_xy[1], v_lo = knots_xy[2], v_hi = knots_xy[3];
    if (!std::isfinite(u_lo) || !std::isfinite(u_hi) || !std::isfinite(v_lo) || !std::isfinite(v_hi) || !(u_hi > u_lo) ||
        !(v_hi > v_lo))
        return ANTS_ERR_INVALID;
    const bool composite = coeffs_ax != nullptr;
    double a_lo = 0.0, a_hi = 1.0;
    if (composite) {
        if (!knots_ax || n_int_r < 1 || n_int_r > 4096) return ANTS_ERR_INVALID;
        a_lo = knots_ax[0];
        a_hi = knots_ax[1];
        if (!std::isfinite(a_lo) || !std::isfinite(a_hi) || !(a_lo >= 0.0) || !(a_hi > a_lo)) return ANTS_ERR_INVALID;
    }
    for (int i = 0; i < N; ++i)
        if (gains && !(gains[i] > 0.f && std::isfinite(gains[i]))) return ANTS_ERR_INVALID;
    const int ncu = nx + 3, nc = ncu * (ny + 3);
    if (nc > 768) return ANTS_ERR_UNSUPPORTED;
    const size_t total = (size_t)nc * 29, smem = total * sizeof(double);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    const bool scaled = group != nullptr || n_lrf == 1;
    std::vector<float> g(N, 1.f);
    if (gains && scaled) std::copy(gains, gains + N, g.begin());
    float *d_xy = nullptr, *d_g = nullptr, *d_xf = nullptr, *d_ax = nullptr;
    int *d_mem = nullptr;
    double *d_acc = nullptr;
    unsigned long long *d_used = nullptr;
    auto cleanup = [&]() { cudaGetLastError(); };
    std::lock_guard<std::mutex> arena_lock(g_fit_arena.mu);
    if (!g_fit_arena.begin((size_t)N * 32 + smem + (size_t)(n_int_r + 3) * 4 + 4096)) return ANTS_ERR_NOMEM;
    d_xy = g_fit_arena.take<float>((size_t)N * 2);
    d_g = g_fit_arena.take<float>(N);
    d_mem = g_fit_arena.take<int>(N);
    d_acc = g_fit_arena.take<double>(total);
    d_used = g_fit_arena.take<unsigned long long>(1);
    if (xform) d_xf = g_fit_arena.take<float>((size_t)N * 4);
    if (composite) d_ax = g_fit_arena.take<float>(n_int_r + 3);
    if (!d_xy || !d_g || !d_mem || !d_acc || !d_used || (xform && !d_xf) || (composite && !d_ax)) return ANTS_ERR_NOMEM;
    bool ok = cudaMemcpyAsync(d_xy, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(d_g, g.data(), (size_t)N * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              (!xform || cudaMemcpyAsync(d_xf, xform, (size_t)N * 4 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess);
    const int warps = 8;
    int occ = 0;
    ok = ok && cudaFuncSetAttribute((const void *)lrf_fit_xy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
         cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_fit_xy_kernel, warps * 32, smem) == cudaSuccess && occ >= 1;
    int rc = ok ? ANTS_OK : ANTS_ERR_CUDA;
    std::vector<double> acc(total), M((size_t)nc * nc), b(nc);
    std::vector<int> members;
    for (int t = 0; t < n_lrf && rc == ANTS_OK; ++t) {
        members.clear();
        for (int i = 0; i < N; ++i)
            if ((group ? group[i] : (n_lrf == 1 ? 0 : i)) == t) members.push_back(i);
        unsigned long long used = 0;
        ok = cudaMemsetAsync(d_acc, 0, smem, st) == cudaSuccess && cudaMemsetAsync(d_used, 0, sizeof(unsigned long long), st) == cudaSuccess &&
             (members.empty() || cudaMemcpyAsync(d_mem, members.data(), members.size() * sizeof(int), cudaMemcpyHostToDevice, st) == cudaSuccess) &&
             (!composite || cudaMemcpyAsync(d_ax, coeffs_ax + (size_t)t * (n_int_r + 3), (size_t)(n_int_r + 3) * sizeof(float),
                                            cudaMemcpyHostToDevice, st) == cudaSuccess);
        if (ok && n_events > 0 && !members.empty()) {
            FitXYParams p{};
            p.sens_xy = d_xy; p.gains = d_g; p.xform = xform ? d_xf : nullptr; p.members = d_mem; p.n_members = (int)members.size();
            p.signals = signals; p.xyzA = xyzA; p.n_events = n_events; p.N = N; p.nx = nx; p.ny = ny; p.ncu = ncu; p.nc = nc;
            p.u_lo = u_lo; p.u_hi = u_hi; p.hu = (u_hi - u_lo) / nx; p.v_lo = v_lo; p.v_hi = v_hi; p.hv = (v_hi - v_lo) / ny;
            p.axial = composite ? d_ax : nullptr; p.a_n = n_int_r; p.a_lo = a_lo; p.a_hi = a_hi;
            p.acc = d_acc; p.n_used = d_used; p.slab = -1;
            const long long want = (n_events + warps - 1) / warps;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            void *args[] = {&p};
            ok = cudaLaunchKernel((const void *)lrf_fit_xy_kernel, dim3(grid), dim3(warps * 32), args, smem, st) == cudaSuccess;
            if (ok) g_launches.fetch_add(1);
        }
        // (the host buffers of this table are read by the stream: wait before they are reused for the next one)
        ok = ok && cudaMemcpyAsync(acc.data(), d_acc, smem, cudaMemcpyDeviceToHost, st) == cudaSuccess &&
             cudaMemcpyAsync(&used, d_used, sizeof(used), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
             cudaStreamSynchronize(st) == cudaSuccess;
        if (!ok) { rc = ANTS_ERR_CUDA; break; }
        if (n_used_out) n_used_out[t] = (double)used;
        std::fill(M.begin(), M.end(), 0.0);
        for (int j1 = 0; j1 < nc; ++j1) {
            const int ju1 = j1 % ncu;
            b[j1] = acc[(size_t)j1 * 29 + 28];
            for (int dv = 0; dv < 4; ++dv)
                for (int du = -3; du <= 3; ++du) {
                    const int ju2 = ju1 + du, j2 = j1 + dv * ncu + du;
                    if (ju2 < 0 || ju2 >= ncu || j2 >= nc || j2 < j1) continue;
                    const double v = acc[(size_t)j1 * 29 + dv * 7 + du + 3];
                    M[(size_t)j1 * nc + j2] = v;
                    M[(size_t)j2 * nc + j1] = v;
                }
        }
        if (!solve_dense_spd(M, b, nc)) { rc = ANTS_ERR_SINGULAR; break; }
        for (int j = 0; j < nc; ++j) coeffs_out[(size_t)t * nc + j] = (float)b[j];
    }
    if (rc != ANTS_OK) cudaStreamSynchronize(st);
    cleanup();
    return rc;
}

// ---------------------------------------------------------------------------
// LRF calculation for Sliced tables (R36): all planes of a table jointly.  The normal matrix is block tridiagonal in
// the planes, every block banded like an XY table's; per table 3 (n_planes - 1) launches of lrf_fit_xy_kernel (one
// per slab and kind of block), one download, one banded Cholesky on the host.
// ---------------------------------------------------------------------------
// banded Cholesky solve: lower band storage B [n][bw + 1], B[i][bw - (i - j)] = M[i][j] for i - bw <= j <= i
static bool solve_banded_spd(std::vector<double> &B, std::vector<double> &b, int n, int bw) {
    const size_t ld = (size_t)bw + 1;
    for (int i = 0; i < n; ++i) {
        double *ri = &B[(size_t)i * ld];
        const int j0 = std::max(0, i - bw);
        for (int j = j0; j <= i; ++j) {
            const double *rj = &B[(size_t)j * ld];
            const int k0 = std::max(j0, j - bw);
            double s = ri[bw - (i - j)];
            const double *a = ri + (bw - (i - k0)), *c = rj + (bw - (j - k0));
            for (int k = 0; k < j - k0; ++k) s -= a[k] * c[k];
            if (j < i) {
                ri[bw - (i - j)] = s / rj[bw];
            } else {
                if (!(s > 0.0) || !std::isfinite(s)) return false;
                ri[bw] = std::sqrt(s);
            }
        }
    }
    for (int i = 0; i < n; ++i) {
        const double *ri = &B[(size_t)i * ld];
        const int j0 = std::max(0, i - bw);
        double s = b[i];
        for (int j = j0; j < i; ++j) s -= ri[bw - (i - j)] * b[j];
        b[i] = s / ri[bw];
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = b[i];
        const int j1 = std::min(n - 1, i + bw);
        for (int j = i + 1; j <= j1; ++j) s -= B[(size_t)j * ld + (bw - (j - i))] * b[j];
        b[i] = s / B[(size_t)i * ld + bw];
    }
    return true;
}

extern "C" int ants_lrf_fit_sliced(const float *sensor_xy, const float *gains, const int32_t *group, const float *xform,
                                   const float *knots_xy, int32_t N, int32_t n_lrf, int32_t nx, int32_t ny,
                                   int32_t n_planes, const float *signals, const float *xyzA, int64_t n_events,
                                   float *coeffs_out, double *n_used_out, void *cuda_stream) {
    if (!sensor_xy || !knots_xy || !coeffs_out || N < 1 || nx < 1 || ny < 1 || n_planes < 2 || n_events < 0)
        return ANTS_ERR_INVALID;
    if (n_events > 0 && (!signals || !xyzA)) return ANTS_ERR_INVALID;
    if (group) {
        if (n_lrf < 1 || n_lrf > N) return ANTS_ERR_INVALID;
        for (int i = 0; i < N; ++i)
            if (group[i] < 0 || group[i] >= n_lrf) return ANTS_ERR_INVALID;
    } else if (n_lrf != 1 && n_lrf != N) {
        return ANTS_ERR_INVALID;
    }
    const double u_lo = knots_xy[0], u_hi = knots_xy[1], v_lo = knots_xy[2], v_hi = knots_xy[3];
    const double z_lo = knots_xy[4], z_hi = knots_xy[5];
    for (int k = 0; k < 6; ++k)
        if (!std::isfinite(knots_xy[k])) return ANTS_ERR_INVALID;
    if (!(u_hi > u_lo) || !(v_hi > v_lo) || !(z_hi > z_lo)) return ANTS_ERR_INVALID;
    for (int i = 0; i < N; ++i)
        if (gains && !(gains[i] > 0.f && std::isfinite(gains[i]))) return ANTS_ERR_INVALID;
    const int ncu = nx + 3, nc = ncu * (ny + 3);
    const long long n_unknown = (long long)n_planes * nc;
    if (nc > 768 || n_unknown > 8192) return ANTS_ERR_UNSUPPORTED;
    const int n = (int)n_unknown, bw = nc + 3 * ncu + 3, n_slabs = n_planes - 1;
    const size_t block = (size_t)nc * 29, total = block * 3 * n_slabs, smem = block * sizeof(double);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return ANTS_ERR_CUDA;
    }
    const bool scaled = group != nullptr || n_lrf == 1;
    std::vector<float> g(N, 1.f);
    if (gains && scaled) std::copy(gains, gains + N, g.begin());
    std::lock_guard<std::mutex> arena_lock(g_fit_arena.mu);
    if (!g_fit_arena.begin((size_t)N * 32 + total * sizeof(double) + 4096)) return ANTS_ERR_NOMEM;
    float *d_xy = g_fit_arena.take<float>((size_t)N * 2);
    float *d_g = g_fit_arena.take<float>(N);
    int *d_mem = g_fit_arena.take<int>(N);
    double *d_acc = g_fit_arena.take<double>(total);
    unsigned long long *d_used = g_fit_arena.take<unsigned long long>(1);
    float *d_xf = xform ? g_fit_arena.take<float>((size_t)N * 4) : nullptr;
    if (!d_xy || !d_g || !d_mem || !d_acc || !d_used || (xform && !d_xf)) return ANTS_ERR_NOMEM;
    bool ok = cudaMemcpyAsync(d_xy, sensor_xy, (size_t)N * 2 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(d_g, g.data(), (size_t)N * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              (!xform || cudaMemcpyAsync(d_xf, xform, (size_t)N * 4 * sizeof(float), cudaMemcpyHostToDevice, st) == cudaSuccess);
    const int warps = 8;
    int occ = 0;
    ok = ok && cudaFuncSetAttribute((const void *)lrf_fit_xy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
         cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)lrf_fit_xy_kernel, warps * 32, smem) == cudaSuccess && occ >= 1;
    int rc = ok ? ANTS_OK : ANTS_ERR_CUDA;
    std::vector<double> acc(total), B, b(n);
    std::vector<int> members;
    for (int t = 0; t < n_lrf && rc == ANTS_OK; ++t) {
        members.clear();
        for (int i = 0; i < N; ++i)
            if ((group ? group[i] : (n_lrf == 1 ? 0 : i)) == t) members.push_back(i);
        unsigned long long used = 0;
        ok = cudaMemsetAsync(d_acc, 0, total * sizeof(double), st) == cudaSuccess &&
             cudaMemsetAsync(d_used, 0, sizeof(unsigned long long), st) == cudaSuccess &&
             (members.empty() || cudaMemcpyAsync(d_mem, members.data(), members.size() * sizeof(int), cudaMemcpyHostToDevice, st) == cudaSuccess);
        if (ok && n_events > 0 && !members.empty()) {
            FitXYParams p{};
            p.sens_xy = d_xy; p.gains = d_g; p.xform = xform ? d_xf : nullptr; p.members = d_mem; p.n_members = (int)members.size();
            p.signals = signals; p.xyzA = xyzA; p.n_events = n_events; p.N = N; p.nx = nx; p.ny = ny; p.ncu = ncu; p.nc = nc;
            p.u_lo = u_lo; p.u_hi = u_hi; p.hu = (u_hi - u_lo) / nx; p.v_lo = v_lo; p.v_hi = v_hi; p.hv = (v_hi - v_lo) / ny;
            p.axial = nullptr; p.n_used = d_used;
            p.n_planes = n_planes; p.z_lo = z_lo; p.z_hi = z_hi; p.dz = (z_hi - z_lo) / (n_planes - 1);
            const long long want = (n_events + warps - 1) / warps;
            const int grid = (int)std::min<long long>(want, (long long)sms * occ);
            for (int s = 0; s < n_slabs && ok; ++s)
                for (int part = 0; part < 3 && ok; ++part) {
                    p.slab = s; p.part = part; p.acc = d_acc + (size_t)(3 * s + part) * block;
                    void *args[] = {&p};
                    ok = cudaLaunchKernel((const void *)lrf_fit_xy_kernel, dim3(grid), dim3(warps * 32), args, smem, st) == cudaSuccess;
                    if (ok) g_launches.fetch_add(1);
                }
        }
        ok = ok && cudaMemcpyAsync(acc.data(), d_acc, total * sizeof(double), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
             cudaMemcpyAsync(&used, d_used, sizeof(used), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
             cudaStreamSynchronize(st) == cudaSuccess;
        if (!ok) { rc = ANTS_ERR_CUDA; break; }
        if (n_used_out) n_used_out[t] = (double)used;
        // assemble the lower band: rows/columns ordered plane by plane
        const size_t ld = (size_t)bw + 1;
        B.assign((size_t)n * ld, 0.0);
        std::fill(b.begin(), b.end(), 0.0);
        auto at = [&](int i, int j) -> double & { return i >= j ? B[(size_t)i * ld + (bw - (i - j))] : B[(size_t)j * ld + (bw - (j - i))]; };
        auto band = [&](const double *blk, int j1, int dv, int du, int &j2) -> const double * {
            const int ju2 = j1 % ncu + du;
            j2 = j1 + dv * ncu + du;
            if (ju2 < 0 || ju2 >= ncu || j2 >= nc || j2 < j1) return nullptr;
            return blk + (size_t)j1 * 29 + dv * 7 + du + 3;
        };
        for (int s = 0; s < n_slabs; ++s) {
            const double *b0 = &acc[(size_t)(3 * s) * block], *b1 = b0 + block, *b2 = b1 + block;
            const int o0 = s * nc, o1 = (s + 1) * nc;
            for (int j1 = 0; j1 < nc; ++j1) {
                b[o0 + j1] += b0[(size_t)j1 * 29 + 28];
                b[o1 + j1] += b1[(size_t)j1 * 29 + 28];
                for (int dv = 0; dv < 4; ++dv)
                    for (int du = -3; du <= 3; ++du) {
                        int j2;
                        const double *v0 = band(b0, j1, dv, du, j2);
                        if (!v0) continue;
                        at(o0 + j2, o0 + j1) += *v0;                                   // plane s with itself
                        at(o1 + j2, o1 + j1) += *band(b1, j1, dv, du, j2);             // plane s + 1 with itself
                        const double x = *band(b2, j1, dv, du, j2);                    // plane s with plane s + 1
                        at(o1 + j2, o0 + j1) += x;
                        if (j2 != j1) at(o1 + j1, o0 + j2) += x;
                    }
            }
        }
        if (!solve_banded_spd(B, b, n, bw)) { rc = ANTS_ERR_SINGULAR; break; }
        for (int j = 0; j < n; ++j) coeffs_out[(size_t)t * n + j] = (float)b[j];
    }
    if (rc != ANTS_OK) cudaStreamSynchronize(st);
    cudaGetLastError();
    return rc;
}
