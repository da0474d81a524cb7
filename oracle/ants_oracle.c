/*
 * ants_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * A plain, slow, double-precision restatement of the statistical event
 * reconstruction by contracting grids of the ANTS2 paper
 * (/root/reference/PAPER.md, arXiv:1602.07247).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or
 * constant with the CUDA path under paper_1602_07247_b200/csrc/.
 *
 * What it computes, in the paper's order (section 5.1.2.2):
 *   "For each event, a regular grid of nodes is defined, centered at the start
 *    search position. ... For each node, the algorithm evaluates the difference
 *    between the measured photosensor signals and the corresponding expected
 *    signal values given by the LRFs assuming that the light was emitted from
 *    this node.  The position resulting in the best match is selected and used
 *    as the center of a finer grid with the same number of nodes.  The
 *    procedure is repeated for the preconfigured number of iterations. ...
 *    The event energy is evaluated at each node as the ratio of two sums over
 *    all photosensors: the sum of the photosensor signals and that of the LRF
 *    values."
 * Start position = centroid (section 5.1.1).  Match = Maximum
 * Likelihood or Least Squares (section 5.1.2).  LRF = cubic
 * B-spline of the distance to the sensor axis, optionally times a Z
 * dependence (sections 6, 6.1.1, 6.1.2), shared
 * between sensors up to a relative gain (section 6.2).
 *
 * Readings of points on which the paper is silent are listed in DESIGN.md
 * ("Readings"); each is marked R<n> below.
 *
 * All arithmetic is IEEE double; inputs are the float32 arrays handed to the
 * CUDA library, widened; sums run left to right in sensor order; no blocking,
 * no fusion, no reordering.  OpenMP only splits the independent events.
 *
 * XY, Composite and Sliced parameterisations (R30-R33) are pinned in
 * tests/test_oracle_xy.py against scipy design matrices, plane/midplane values and
 * a numpy argmin.
 *
 * Pins (tests/test_oracle_pins.py): partition of unity, polynomial
 * reproduction by blossoming, scipy BSpline agreement, separable tensor
 * product, centroid special cases, energy vs 1-D minimisation, D >= 0 and
 * D = 0 iff mu = S, K=1 vs numpy argmin, lattice brute force, noise-free
 * recovery, mirror symmetry, power-of-two scaling; sensor selection (passive,
 * signal threshold, distance from start; tests/test_oracle_selection.py) against
 * the detector rebuilt without the ignored sensors.  The greedy search itself
 * (whether a noisy event reaches its global minimum) is a property of the
 * heuristic: "parity unpinned" beyond those pins.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n_sensors;       /* N */
    int32_t n_lrf;           /* 1: shared profile scaled by gains[i]; N: individual */
    int32_t lrf_dim;         /* LRF parameterisation (section 6.1): 1 Axial L(r); 2 Axial+Z L(r,z)
                                tensor product; 3 XY; 4 Composite = Axial + XY; 5 Sliced = XY LRFs on z planes */
    int32_t n_int_r;         /* uniform intervals in r, n_int_r+3 coefficients */
    int32_t n_int_z;         /* uniform intervals in z (0 if lrf_dim==1) */
    const float *sensor_xy;  /* [N][2] */
    const float *gains;      /* [N] */
    const float *knots;      /* {r_lo,r_hi[,z_lo,z_hi]} */
    const float *coeffs;     /* [n_lrf][n_int_z+3 or 1][n_int_r+3] */
    /* sensor selection (section 5.3 passive photosensors; section 5.1.2
     * "ignore photosensors with the signals below a certain threshold or situated further than a
     * given distance from the initial search position"); reading R19 in DESIGN.md */
    const uint8_t *passive;  /* [N] non-zero = passive, or NULL (none) */
    float signal_min;        /* sensors with S < signal_min are ignored; -inf (or NaN) = off */
    float dist_max;          /* sensors farther than this from the start position are ignored; +inf (NaN) = off */
    /* photosensor grouping (section 6.2: "assign a number of photosensors to a group and use
     * the same LRF for all photosensors within it ... a scaling parameter (relative gain) has to be assigned
     * to each of them"); reading R28.  NULL = no explicit grouping (n_lrf == 1 or n_lrf == N as above) */
    const int32_t *group;    /* [N] table index 0..n_lrf-1 of every sensor, or NULL */
    /* XY-type parameterisations (lrf_dim 3, 4, 5; "XY LRF", "Composite LRF",
     * PAPER.md:396 "Sliced LRF"); readings R30-R33 */
    int32_t n_int_x, n_int_y;  /* uniform intervals of the XY spline in the sensor-local coordinates (u, v) */
    int32_t n_planes;          /* Sliced: number of z planes (>= 2), uniformly spaced from z_lo to z_hi; else 0 */
    const float *knots_xy;     /* {u_lo, u_hi, v_lo, v_hi} and, for Sliced, {z_lo, z_hi} after them */
    const float *coeffs_xy;    /* [n_lrf][n_planes or 1][n_int_y+3][n_int_x+3], u fastest */
    const float *xform;        /* [N][4] or NULL: T_i row-major, (u, v) = T_i (p_xy - P_i) (R33: a sensor that a
                                  rotation/reflection of the array maps onto its group's reference sensor sees the
                                  reference LRF in a frame turned with it); NULL = identity */
} oracle_model_t;

typedef struct {
    int32_t dim;             /* 2 or 3 */
    int32_t nodes_per_axis;  /* G */
    float step0_xy, step0_z, factor;
    int32_t n_iter;          /* K */
    int32_t seed_mode;       /* 0 = centroid; 1 = position of the sensor with the strongest signal (R20) */
    float z_seed;            /* NaN => (z_lo+z_hi)/2 */
} oracle_grid_t;

/* ---- uniform cubic B-spline (R7: textbook basis, n+3 coefficients, no end
 * conditions; "B-splines [27]"; clamped argument R5) ---------- */
static void basis4(double u, double b[4])
{
    b[0] = (1.0 - u) * (1.0 - u) * (1.0 - u) / 6.0;
    b[1] = (3.0 * u * u * u - 6.0 * u * u + 4.0) / 6.0;
    b[2] = (-3.0 * u * u * u + 3.0 * u * u + 3.0 * u + 1.0) / 6.0;
    b[3] = u * u * u / 6.0;
}

/* interval index k and local coordinate u of x on [lo,hi] split in n intervals */
static void locate(double x, double lo, double hi, int n, int *k, double *u)
{
    double h = (hi - lo) / n;
    double xc = x < lo ? lo : (x > hi ? hi : x);
    double t = (xc - lo) / h;
    int kk = (int)floor(t);
    if (kk > n - 1) kk = n - 1;
    if (kk < 0) kk = 0;
    *k = kk;
    *u = t - kk;
}

double oracle_spline1(const float *c, int n, double lo, double hi, double x)
{
    int k; double u, b[4];
    locate(x, lo, hi, n, &k, &u);
    basis4(u, b);
    return (double)c[k] * b[0] + (double)c[k + 1] * b[1] + (double)c[k + 2] * b[2] + (double)c[k + 3] * b[3];
}

double oracle_spline2(const float *c, int nr, int nz, double r_lo, double r_hi,
                      double z_lo, double z_hi, double r, double z)
{
    int kr, kz; double ur, uz, br[4], bz[4], s = 0.0;
    locate(r, r_lo, r_hi, nr, &kr, &ur);
    locate(z, z_lo, z_hi, nz, &kz, &uz);
    basis4(ur, br);
    basis4(uz, bz);
    for (int b = 0; b < 4; ++b)
        for (int a = 0; a < 4; ++a)
            s += (double)c[(kz + b) * (nr + 3) + kr + a] * br[a] * bz[b];
    return s;
}

/* ---- LRF of sensor i at (x,y,z): L_i = g*_i s_m(i)(|p_xy - P_i|[, z])
 * (PAPER.md:388 axial; PAPER.md:394 axial+z; PAPER.md:400 shared profile +
 * relative gain; PAPER.md:402-406 sensor groups; PAPER.md:388-396 XY, Composite
 * and Sliced parameterisations) ---------------------------------------------- */
double oracle_lrf(const oracle_model_t *m, int i, double x, double y, double z)
{
    double dx = x - (double)m->sensor_xy[2 * i], dy = y - (double)m->sensor_xy[2 * i + 1];
    double r = sqrt(dx * dx + dy * dy);
    /* table and scale of sensor i: a group's profile times the sensor's relative gain;
     * one shared profile is the one-group case; a table of the sensor's own is not scaled */
    size_t tab = (size_t)(m->group ? m->group[i] : (m->n_lrf == 1 ? 0 : i));
    double g = (m->group || m->n_lrf == 1) ? (double)m->gains[i] : 1.0;
    double s = 0.0;
    if (m->lrf_dim == 1 || m->lrf_dim == 4) {           /* Axial, or the axial component of Composite */
        const float *c = m->coeffs + tab * (size_t)(m->n_int_r + 3);
        s += oracle_spline1(c, m->n_int_r, m->knots[0], m->knots[1], r);
    }
    if (m->lrf_dim == 2) {                              /* Axial+Z */
        const float *c = m->coeffs + tab * (size_t)((m->n_int_r + 3) * (m->n_int_z + 3));
        s += oracle_spline2(c, m->n_int_r, m->n_int_z, m->knots[0], m->knots[1], m->knots[2], m->knots[3], r, z);
    }
    if (m->lrf_dim >= 3) {
        /* R30: "LRF is a function of X and Y and no other type of symmetry can be assumed":
         * a tensor-product cubic B-spline of the position relative to the sensor, (u, v) = T_i (p_xy - P_i),
         * each coordinate clamped into the tabulated range like r (R5).
         * R31: "a sum of two components: an Axial LRF and an XY LRF".
         * R32: "a set of several XY LRFs, each defined on a specific Z plane.  The LRF values for the points
         * between the planes are calculated using linear interpolation of the LRF values at two closest
         * points from two closest planes": planes z_p = z_lo + p dz, p = 0 .. n_planes-1. */
        double u = dx, v = dy;
        if (m->xform) {
            const float *T = m->xform + 4 * i;
            u = (double)T[0] * dx + (double)T[1] * dy;
            v = (double)T[2] * dx + (double)T[3] * dy;
        }
        const float *kx = m->knots_xy;
        size_t per_plane = (size_t)(m->n_int_x + 3) * (size_t)(m->n_int_y + 3);
        if (m->lrf_dim == 5) {
            double z_lo = (double)kx[4], z_hi = (double)kx[5];
            double dz = (z_hi - z_lo) / (m->n_planes - 1);
            double zc = z < z_lo ? z_lo : (z > z_hi ? z_hi : z);
            int p = (int)floor((zc - z_lo) / dz);
            if (p > m->n_planes - 2) p = m->n_planes - 2;
            if (p < 0) p = 0;
            double w = (zc - (z_lo + p * dz)) / dz;
            const float *c0 = m->coeffs_xy + (tab * (size_t)m->n_planes + (size_t)p) * per_plane;
            double s0 = oracle_spline2(c0, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v);
            double s1 = oracle_spline2(c0 + per_plane, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v);
            s += (1.0 - w) * s0 + w * s1;
        } else {
            const float *c = m->coeffs_xy + tab * per_plane;
            s += oracle_spline2(c, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v);
        }
    }
    return g * s;
}

/* z range inside which a node is valid (R6), if the parameterisation depends on z: returns 1 and the range */
static int z_range(const oracle_model_t *m, double *z_lo, double *z_hi)
{
    if (m->lrf_dim == 2) { *z_lo = (double)m->knots[2]; *z_hi = (double)m->knots[3]; return 1; }
    if (m->lrf_dim == 5) { *z_lo = (double)m->knots_xy[4]; *z_hi = (double)m->knots_xy[5]; return 1; }
    return 0;
}

/* signals as the method sees them: Poisson ML clips negatives to 0 (R18) */
static void prepare_signals(const float *sig, int N, int method, double *S)
{
    for (int i = 0; i < N; ++i) {
        double s = (double)sig[i];
        S[i] = (method == 0 && s < 0.0) ? 0.0 : s;
    }
}

/* sensor i takes part in the centroid unless it is passive */
static int not_passive(const oracle_model_t *m, int i) { return !(m->passive && m->passive[i]); }

/* active[i] = 1 if sensor i takes part in the statistical reconstruction of this event (R19): not
 * passive, signal (as the method sees it) >= signal_min, axis within dist_max of the start position.
 * Returns the number of active sensors. */
static int select_sensors(const oracle_model_t *m, const double *S, const double *start_xy, uint8_t *active)
{
    int n = 0;
    for (int i = 0; i < m->n_sensors; ++i) {
        int a = not_passive(m, i);
        if (a && !isnan(m->signal_min) && S[i] < (double)m->signal_min) a = 0;
        if (a && !isnan(m->dist_max)) {
            double dx = start_xy[0] - (double)m->sensor_xy[2 * i], dy = start_xy[1] - (double)m->sensor_xy[2 * i + 1];
            if (sqrt(dx * dx + dy * dy) > (double)m->dist_max) a = 0;
        }
        active[i] = (uint8_t)a;
        n += a;
    }
    return n;
}

/* ---- centroid: x = sum X_i S_i/g_i / sum S_i/g_i ----------
 * returns 0 ok, 1 event unusable (non-finite signal, sum S <= 0 or sum S/g <= 0) */
int oracle_centroid(const oracle_model_t *m, const float *sig, int method, double *xy)
{
    int N = m->n_sensors;
    double *S = (double *)malloc(sizeof(double) * N);
    double sx = 0.0, sy = 0.0, sw = 0.0, ss = 0.0;
    int bad = 0;
    prepare_signals(sig, N, method, S);
    for (int i = 0; i < N; ++i) {
        if (!not_passive(m, i)) continue;             /* passive sensors are ignored altogether */
        if (!isfinite((double)sig[i])) bad = 1;       /* the raw signal: -inf must not be clipped away */
        double w = S[i] / (double)m->gains[i];
        sx += (double)m->sensor_xy[2 * i] * w;
        sy += (double)m->sensor_xy[2 * i + 1] * w;
        sw += w;
        ss += S[i];
    }
    free(S);
    if (bad || !(ss > 0.0) || !(sw > 0.0)) { xy[0] = xy[1] = NAN; return 1; }
    xy[0] = sx / sw;
    xy[1] = sy / sw;
    return 0;
}

/* ---- energy + score at one position (PAPER.md:328 energy = sum S / sum LRF;
 * PAPER.md:316 ML or LS).  S = prepared signals.  Returns 0 valid, 1 invalid
 * node (score = +inf, A = NaN).
 *   Poisson (R2): A = sum S / sum L, mu_i = A L_i,
 *       D = 2 sum_i t_i, t_i = mu_i - S_i - S_i ln(mu_i/S_i) (S_i>0), mu_i (S_i=0)
 *   chi-square (R3,R4): w_i = 1/max(S_i,1), A = sum w S L / sum w L^2,
 *       chi2 = sum w (S - A L)^2
 *   chi-square, sum-ratio energy (method 2, R27): A = sum S / sum L, same chi2   */
static int score_prepared(const oracle_model_t *m, const double *S, const uint8_t *active, int method,
                          double x, double y, double z, double *L, double *A_out, double *score_out)
{
#define ACTIVE(i) (!active || active[i])   /* sums run over the event's active sensors only (R19) */
    int N = m->n_sensors;
    double sumL = 0.0;
    *A_out = NAN;
    *score_out = INFINITY;
    double z_lo, z_hi;
    if (z_range(m, &z_lo, &z_hi) && !(z >= z_lo && z <= z_hi)) return 1; /* R6 */
    for (int i = 0; i < N; ++i) { if (!ACTIVE(i)) continue; L[i] = oracle_lrf(m, i, x, y, z); sumL += L[i]; }
    if (!(sumL > 0.0)) return 1;
    if (method == 0) {
        double sumS = 0.0, D = 0.0;
        for (int i = 0; i < N; ++i) if (ACTIVE(i)) sumS += S[i];
        double A = sumS / sumL;
        for (int i = 0; i < N; ++i) {
            if (!ACTIVE(i)) continue;
            double mu = A * L[i];
            if (S[i] > 0.0) {
                if (!(L[i] > 0.0)) return 1;
                D += mu - S[i] - S[i] * log(mu / S[i]);
            } else {
                D += mu;
            }
        }
        *A_out = A;
        *score_out = 2.0 * D;
    } else if (method == 2) {
        /* R27: least squares with the energy exactly as PAPER.md:328 states it for contracting grids,
         * "the ratio of two sums over all photosensors: the sum of the photosensor signals and that of
         * the LRF values": A = sum S / sum L, chi2 = sum w (S - A L)^2, w = 1/max(S,1) (R4) */
        double sumS = 0.0, chi2 = 0.0;
        for (int i = 0; i < N; ++i) if (ACTIVE(i)) sumS += S[i];
        double A = sumS / sumL;
        for (int i = 0; i < N; ++i) {
            if (!ACTIVE(i)) continue;
            double w = 1.0 / (S[i] > 1.0 ? S[i] : 1.0);
            double d = S[i] - A * L[i];
            chi2 += w * d * d;
        }
        *A_out = A;
        *score_out = chi2;
    } else {
        double swsl = 0.0, swll = 0.0, chi2 = 0.0;
        for (int i = 0; i < N; ++i) {
            if (!ACTIVE(i)) continue;
            double w = 1.0 / (S[i] > 1.0 ? S[i] : 1.0);
            swsl += w * S[i] * L[i];
            swll += w * L[i] * L[i];
        }
        if (!(swll > 0.0)) return 1;
        double A = swsl / swll;
        for (int i = 0; i < N; ++i) {
            if (!ACTIVE(i)) continue;
            double w = 1.0 / (S[i] > 1.0 ? S[i] : 1.0);
            double d = S[i] - A * L[i];
            chi2 += w * d * d;
        }
        *A_out = A;
        *score_out = chi2;
    }
    return 0;
#undef ACTIVE
}

/* ---- start search position ("the position reconstructed with the centroid method
 * or just the coordinates of the photosensor with the strongest signal").  R20: strongest = largest
 * signal as the method sees it among the non-passive sensors, first one on ties; the event is
 * unusable under the same conditions as for the centroid except that sum S/g is not needed.
 * returns 0 ok, 1 event unusable */
int oracle_start(const oracle_model_t *m, const float *sig, int method, int seed_mode, double *xy)
{
    if (seed_mode == 0) return oracle_centroid(m, sig, method, xy);
    int N = m->n_sensors, best = -1, bad = 0;
    double *S = (double *)malloc(sizeof(double) * (size_t)(unsigned)N);
    double ss = 0.0;
    prepare_signals(sig, N, method, S);
    for (int i = 0; i < N; ++i) {
        if (!not_passive(m, i)) continue;
        if (!isfinite((double)sig[i])) bad = 1;       /* the raw signal, before the clipping of R18 */
        ss += S[i];
        if (best < 0 || S[i] > S[best]) best = i;
    }
    free(S);
    if (bad || best < 0 || !(ss > 0.0)) { xy[0] = xy[1] = NAN; return 1; }
    xy[0] = (double)m->sensor_xy[2 * best];
    xy[1] = (double)m->sensor_xy[2 * best + 1];
    return 0;
}

/* needs_selection: any of the three selection options is on */
static int needs_selection(const oracle_model_t *m)
{
    return m->passive || !isnan(m->signal_min) || !isnan(m->dist_max);
}

int oracle_score_at(const oracle_model_t *m, const float *sig, int method, int seed_mode,
                    double x, double y, double z, double *A_out, double *score_out)
{
    int N = m->n_sensors;
    double *S = (double *)malloc(sizeof(double) * 2 * N);
    uint8_t *active = 0;
    prepare_signals(sig, N, method, S);
    if (needs_selection(m)) {           /* the event's active set hangs on its start position (R19) */
        double xy[2];
        active = (uint8_t *)malloc((size_t)(unsigned)N);
        if (oracle_start(m, sig, method, seed_mode, xy) || select_sensors(m, S, xy, active) == 0) {
            *A_out = NAN; *score_out = INFINITY;
            free(S); free(active);
            return 1;
        }
    }
    int rc = score_prepared(m, S, active, method, x, y, z, S + N, A_out, score_out);
    free(S);
    free(active);
    return rc;
}

/* fixed or start z (R10): z_seed, else mid-domain; 0 for purely axial LRFs */
static double start_z(const oracle_model_t *m, const oracle_grid_t *g)
{
    double z_lo, z_hi;
    if (!z_range(m, &z_lo, &z_hi)) return 0.0;
    if (isnan(g->z_seed)) return 0.5 * (z_lo + z_hi);
    return (double)g->z_seed;
}

/* ---- contracting grids for one event ---------------------- */
static void reconstruct_one(const oracle_model_t *m, const float *sig, const oracle_grid_t *g,
                            int method, double *xyzA, double *score,
                            int32_t *tr_idx, double *tr_best, double *tr_second,
                            double *S, double *L)
{
    int N = m->n_sensors, G = g->nodes_per_axis, K = g->n_iter;
    int Gz = g->dim == 3 ? G : 1;
    double c[3], xy[2];
    for (int k = 0; k < K; ++k) {
        if (tr_idx) tr_idx[k] = -1;
        if (tr_best) tr_best[k] = INFINITY;
        if (tr_second) tr_second[k] = INFINITY;
    }
    if (oracle_start(m, sig, method, g->seed_mode, xy)) {
        xyzA[0] = xyzA[1] = xyzA[2] = xyzA[3] = NAN;
        *score = INFINITY;
        return;
    }
    prepare_signals(sig, N, method, S);
    uint8_t *active = 0;
    if (needs_selection(m)) {
        active = (uint8_t *)malloc((size_t)(unsigned)N);
        double ssum = 0.0;
        int n_act = select_sensors(m, S, xy, active);
        for (int i = 0; i < N; ++i) if (active[i]) ssum += S[i];
        if (n_act == 0 || !(ssum > 0.0)) {              /* nothing left to reconstruct from */
            xyzA[0] = xyzA[1] = xyzA[2] = xyzA[3] = NAN;
            *score = INFINITY;
            free(active);
            return;
        }
    }
    c[0] = xy[0]; c[1] = xy[1]; c[2] = start_z(m, g);
    double h_xy = (double)g->step0_xy, h_z = (double)g->step0_z;   /* h_k = h_0 f^k (R1) */
    double half = 0.5 * (G - 1);
    for (int k = 0; k < K; ++k) {
        double best = INFINITY, second = INFINITY, bp[3] = { c[0], c[1], c[2] };
        int best_idx = -1;
        for (int iz = 0; iz < Gz; ++iz)
            for (int iy = 0; iy < G; ++iy)
                for (int ix = 0; ix < G; ++ix) {
                    double p[3] = { c[0] + (ix - half) * h_xy, c[1] + (iy - half) * h_xy,
                                    g->dim == 3 ? c[2] + (iz - half) * h_z : c[2] };
                    double A, sc;
                    if (score_prepared(m, S, active, method, p[0], p[1], p[2], L, &A, &sc)) continue;
                    if (sc < best) {               /* first strict minimum (R9) */
                        second = best;
                        best = sc; best_idx = (iz * G + iy) * G + ix;
                        bp[0] = p[0]; bp[1] = p[1]; bp[2] = p[2];
                    } else if (sc < second) {
                        second = sc;
                    }
                }
        if (tr_idx) tr_idx[k] = best_idx;
        if (tr_best) tr_best[k] = best;
        if (tr_second) tr_second[k] = second;
        c[0] = bp[0]; c[1] = bp[1]; c[2] = bp[2];      /* all invalid: keep centre */
        h_xy *= (double)g->factor;
        h_z *= (double)g->factor;
    }
    /* result = last best node, its energy and score (R11) */
    xyzA[0] = c[0]; xyzA[1] = c[1]; xyzA[2] = c[2];
    score_prepared(m, S, active, method, c[0], c[1], c[2], L, &xyzA[3], score);
    free(active);
}

/* threads a call with this n_threads argument uses */
int oracle_threads(int n_threads)
{
#ifdef _OPENMP
    return n_threads > 0 ? n_threads : omp_get_max_threads();
#else
    (void)n_threads;
    return 1;
#endif
}

/* signals [E][N] float32; out_xyzA [E][4], out_score [E] double; optional
 * traces [E][K].  n_threads <= 0: all cores.  Returns 0, or -1 on bad args. */
int oracle_reconstruct(const oracle_model_t *m, const float *signals, int64_t n_events,
                       const oracle_grid_t *g, int method, double *out_xyzA, double *out_score,
                       int32_t *tr_idx, double *tr_best, double *tr_second, int n_threads)
{
    if (!m || !g || !out_xyzA || !out_score || n_events < 0 || m->n_sensors < 1) return -1;
    if (g->nodes_per_axis < 2 || g->n_iter < 1 || !(g->factor > 0.0f && g->factor < 1.0f)) return -1;
    if (g->dim != 2 && g->dim != 3) return -1;
    if (g->seed_mode != 0 && g->seed_mode != 1) return -1;
    if (g->dim == 3 && m->lrf_dim != 2 && m->lrf_dim != 5) return -1;
    int N = m->n_sensors, K = g->n_iter;
#ifdef _OPENMP
#pragma omp parallel num_threads(oracle_threads(n_threads))
#endif
    {
        double *S = (double *)malloc(sizeof(double) * 2 * N);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t e = 0; e < n_events; ++e)
            reconstruct_one(m, signals + e * N, g, method, out_xyzA + 4 * e, out_score + e,
                            tr_idx ? tr_idx + e * K : 0, tr_best ? tr_best + e * K : 0,
                            tr_second ? tr_second + e * K : 0, S, S + N);
        free(S);
    }
    return 0;
}

/* score_at for many events: pos [E][3] double, A_out/score_out [E] (interface
 * helper for the parity tests; the arithmetic is oracle_score_at's). */
int oracle_score_at_many(const oracle_model_t *m, const float *signals, int64_t n_events, int method,
                         int seed_mode, const double *pos, double *A_out, double *score_out)
{
    if (!m || !signals || !pos || !A_out || !score_out || n_events < 0) return -1;
    for (int64_t e = 0; e < n_events; ++e)
        oracle_score_at(m, signals + e * m->n_sensors, method, seed_mode, pos[3 * e], pos[3 * e + 1], pos[3 * e + 2],
                        A_out + e, score_out + e);
    return 0;
}

/* =====================================================================================================
 * Continuous refinement of a reconstructed position (section 5.1.2: "The best match position is
 * found using either the algorithms provided in the Minuit2 minimization library ... or the contracting
 * grids method"; section 5.1.2.1: gradient-based minimisation "versus two (XY) or three
 * (XYZ) spatial coordinates", started from a given position).  Minuit2 itself is out of scope; reading R34
 * states the minimiser that takes its role here, started from a contracting-grid result:
 *
 *   objective F(p) = the node score of section 5.1.2.2 with the energy eliminated by its closed form
 *       (R2-R4, R27), over the event's active sensors (R19);
 *   model derivative m_i = d(A L_i)/dp = A dL_i/dp + L_i dA/dp, with dA/dp from the closed form
 *       (Poisson and method 2: A = sum S / sum L  ->  dA = -A sum dL / sum L;
 *        method 1: A = P/Q, P = sum w S L, Q = sum w L^2  ->  dA = (dP Q - P dQ)/Q^2);
 *   gradient g = 2 sum (1 - S_i/mu_i) m_i (Poisson), g = -2 sum w_i (S_i - mu_i) m_i (least squares);
 *   Gauss-Newton (Fisher) matrix H = 2 sum m_i m_i^T / mu_i (Poisson, terms with mu_i > 0),
 *       H = 2 sum w_i m_i m_i^T (least squares);
 *   Levenberg-Marquardt iteration with the damping update of Nielsen (Madsen, Nielsen, Tingleff, "Methods for
 *       non-linear least squares problems", 2004, algorithm 3.16), n_steps times: solve (H + lambda I) delta =
 *       -g; evaluate F, g, H at p + delta; gain ratio rho = (F - F_new) / (delta.(lambda delta - g) / 2);
 *       rho > 0: accept, lambda <- lambda max(1/3, 1 - (2 rho - 1)^3), nu <- 2; else keep p, lambda <-
 *       lambda nu, nu <- 2 nu.  lambda starts at 1e-3 max_a H_aa, nu at 2; a trial z outside the LRF's z range
 *       is moved to the nearest end of the range (projected step, delta taken as the projected one); a trial
 *       point that is invalid by the validity rules of the score, or a system without positive pivots, is a
 *       rejected step.
 * Spline derivatives are analytic (the B-spline basis differentiated); a clamped coordinate (R5) has zero
 * derivative; at r = 0 the radial direction is undefined and the axial gradient is taken as 0.
 * Pins (tests/test_oracle_refine.py): gradient against central differences of the pinned score; final point
 * against scipy.optimize.minimize on the same score from the same start; F never increases.
 * ===================================================================================================== */
static void dbasis4(double u, double d[4])
{
    d[0] = -(1.0 - u) * (1.0 - u) / 2.0;
    d[1] = (9.0 * u * u - 12.0 * u) / 6.0;
    d[2] = (-9.0 * u * u + 6.0 * u + 3.0) / 6.0;
    d[3] = u * u / 2.0;
}

/* value and derivative d/dx of the 1-D spline (0 outside [lo, hi], where the argument is clamped) */
static double spline1_d(const float *c, int n, double lo, double hi, double x, double *ds)
{
    int k; double u, b[4], d[4];
    locate(x, lo, hi, n, &k, &u);
    basis4(u, b);
    dbasis4(u, d);
    double h = (hi - lo) / n;
    *ds = (x < lo || x > hi) ? 0.0
        : ((double)c[k] * d[0] + (double)c[k + 1] * d[1] + (double)c[k + 2] * d[2] + (double)c[k + 3] * d[3]) / h;
    return (double)c[k] * b[0] + (double)c[k + 1] * b[1] + (double)c[k + 2] * b[2] + (double)c[k + 3] * b[3];
}

/* value and partial derivatives of the tensor-product spline c[nb+3][na+3] at (a, b) */
static double spline2_d(const float *c, int na, int nb, double a_lo, double a_hi, double b_lo, double b_hi,
                        double a, double b, double *d_a, double *d_b)
{
    int ka, kb; double ua, ub, ba[4], bb[4], da[4], db[4], s = 0.0, sa = 0.0, sb = 0.0;
    locate(a, a_lo, a_hi, na, &ka, &ua);
    locate(b, b_lo, b_hi, nb, &kb, &ub);
    basis4(ua, ba); basis4(ub, bb);
    dbasis4(ua, da); dbasis4(ub, db);
    for (int j = 0; j < 4; ++j)
        for (int i = 0; i < 4; ++i) {
            double cc = (double)c[(kb + j) * (na + 3) + ka + i];
            s += cc * ba[i] * bb[j];
            sa += cc * da[i] * bb[j];
            sb += cc * ba[i] * db[j];
        }
    *d_a = (a < a_lo || a > a_hi) ? 0.0 : sa / ((a_hi - a_lo) / na);
    *d_b = (b < b_lo || b > b_hi) ? 0.0 : sb / ((b_hi - b_lo) / nb);
    return s;
}

/* L_i(p) and its gradient with respect to (x, y, z) */
double oracle_lrf_grad(const oracle_model_t *m, int i, double x, double y, double z, double grad[3])
{
    double dx = x - (double)m->sensor_xy[2 * i], dy = y - (double)m->sensor_xy[2 * i + 1];
    double r = sqrt(dx * dx + dy * dy);
    double ex = r > 0.0 ? dx / r : 0.0, ey = r > 0.0 ? dy / r : 0.0;     /* dr/dx, dr/dy */
    size_t tab = (size_t)(m->group ? m->group[i] : (m->n_lrf == 1 ? 0 : i));
    double g = (m->group || m->n_lrf == 1) ? (double)m->gains[i] : 1.0;
    double s = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    if (m->lrf_dim == 1 || m->lrf_dim == 4) {
        double ds;
        s += spline1_d(m->coeffs + tab * (size_t)(m->n_int_r + 3), m->n_int_r, m->knots[0], m->knots[1], r, &ds);
        gx += ds * ex; gy += ds * ey;
    }
    if (m->lrf_dim == 2) {
        double dr, dz;
        s += spline2_d(m->coeffs + tab * (size_t)((m->n_int_r + 3) * (m->n_int_z + 3)), m->n_int_r, m->n_int_z,
                       m->knots[0], m->knots[1], m->knots[2], m->knots[3], r, z, &dr, &dz);
        gx += dr * ex; gy += dr * ey; gz += dz;
    }
    if (m->lrf_dim >= 3) {
        double T[4] = { 1.0, 0.0, 0.0, 1.0 };
        if (m->xform) for (int j = 0; j < 4; ++j) T[j] = (double)m->xform[4 * i + j];
        double u = T[0] * dx + T[1] * dy, v = T[2] * dx + T[3] * dy;
        const float *kx = m->knots_xy;
        size_t per_plane = (size_t)(m->n_int_x + 3) * (size_t)(m->n_int_y + 3);
        double su, sv, val;
        if (m->lrf_dim == 5) {
            double z_lo = (double)kx[4], z_hi = (double)kx[5];
            double dzp = (z_hi - z_lo) / (m->n_planes - 1);
            double zc = z < z_lo ? z_lo : (z > z_hi ? z_hi : z);
            int p = (int)floor((zc - z_lo) / dzp);
            if (p > m->n_planes - 2) p = m->n_planes - 2;
            if (p < 0) p = 0;
            double w = (zc - (z_lo + p * dzp)) / dzp;
            const float *c0 = m->coeffs_xy + (tab * (size_t)m->n_planes + (size_t)p) * per_plane;
            double su0, sv0, su1, sv1;
            double s0 = spline2_d(c0, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v, &su0, &sv0);
            double s1 = spline2_d(c0 + per_plane, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v, &su1, &sv1);
            val = (1.0 - w) * s0 + w * s1;
            su = (1.0 - w) * su0 + w * su1;
            sv = (1.0 - w) * sv0 + w * sv1;
            gz += (z < z_lo || z > z_hi) ? 0.0 : (s1 - s0) / dzp;
        } else {
            val = spline2_d(m->coeffs_xy + tab * per_plane, m->n_int_x, m->n_int_y, kx[0], kx[1], kx[2], kx[3], u, v, &su, &sv);
        }
        s += val;
        gx += su * T[0] + sv * T[2];          /* du/dx = T00, dv/dx = T10 */
        gy += su * T[1] + sv * T[3];
    }
    grad[0] = g * gx; grad[1] = g * gy; grad[2] = g * gz;
    return g * s;
}

/* F, A, g[3], H[3][3] at p over the active sensors; dim = 2: (x, y), 3: (x, y, z).  Returns 0 valid, 1 invalid. */
static int score_grad_prepared(const oracle_model_t *m, const double *S, const uint8_t *active, int method, int dim,
                               const double p[3], double *A_out, double *F_out, double g[3], double H[9])
{
    int N = m->n_sensors;
    double z_lo, z_hi;
    *A_out = NAN; *F_out = INFINITY;
    for (int a = 0; a < 3; ++a) g[a] = 0.0;
    for (int a = 0; a < 9; ++a) H[a] = 0.0;
    if (z_range(m, &z_lo, &z_hi) && !(p[2] >= z_lo && p[2] <= z_hi)) return 1;
    double *L = (double *)malloc(sizeof(double) * 4 * (size_t)N), *dL = L + N;     /* L[N], dL[N][3] */
    double sumL = 0.0, sumS = 0.0, sdL[3] = { 0, 0, 0 }, P = 0.0, Q = 0.0, dP[3] = { 0, 0, 0 }, dQ[3] = { 0, 0, 0 };
    for (int i = 0; i < N; ++i) {
        if (active && !active[i]) continue;
        L[i] = oracle_lrf_grad(m, i, p[0], p[1], p[2], dL + 3 * i);
        if (dim == 2) dL[3 * i + 2] = 0.0;
        double w = 1.0 / (S[i] > 1.0 ? S[i] : 1.0);
        sumL += L[i]; sumS += S[i];
        P += w * S[i] * L[i]; Q += w * L[i] * L[i];
        for (int a = 0; a < 3; ++a) {
            sdL[a] += dL[3 * i + a];
            dP[a] += w * S[i] * dL[3 * i + a];
            dQ[a] += 2.0 * w * L[i] * dL[3 * i + a];
        }
    }
    int bad = !(sumL > 0.0) || (method == 1 && !(Q > 0.0));
    double A = 0.0, dA[3] = { 0, 0, 0 }, F = 0.0;
    if (!bad) {
        if (method == 1) { A = P / Q; for (int a = 0; a < 3; ++a) dA[a] = (dP[a] * Q - P * dQ[a]) / (Q * Q); }
        else { A = sumS / sumL; for (int a = 0; a < 3; ++a) dA[a] = -A * sdL[a] / sumL; }
        for (int i = 0; i < N && !bad; ++i) {
            if (active && !active[i]) continue;
            double mu = A * L[i], mi[3];
            for (int a = 0; a < 3; ++a) mi[a] = A * dL[3 * i + a] + L[i] * dA[a];
            if (method == 0) {
                if (S[i] > 0.0) {
                    if (!(L[i] > 0.0)) { bad = 1; break; }
                    F += mu - S[i] - S[i] * log(mu / S[i]);
                } else {
                    F += mu;
                }
                if (mu > 0.0) {
                    double q = 1.0 - S[i] / mu;
                    for (int a = 0; a < 3; ++a) {
                        g[a] += 2.0 * q * mi[a];
                        for (int b = 0; b < 3; ++b) H[3 * a + b] += 2.0 * mi[a] * mi[b] / mu;
                    }
                }
            } else {
                double w = 1.0 / (S[i] > 1.0 ? S[i] : 1.0), d = S[i] - mu;
                F += w * d * d;
                for (int a = 0; a < 3; ++a) {
                    g[a] += -2.0 * w * d * mi[a];
                    for (int b = 0; b < 3; ++b) H[3 * a + b] += 2.0 * w * mi[a] * mi[b];
                }
            }
        }
        if (method == 0) F *= 2.0;
    }
    free(L);
    if (bad) return 1;
    *A_out = A; *F_out = F;
    return 0;
}

/* solve (H + lambda I) delta = -g for the leading dim x dim block by Gaussian elimination without
 * pivoting (the matrix is symmetric positive definite when the step is usable); returns 0 ok, 1 no step */
static int lm_step(const double H[9], const double g[3], double lambda, int dim, double delta[3])
{
    double M[3][4];
    for (int a = 0; a < dim; ++a) {
        for (int b = 0; b < dim; ++b) M[a][b] = H[3 * a + b];
        M[a][a] += lambda;
        M[a][dim] = -g[a];
    }
    for (int a = 0; a < dim; ++a) {
        if (!(M[a][a] > 0.0) || !isfinite(M[a][a])) return 1;
        for (int r = a + 1; r < dim; ++r) {
            double f = M[r][a] / M[a][a];
            for (int c = a; c <= dim; ++c) M[r][c] -= f * M[a][c];
        }
    }
    delta[0] = delta[1] = delta[2] = 0.0;
    for (int a = dim - 1; a >= 0; --a) {
        double s = M[a][dim];
        for (int c = a + 1; c < dim; ++c) s -= M[a][c] * delta[c];
        delta[a] = s / M[a][a];
    }
    for (int a = 0; a < dim; ++a) if (!isfinite(delta[a])) return 1;
    return 0;
}

/* gradient and Gauss-Newton matrix of one event at one position (for the pins) */
int oracle_score_grad(const oracle_model_t *m, const float *sig, int method, int seed_mode, int dim,
                      double x, double y, double z, double *A_out, double *F_out, double g[3], double H[9])
{
    int N = m->n_sensors;
    double *S = (double *)malloc(sizeof(double) * (size_t)N);
    uint8_t *active = 0;
    prepare_signals(sig, N, method, S);
    if (needs_selection(m)) {
        double xy[2];
        active = (uint8_t *)malloc((size_t)(unsigned)N);
        if (oracle_start(m, sig, method, seed_mode, xy) || select_sensors(m, S, xy, active) == 0) {
            free(S); free(active);
            *A_out = NAN; *F_out = INFINITY;
            return 1;
        }
    }
    double p[3] = { x, y, z };
    int rc = score_grad_prepared(m, S, active, method, dim, p, A_out, F_out, g, H);
    free(S); free(active);
    return rc;
}

static void refine_one(const oracle_model_t *m, const float *sig, int method, int seed_mode, int dim, int n_steps,
                       double *xyzA, double *score)
{
    int N = m->n_sensors;
    double xy0[2];
    if (!(isfinite(xyzA[0]) && isfinite(xyzA[1]) && isfinite(xyzA[2]))) return;       /* failed event: left as it is */
    if (oracle_start(m, sig, method, seed_mode, xy0)) { xyzA[0] = xyzA[1] = xyzA[2] = xyzA[3] = NAN; *score = INFINITY; return; }
    double *S = (double *)malloc(sizeof(double) * (size_t)N);
    uint8_t *active = 0;
    prepare_signals(sig, N, method, S);
    if (needs_selection(m)) {
        active = (uint8_t *)malloc((size_t)(unsigned)N);
        if (select_sensors(m, S, xy0, active) == 0) { free(S); free(active); xyzA[0] = xyzA[1] = xyzA[2] = xyzA[3] = NAN; *score = INFINITY; return; }
    }
    double p[3] = { xyzA[0], xyzA[1], xyzA[2] }, A, F, g[3], H[9];
    if (score_grad_prepared(m, S, active, method, dim, p, &A, &F, g, H) == 0) {
        double hmax = 0.0, nu = 2.0;
        for (int a = 0; a < dim; ++a) if (H[3 * a + a] > hmax) hmax = H[3 * a + a];
        double lambda = 1e-3 * hmax;
        for (int it = 0; it < n_steps; ++it) {
            double delta[3], q[3], A2, F2, g2[3], H2[9], rho = -1.0;
            int ok = lm_step(H, g, lambda, dim, delta) == 0;
            if (ok) {
                for (int a = 0; a < 3; ++a) q[a] = p[a] + delta[a];
                double z_lo, z_hi;
                if (dim == 3 && z_range(m, &z_lo, &z_hi)) {        /* projected step: z stays in its range (R6) */
                    q[2] = q[2] < z_lo ? z_lo : (q[2] > z_hi ? z_hi : q[2]);
                    delta[2] = q[2] - p[2];
                }
                ok = score_grad_prepared(m, S, active, method, dim, q, &A2, &F2, g2, H2) == 0;
            }
            if (ok) {
                double pred = 0.0;
                for (int a = 0; a < dim; ++a) pred += 0.5 * delta[a] * (lambda * delta[a] - g[a]);
                rho = pred > 0.0 ? (F - F2) / pred : -1.0;
            }
            if (ok && rho > 0.0) {
                for (int a = 0; a < 3; ++a) { p[a] = q[a]; g[a] = g2[a]; }
                for (int a = 0; a < 9; ++a) H[a] = H2[a];
                A = A2; F = F2;
                double t = 2.0 * rho - 1.0, f = 1.0 - t * t * t;
                lambda *= f > 1.0 / 3.0 ? f : 1.0 / 3.0;
                nu = 2.0;
            } else {
                lambda *= nu;
                nu *= 2.0;
            }
        }
        xyzA[0] = p[0]; xyzA[1] = p[1]; xyzA[2] = p[2]; xyzA[3] = A; *score = F;
    } else {
        xyzA[3] = NAN; *score = INFINITY;          /* the start point itself is invalid: position kept, no result */
    }
    free(S); free(active);
}

/* xyzA [E][4] in/out (x, y, z start; A out), score [E] out */
int oracle_refine(const oracle_model_t *m, const float *signals, int64_t n_events, int method, int seed_mode, int dim,
                  int n_steps, double *xyzA, double *score, int n_threads)
{
    if (!m || !signals || !xyzA || !score || n_events < 0 || n_steps < 0 || (dim != 2 && dim != 3)) return -1;
    if (dim == 3 && m->lrf_dim != 2 && m->lrf_dim != 5) return -1;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(oracle_threads(n_threads))
#endif
    for (int64_t e = 0; e < n_events; ++e)
        refine_one(m, signals + e * m->n_sensors, method, seed_mode, dim, n_steps, xyzA + 4 * e, score + e);
    return 0;
}
