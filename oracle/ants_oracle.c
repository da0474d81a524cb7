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
