/*
 * ants_recon.h -- C ABI of the B200-native statistical event reconstruction
 * (contracting grids over B-spline LRFs) of the ANTS2 paper, arXiv:1602.07247.
 *
 * Problem statement (section 5.1.2): "For each event, statistical
 * methods search for the position (and, optionally, the event energy) which
 * results in the best match between the ... photosensor signals and those
 * provided by a mathematical model of the detector ... constructed using the
 * light response functions of the photosensors."
 *
 * Method (section 5.1.2.2 "Contracting Grids"): a regular grid of
 * nodes centred at the start position (the centroid); at every
 * node each sensor's LRF gives the expected signal, the energy is "the ratio
 * of two sums over all photosensors: the sum of the photosensor signals and
 * that of the LRF values", the match is Maximum Likelihood or Least Squares
 * (PAPER.md:316); the best node becomes the centre of a finer grid with the
 * same number of nodes; repeated a preconfigured number of iterations.
 * LRFs are cubic B-splines (section 6): axial L(r)
 * or axial+z L(r,z), one shared profile scaled
 * by relative gains or one table per sensor (section 6.2).
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU
 * fallback.  All functions return an ants_status code (0 = OK) and never throw.
 * Points on which the paper is silent follow DESIGN.md "Readings" (R1..R36).
 */
#ifndef ANTS_RECON_H
#define ANTS_RECON_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum ants_status {
    ANTS_OK = 0,
    ANTS_ERR_INVALID = -1,     /* NULL pointer, N < 1, bad knots/dims, G < 2, factor not in (0,1), K < 1, ... */
    ANTS_ERR_UNSUPPORTED = -2, /* valid request outside the compiled limits (see ants_reconstruct) */
    ANTS_ERR_CUDA = -3,        /* a CUDA runtime call failed (no device, launch error, ...) */
    ANTS_ERR_NOMEM = -4,       /* host or device allocation failed */
    ANTS_ERR_SINGULAR = -5     /* ants_lrf_fit_axial: a table is underdetermined (an interval without data) */
};

enum ants_method {
    ANTS_POISSON_ML = 0,  /* A = sum S / sum L; score = Poisson deviance 2 sum[mu - S + S ln(S/mu)], mu = A L (R2) */
    ANTS_CHI_SQUARE = 1,  /* w = 1/max(S,1); A = sum w S L / sum w L^2; score = sum w (S - A L)^2 (R3, R4) */
    ANTS_CHI_SQUARE_SUMRATIO = 2  /* the same score with the energy as PAPER.md:328 states it, A = sum S / sum L (R27);
                                     axial LRFs only */
};

/* Opaque LRF model living in device memory.  Sensor positions, gains and tables are immutable after
 * create; the only mutable state is the sensor selection (ants_lrf_set_selection), which must not be
 * changed while a reconstruction that uses the handle is in flight. */
typedef struct ants_lrf ants_lrf_t;

typedef struct {
    int32_t n_sensors; /* N >= 1 */
    int32_t n_lrf;     /* number of tables.  ants_lrf_create: 1 = one shared profile, L_i = gains[i] * s(.);
                          N = one table per sensor, L_i = s_i(.).  ants_lrf_create_grouped: the number of
                          sensor groups, L_i = gains[i] * s_group[i](.) */
    int32_t lrf_dim;   /* LRF parameterisation (section 6.1): 1 = Axial s(r);
                          2 = Axial+Z s(r,z) tensor product; with ants_lrf_create_xy also
                          3 = XY, 4 = Composite (Axial + XY), 5 = Sliced (XY LRFs on z planes) */
    int32_t n_int_r;   /* uniform intervals in r: n_int_r + 3 coefficients */
    int32_t n_int_z;   /* uniform intervals in z (ignored when lrf_dim == 1) */
} ants_lrf_dims_t;

/*
 * ants_lrf_create -- build the device-resident LRF model (step a0).
 *   sensor_xy HOST [N][2] float, sensor axis positions in mm.
 *   gains     HOST [N] float, all > 0; NULL means all 1.  Used in the centroid
 *              and, when n_lrf == 1, as the profile scale.
 *   knots     HOST {r_lo, r_hi} (lrf_dim 1) or {r_lo, r_hi, z_lo, z_hi} (lrf_dim 2);
 *             breakpoints are uniform inside; requires 0 <= r_lo < r_hi, z_lo < z_hi.
 *   coeffs    HOST [n_lrf][n_int_z + 3 (or 1)][n_int_r + 3] float, r fastest: uniform
 *             cubic B-spline coefficients, no end conditions (R7).  r outside
 *             [r_lo, r_hi] is clamped (R5); z outside [z_lo, z_hi] makes a node invalid (R6).
 *   out       receives the handle; the library owns device copies of everything,
 *             the caller may free its arrays on return.
 * The model is created on the current CUDA device and must be used there.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_UNSUPPORTED (lrf_dim 2 with n_lrf != 1;
 * tables larger than the shared-memory budget), ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_lrf_create(const float *sensor_xy, const float *gains, const float *knots,
                    const float *coeffs, const ants_lrf_dims_t *dims, ants_lrf_t **out);

/*
 * ants_lrf_create_grouped -- the same model with an explicit photosensor grouping (PAPER.md:400-406,
 * section 6.2: "assign a number of photosensors to a group and use the same LRF for all photosensors within
 * it ... a scaling parameter (relative gain) has to be assigned to each of them").  Reading R28:
 *   group   HOST [N] int32, the table index of every sensor, 0 <= group[i] < dims->n_lrf;
 *   coeffs  HOST [n_lrf][n_int_r + 3]: one profile per group;  L_i = gains[i] * s_group[i](r).
 * Axial LRFs only (lrf_dim == 1).  The group tables are shared in shared memory by all sensors of a
 * group.  Other arguments and errors as ants_lrf_create; a group index out of range is ANTS_ERR_INVALID.
 */
int ants_lrf_create_grouped(const float *sensor_xy, const float *gains, const int32_t *group,
                            const float *knots, const float *coeffs, const ants_lrf_dims_t *dims,
                            ants_lrf_t **out);

/* The XY part of an XY-type model (lrf_dim 3, 4, 5). */
typedef struct {
    int32_t n_int_x, n_int_y;  /* uniform intervals of the XY spline in the sensor-local coordinates (u, v) */
    int32_t n_planes;          /* Sliced: number of z planes (>= 2), uniformly spaced from z_lo to z_hi; else 0 */
    const float *knots_xy;     /* HOST {u_lo, u_hi, v_lo, v_hi}, followed by {z_lo, z_hi} for Sliced */
    const float *coeffs_xy;    /* HOST [n_lrf][n_planes or 1][n_int_y + 3][n_int_x + 3] float, u fastest */
    const float *xform;        /* HOST [N][4] or NULL (identity): per-sensor frame T_i, row-major;
                                  (u, v) = T_i (p_xy - P_i) */
    const int32_t *group;      /* HOST [N] table index of every sensor, or NULL (n_lrf = 1 or N as in create) */
} ants_lrf_xy_t;

/*
 * ants_lrf_create_xy -- model with one of the XY-type parameterisations of PAPER.md:388-396 (section 6.1):
 *   lrf_dim 3 "XY LRF": "LRF is a function of X and Y and no other type of symmetry can be assumed" --
 *             L_i = g_i s_t(u, v), a tensor-product cubic B-spline of the position relative to the sensor,
 *             each coordinate clamped into the tabulated range (R30, R5);
 *   lrf_dim 4 "Composite LRF": "a sum of two components: an Axial LRF and an XY LRF" -- L_i = g_i (s_t(r) +
 *             s_t(u, v)); knots/coeffs/dims->n_int_r describe the axial component as in ants_lrf_create (R31);
 *   lrf_dim 5 "Sliced LRF": "a set of several XY LRFs, each defined on a specific Z plane ... linear
 *             interpolation of the LRF values at two closest points from two closest planes" -- planes at
 *             z_lo + p (z_hi - z_lo)/(n_planes - 1); a node with z outside [z_lo, z_hi] is invalid (R32, R6);
 *             searched over (x, y, z) with grid dim 3, or over (x, y) at the fixed z_seed with dim 2.
 * t = group[i], or 0 / i without a grouping; g_i = gains[i] for a shared or group table, 1 for per-sensor
 * tables.  Per-sensor frames serve the grouping "based on rotation or/and reflection symmetry of the sensor
 * array" (ants_group_by_symmetry makes them; R33).  knots and coeffs may be NULL unless
 * lrf_dim == 4.  These models run the general kernel (recon_gen.cuh): FP32 scores on the coarse grids, FP64 on
 * the fine ones.  Errors as ants_lrf_create; ANTS_ERR_UNSUPPORTED if the tables exceed the shared memory.
 */
int ants_lrf_create_xy(const float *sensor_xy, const float *gains, const float *knots, const float *coeffs,
                       const ants_lrf_dims_t *dims, const ants_lrf_xy_t *xy, ants_lrf_t **out);

/*
 * ants_group_by_symmetry -- photosensor groups "based on rotation or/and reflection symmetry of the sensor
 * array (square, rectangular or hexagonal)".  Reading R33: the operations are the rotations by
 * 2 pi k / n_fold about the origin, k = 0 .. n_fold-1 (4 square, 2 rectangular, 6 hexagonal) and, with reflect
 * != 0, each of them applied after the mirror y -> -y.  Sensors are taken in index order; one without a group
 * founds the next group as its reference (identity frame); every operation Q, in the order above, maps the
 * reference position to Q P_ref, and a sensor without a group within tol (mm) of that image (lowest index)
 * joins with the frame T_i = Q^T.
 *   sensor_xy HOST [N][2]; group_out HOST [N] int32; xform_out HOST [N][4] float or NULL; n_groups_out HOST.
 * Host-only.  Errors: ANTS_ERR_INVALID (NULL, N < 1, n_fold < 1, tol < 0 or not finite), ANTS_ERR_NOMEM.
 */
int ants_group_by_symmetry(const float *sensor_xy, int32_t n_sensors, int32_t n_fold, int32_t reflect, float tol,
                           int32_t *group_out, float *xform_out, int32_t *n_groups_out);

/*
 * ants_group_by_radius -- photosensor groups "according to the distance from the sensor center to the
 * detector center" (section 6.2).  Reading R28: sensors are ordered by their distance from
 * the origin (ties: lower index first); a new group starts wherever the distance exceeds the first
 * distance of the current group by more than tol (mm); groups are numbered outward from 0.
 *   sensor_xy HOST [N][2]; group_out HOST [N] int32; n_groups_out HOST int32.  Host-only, no GPU work.
 * Errors: ANTS_ERR_INVALID (NULL, N < 1, tol < 0 or not finite, non-finite position), ANTS_ERR_NOMEM.
 */
int ants_group_by_radius(const float *sensor_xy, int32_t n_sensors, float tol, int32_t *group_out,
                         int32_t *n_groups_out);

/* Number of photosensors of a model (0 for NULL): lets a binding check its buffers. */
int32_t ants_lrf_n_sensors(const ants_lrf_t *lrf);

typedef struct {
    int32_t dim;            /* 2 = search (x,y); 3 = search (x,y,z), requires lrf_dim == 2 or 5 */
    int32_t nodes_per_axis; /* G >= 2; the grid has G^dim nodes */
    float step0_xy;         /* first-iteration node spacing in x and y, mm, > 0 */
    float step0_z;          /* first-iteration node spacing in z, mm (dim == 3), > 0 */
    float factor;           /* contraction factor in (0,1): h_k = h_0 * factor^k (R1) */
    int32_t n_iter;         /* K >= 1 iterations */
    int32_t seed_mode;      /* start position: 0 = centroid, 1 = axis of the
                               sensor with the strongest signal, first one on ties (R20) */
    float z_seed;           /* start z (dim 3) or fixed z (dim 2 with lrf_dim 2); NaN = (z_lo+z_hi)/2 (R10) */
} ants_grid_params_t;

/*
 * ants_lrf_set_selection -- which sensors take part (R19).
 *   passive    HOST [N] bytes, non-zero = passive photosensor (section 5.3: "ignored during
 *              position reconstruction procedures"): left out of the centroid and of every sum; its
 *              signal is never looked at.  NULL = none.
 *   signal_min sensors whose signal (as the method sees it) is below this are ignored in the statistical
 *              part (section 5.1.2); NaN = off.
 *   dist_max   sensors whose axis is farther than this (mm) from the start position (the centroid of the
 *              non-passive sensors) are ignored in the statistical part; NaN = off.
 * The active set is fixed per event before the grid search.  An event with no sensor left, or with
 * sum S <= 0 over them, fails (NaN row, score +inf).  Must not be called while a reconstruction that
 * uses the handle is in flight.  Errors: ANTS_ERR_INVALID (NULL handle), ANTS_ERR_CUDA, ANTS_ERR_NOMEM;
 * ants_reconstruct then returns ANTS_ERR_UNSUPPORTED for an LRF that is not strictly positive.
 */
int ants_lrf_set_selection(ants_lrf_t *lrf, const uint8_t *passive, float signal_min, float dist_max);

/*
 * ants_reconstruct -- steps a1..a6 for a batch of events, ONE kernel launch,
 * asynchronous on `cuda_stream`, no allocation, no host synchronisation.  The launch plan (kernel
 * variant, shared-memory carve-up, occupancy) is computed on the first call with a given
 * (grid, method) and cached in the handle; later calls only fill the parameter block and launch.
 * The handle must be used on the device it was created on (else ANTS_ERR_INVALID).  Up to 1024
 * launches of one handle may be in flight at once; a further launch waits on the device (not on
 * the host) for the launch that used its counter slot 1024 launches earlier.
 *   signals   DEVICE [n_events][N] float row-major, caller-owned, read-only.
 *   out_xyzA  DEVICE [n_events][4] float: x, y, z (0 for axial LRFs), energy A
 *             at the last best node (R11).
 *   out_score DEVICE [n_events] float: the score at that node (deviance or chi-square).
 *   cuda_stream  a cudaStream_t (NULL = default stream).
 * Node order: linear index (iz*G + iy)*G + ix, x fastest; the first strict
 * minimum in that order wins (R9); a node is invalid if z is outside the LRF
 * range, if sum L <= 0 or (Poisson) some L_i <= 0 with S_i > 0.  Poisson ML
 * clips negative signals to 0 first (R18).
 * Per-event failure does not fail the call: an event with a non-finite signal,
 * sum S <= 0 or (centroid start) sum S/g <= 0 gets x = y = z = A = NaN and score = +inf.
 * Errors: ANTS_ERR_INVALID (NULL pointers with n_events > 0, bad grid values,
 * dim 3 with an LRF that does not depend on z, method not 0/1/2), ANTS_ERR_UNSUPPORTED (method 2 with an
 * Axial+Z LRF; packed kernels: G^dim above the compiled limit, 256 nodes in 2-D, 512 in 3-D; general kernel:
 * more than 65535 nodes), ANTS_ERR_CUDA.
 * n_events == 0 is a valid no-op.
 */
int ants_reconstruct(const ants_lrf_t *lrf, const float *signals, int64_t n_events,
                     const ants_grid_params_t *grid, int32_t method,
                     float *out_xyzA, float *out_score, void *cuda_stream);

/*
 * ants_reconstruct_trace -- ants_reconstruct plus, for the parity tests,
 * out_path DEVICE [n_events][K] uint16: the winning linear node index of every
 * iteration (0xFFFF when no node was valid or the event failed).
 */
int ants_reconstruct_trace(const ants_lrf_t *lrf, const float *signals, int64_t n_events,
                           const ants_grid_params_t *grid, int32_t method,
                           float *out_xyzA, float *out_score, uint16_t *out_path,
                           void *cuda_stream);

/*
 * ants_reconstruct_host -- the same reconstruction for HOST buffers: signals,
 * out_xyzA, out_score are host arrays (pinned memory makes the copies
 * asynchronous).  The events are cut into chunks of `chunk_events` (<= 0: 2^20)
 * which are copied in, reconstructed and copied back on a ring of three CUDA
 * streams so that transfers overlap the kernels (BASELINE.json config 5:
 * "processed in 8 streamed batches").  Returns after all results are in host
 * memory.  Errors as ants_reconstruct, plus ANTS_ERR_NOMEM.
 */
int ants_reconstruct_host(const ants_lrf_t *lrf, const float *signals_host, int64_t n_events,
                          const ants_grid_params_t *grid, int32_t method,
                          float *out_xyzA_host, float *out_score_host, int64_t chunk_events);

/*
 * ants_refine -- continuous refinement of reconstructed positions (section 5.1.2: "The best match
 * position is found using either the algorithms provided in the Minuit2 minimization library ... or the
 * contracting grids method"; section 5.1.2.1: minimisation "versus two (XY) or three (XYZ)
 * spatial coordinates", started from a given position).  Reading R34: Levenberg-Marquardt with
 * Nielsen's damping update on the score of `method` with the energy eliminated by its closed form, analytic
 * spline derivatives, Gauss-Newton (Fisher) matrix, n_steps evaluations after the start point; a trial z outside
 * the LRF's z range is projected onto it; the score never increases.  Typical use: ants_reconstruct with about
 * five grid iterations, then a few steps here instead of the remaining grid iterations.
 *   signals DEVICE [n_events][N];  xyzA DEVICE [n_events][4], IN: start position x, y, z (the energy is ignored),
 *   OUT: refined position and its energy;  score DEVICE [n_events], OUT: the score there.
 *   dim 2: (x, y) at the given z; 3: (x, y, z), needs an LRF that depends on z.  seed_mode as in the grid
 *   parameters (it fixes the start position that the distance selection refers to, R19).
 * Rows whose start position is not finite (failed events) are left untouched; an event that is unusable (as in
 * ants_reconstruct) becomes a NaN row with score +inf; a start point that is itself an invalid node keeps its
 * position and gets energy NaN, score +inf.  Everything is computed in FP64 (one warp per event, lanes over
 * sensors), one kernel launch, asynchronous on `cuda_stream`.  Every LRF parameterisation is supported.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_UNSUPPORTED (tables exceed the shared memory), ANTS_ERR_CUDA.
 */
int ants_refine(const ants_lrf_t *lrf, const float *signals, int64_t n_events, int32_t method, int32_t dim,
                int32_t seed_mode, int32_t n_steps, float *xyzA, float *score, void *cuda_stream);

/*
 * ants_lrf_fit_axial -- LRF calculation (section 6: "The LRF module calculates these
 * functions from datasets containing photosensor signals and the corresponding event positions";
 * one LRF per sensor or one per group with relative gains; positions reconstructed
 * or true).  This is the other half of the iterative response reconstruction of PAPER.md:428 (section 8):
 * ants_reconstruct gives positions and energies, this call refits the axial B-spline LRFs from them.
 * Readings R21-R23: unweighted least squares of y = S / (A g) against the uniform cubic
 * B-spline at r = |p_xy - P_i|; an event takes part if x, y, A are finite and A > 0; a (event, sensor)
 * pair takes part if r_lo <= r <= r_hi; signals enter as they are.
 *   sensor_xy  HOST [N][2];  gains HOST [N] or NULL (all 1; used only when n_lrf == 1);
 *   knots      HOST {r_lo, r_hi};  n_lrf = 1 (shared profile) or N (one table per sensor);
 *   signals    DEVICE [n_events][N];  xyzA DEVICE [n_events][4] = x, y, z, A (out_xyzA of ants_reconstruct,
 *              or true positions with A = the known light output);
 *   coeffs_out HOST [n_lrf][n_int_r + 3] float;  n_used_out HOST [n_lrf] double or NULL: pairs per table.
 * The normal equations are accumulated on the GPU in FP64 (one kernel launch on `cuda_stream`), the banded
 * systems are solved on the host; scratch comes from a device arena the library keeps (fit calls are serialised
 * by its lock); the call returns after the result is in host memory.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_SINGULAR (an interval of some table received no data), ANTS_ERR_CUDA,
 * ANTS_ERR_NOMEM, ANTS_ERR_UNSUPPORTED (accumulators larger than shared memory).
 */
int ants_lrf_fit_axial(const float *sensor_xy, const float *gains, const float *knots, int32_t n_sensors,
                       int32_t n_lrf, int32_t n_int_r, const float *signals, const float *xyzA, int64_t n_events,
                       float *coeffs_out, double *n_used_out, void *cuda_stream);

/*
 * ants_lrf_fit_gains -- relative gains of the sensors for a FIXED shared profile (section 6.3:
 * "re-calculate the relative gains of the photosensors within already defined groups without affecting the
 * LRF profiles").  Reading R24: g_i = sum_e y s(r_ie) / sum_e s(r_ie)^2, y = S_ie / A_e, over the events and
 * pairs of R22 (as in ants_lrf_fit_axial).
 *   sensor_xy HOST [N][2], knots HOST {r_lo, r_hi}, coeffs HOST [n_int_r + 3] (the shared profile),
 *   signals DEVICE [n_events][N], xyzA DEVICE [n_events][4];
 *   gains_out HOST [N] float (NaN for a sensor without any pair), n_used_out HOST [N] double or NULL.
 * One kernel launch on `cuda_stream` (FP64 sums kept in registers per lane, N <= 128); returns after the
 * result is in host memory.  Errors: ANTS_ERR_INVALID, ANTS_ERR_UNSUPPORTED (N > 128), ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_lrf_fit_gains(const float *sensor_xy, const float *knots, const float *coeffs, int32_t n_sensors,
                       int32_t n_int_r, const float *signals, const float *xyzA, int64_t n_events,
                       float *gains_out, double *n_used_out, void *cuda_stream);

/*
 * ants_lrf_fit_gains_static -- ants_lrf_fit_gains for callers that must not allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same reading (R24), same result
 * (FP64 sums; the order of the final additions differs, so the gains agree to rounding, the pair counts exactly).
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine, and uses no host heap either:
 * the kernel's scratch -- sums, pair counters, the device copies of sensor_xy and coeffs -- is one array of
 * ANTS_STATIC_SCRATCH_BYTES (8 KB) built into the library, which every GPU that loads the library holds until the
 * process exits.  Hence the fixed limits: n_sensors <= ANTS_STATIC_MAX_SENSORS and n_int_r + 3 <=
 * ANTS_STATIC_MAX_COEFFS; a larger request is refused with ANTS_ERR_UNSUPPORTED, nothing is truncated.
 * Every call on a device uses the same array, which keeps the previous call's contents: the call clears the sums
 * and counters and overwrites the rest before its kernel runs, and the library serialises the calls of one process
 * with a lock and returns only after the result is in host memory -- but work that touches the array while a call is
 * in flight on the GPU (there is none in this library) would race with it.  One kernel launch on `cuda_stream`.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_UNSUPPORTED (beyond the limits above; device ordinal >= 64), ANTS_ERR_CUDA.
 */
#define ANTS_STATIC_MAX_SENSORS 128
#define ANTS_STATIC_MAX_COEFFS 1024
#define ANTS_STATIC_SCRATCH_BYTES 8192
int ants_lrf_fit_gains_static(const float *sensor_xy, const float *knots, const float *coeffs, int32_t n_sensors,
                              int32_t n_int_r, const float *signals, const float *xyzA, int64_t n_events,
                              float *gains_out, double *n_used_out, void *cuda_stream);

/*
 * ants_gains_renormalise -- relative gains are defined up to a common factor ("a scaling
 * parameter (relative gain)"); after a re-evaluation (ants_lrf_fit_gains) the iterative procedure of
 * PAPER.md:428-440 carries them on at the scale of the previous set.  Reading R29: a sensor whose new
 * estimate is missing (NaN) or not positive keeps its previous gain; the set is then multiplied by
 * mean(gains_prev) / mean(set), all in double, rounded once to float.
 *   gains_new HOST [N], gains_prev HOST [N] (all > 0), gains_out HOST [N] (may alias gains_new).
 * Host-only.  Errors: ANTS_ERR_INVALID (NULL, N < 1, a previous gain that is not positive and finite).
 */
int ants_gains_renormalise(const float *gains_new, const float *gains_prev, int32_t n_sensors, float *gains_out);

/*
 * ants_lrf_fit_axial_grouped -- ants_lrf_fit_axial with an explicit sensor grouping (section
 * 6.2: one group for all sensors, grouping by the distance from the sensor centre to the detector centre, or
 * by the symmetry of the array).  Reading R28: group HOST [N] int32 gives every sensor's table index in
 * 0 .. n_groups-1; the sensors of a group share one profile, each scaled by its relative gain (gains HOST [N]
 * or NULL).  coeffs_out HOST [n_groups][n_int_r + 3], n_used_out HOST [n_groups] or NULL.  The result goes
 * straight into ants_lrf_create_grouped with the same group array.
 * Other arguments, behaviour and errors as ants_lrf_fit_axial; a group index out of range is ANTS_ERR_INVALID.
 */
int ants_lrf_fit_axial_grouped(const float *sensor_xy, const float *gains, const int32_t *group, const float *knots,
                               int32_t n_sensors, int32_t n_groups, int32_t n_int_r, const float *signals,
                               const float *xyzA, int64_t n_events, float *coeffs_out, double *n_used_out,
                               void *cuda_stream);

/*
 * ants_lrf_fit_axial_z -- LRF calculation for the shared axial+z tensor-product LRF s(r, z) (PAPER.md:394,
 * section 6.1.2).  Reading R25: as ants_lrf_fit_axial with y = S / (A g) against the tensor
 * spline; an event also needs a finite z inside [z_lo, z_hi].
 *   sensor_xy HOST [N][2], gains HOST [N] or NULL, knots HOST {r_lo, r_hi, z_lo, z_hi},
 *   signals DEVICE [n_events][N], xyzA DEVICE [n_events][4] = x, y, z, A;
 *   coeffs_out HOST [n_int_z + 3][n_int_r + 3] float (r fastest), n_used_out HOST [1] double or NULL.
 * Normal equations in FP64 on the GPU (one launch on `cuda_stream`), dense Cholesky on the host.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_SINGULAR, ANTS_ERR_UNSUPPORTED ((n_int_z+3)(n_int_r+3) > 768),
 * ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_lrf_fit_axial_z(const float *sensor_xy, const float *gains, const float *knots, int32_t n_sensors,
                         int32_t n_int_r, int32_t n_int_z, const float *signals, const float *xyzA,
                         int64_t n_events, float *coeffs_out, double *n_used_out, void *cuda_stream);

/*
 * ants_lrf_fit_xy -- LRF calculation for XY tables ("XY LRF") and for the XY component
 * of a Composite LRF ("During LRF calculation, the axial component is evaluated first, and the
 * residual is used to calculate the XY LRF component").  Reading R35 = R21-R23 in the sensor-local coordinates
 * (u, v) = T_i (p - P_i): unweighted least squares of y = S / (A g_i) -- minus the table's axial spline at
 * |p - P_i| (argument clamped, R5) when coeffs_ax is given -- against the tensor-product spline; an event takes
 * part if x, y, A are finite and A > 0, a pair if u and v lie inside the tabulated ranges.
 *   sensor_xy HOST [N][2]; gains HOST [N] or NULL; group HOST [N] int32 or NULL (n_lrf = 1 or N then); xform HOST
 *   [N][4] or NULL; knots_xy HOST {u_lo, u_hi, v_lo, v_hi}; knots_ax HOST {r_lo, r_hi} and coeffs_ax HOST
 *   [n_lrf][n_int_r + 3] for a Composite fit (first fitted with ants_lrf_fit_axial / _grouped), else NULL;
 *   signals DEVICE [n_events][N]; xyzA DEVICE [n_events][4];
 *   coeffs_out HOST [n_lrf][n_int_y + 3][n_int_x + 3] float; n_used_out HOST [n_lrf] double or NULL.
 * One kernel launch (FP64 normal equations) and one dense Cholesky solve on the host per table; returns after the
 * result is in host memory.  The result goes straight into ants_lrf_create_xy.  Sliced tables: ants_lrf_fit_sliced.
 * Errors: ANTS_ERR_INVALID, ANTS_ERR_SINGULAR (a cell of some table received no data),
 * ANTS_ERR_UNSUPPORTED ((n_int_x + 3)(n_int_y + 3) > 768), ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_lrf_fit_xy(const float *sensor_xy, const float *gains, const int32_t *group, const float *xform,
                    const float *knots_xy, int32_t n_sensors, int32_t n_lrf, int32_t n_int_x, int32_t n_int_y,
                    const float *knots_ax, const float *coeffs_ax, int32_t n_int_r, const float *signals,
                    const float *xyzA, int64_t n_events, float *coeffs_out, double *n_used_out, void *cuda_stream);

/*
 * ants_lrf_fit_sliced -- LRF calculation for Sliced tables ("a set of several XY LRFs, each defined on
 * a specific Z plane.  The LRF values for the points between the planes are calculated using linear interpolation of
 * the LRF values at two closest points from two closest planes").  The paper does not say how the
 * planes' tables are obtained; reading R36: ALL planes of a table are fitted jointly, unweighted least squares of
 * y = S / (A g_i) against (1 - w) s_p(u, v) + w s_{p+1}(u, v) -- the value the reconstruction evaluates for the pair,
 * p = min(floor((z - z_lo)/dz), n_planes - 2), w = (z - z_p)/dz, dz = (z_hi - z_lo)/(n_planes - 1); an event takes
 * part if x, y, z, A are finite, A > 0 and z_lo <= z <= z_hi, a pair if u and v lie inside the tabulated ranges.
 *   sensor_xy HOST [N][2]; gains HOST [N] or NULL; group HOST [N] int32 or NULL (n_lrf = 1 or N then); xform HOST
 *   [N][4] or NULL; knots_xy HOST {u_lo, u_hi, v_lo, v_hi, z_lo, z_hi}; signals DEVICE [n_events][N];
 *   xyzA DEVICE [n_events][4];
 *   coeffs_out HOST [n_lrf][n_planes][n_int_y + 3][n_int_x + 3] float; n_used_out HOST [n_lrf] double or NULL.
 * Per table 3 (n_planes - 1) kernel launches (FP64 normal equations: per slab the blocks plane-plane, next-next and
 * plane-next of the block-tridiagonal matrix) and one banded Cholesky solve on the host; returns after the result is
 * in host memory.  The result goes straight into ants_lrf_create_xy (lrf_dim 5).  Errors: ANTS_ERR_INVALID,
 * ANTS_ERR_SINGULAR (some coefficient received no data), ANTS_ERR_UNSUPPORTED ((n_int_x + 3)(n_int_y + 3) > 768 or
 * more than 8192 unknowns per table), ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_lrf_fit_sliced(const float *sensor_xy, const float *gains, const int32_t *group, const float *xform,
                        const float *knots_xy, int32_t n_sensors, int32_t n_lrf, int32_t n_int_x, int32_t n_int_y,
                        int32_t n_planes, const float *signals, const float *xyzA, int64_t n_events,
                        float *coeffs_out, double *n_used_out, void *cuda_stream);

/* Event-filter criteria (section 5.2); NaN switches a criterion off. */
typedef struct {
    float score_max;    /* keep score <= score_max (chi-square / deviance of the reconstruction) */
    float energy_min;   /* keep A >= energy_min */
    float energy_max;   /* keep A <= energy_max */
    float radius_max;   /* keep x^2 + y^2 <= radius_max^2 */
} ants_filter_t;

/*
 * ants_filter_events -- event filters on the reconstruction's own outputs (events "can be
 * filtered out according to ... reconstructed ... event energy, chi-squared value of the reconstruction, and
 * the event position"; "Only those events which pass all the activated filters are used in LRF
 * reconstruction").  Reading R26.  Rows of xyzA (DEVICE [n_events][4], modified IN PLACE) that fail, and rows
 * of failed reconstructions, become NaN -- exactly what ants_lrf_fit_* ignore; score (DEVICE [n_events]) is
 * read only.  n_pass_out (HOST, may be NULL) receives the number of passing events; the call then waits for
 * the stream, otherwise it is asynchronous.  Errors: ANTS_ERR_INVALID, ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_filter_events(float *xyzA, const float *score, int64_t n_events, const ants_filter_t *filter,
                       int64_t *n_pass_out, void *cuda_stream);

/* Release the model and its device memory.  NULL is a no-op. */
void ants_destroy(ants_lrf_t *lrf);

/* Static, NUL-terminated description of a status code. */
const char *ants_strerror(int status);

/* Number of reconstruction kernels this library has launched in this process
 * (bench.py reports it as gpu_launches). */
int64_t ants_launch_count(void);

/*
 * ants_plan_info -- introspection of how a call runs (no kernel launch): first iteration index that
 * uses the differential score (K if none), nodes handled per lane, warps per CTA, resident CTAs per SM
 * (as the runtime's occupancy calculator reports them for the chosen kernel and shared-memory size;
 * 0 if no device can be asked) and dynamic shared-memory bytes per CTA.  Any output pointer may be
 * NULL.  Errors as ants_reconstruct.
 */
int ants_plan_info(const ants_lrf_t *lrf, const ants_grid_params_t *grid, int32_t method,
                   int32_t *first_diff_iter, int32_t *nodes_per_lane, int32_t *warps_per_cta,
                   int32_t *ctas_per_sm, int32_t *smem_bytes);

/*
 * ants_plan_kernel_name -- the name of the kernel instantiation ants_reconstruct launches for this
 * (model, grid, method), as a profiler shows it (e.g. "ants::recon2d_pk_kernel<3,0>"), NUL-terminated
 * and truncated to name_cap bytes.  Host-only.  Errors as ants_plan_info, plus ANTS_ERR_INVALID for a
 * NULL or empty buffer.
 */
int ants_plan_kernel_name(const ants_lrf_t *lrf, const ants_grid_params_t *grid, int32_t method,
                          char *name_out, int32_t name_cap);

/*
 * ants_probe_throughput -- micro-benchmark behind the roofline denominator (bench.py --workload peak):
 * a grid that fills the device runs `iters` x 128 dependent-free instructions per thread of one kind:
 *   0 FFMA (fp32 fused multiply-add, one operand register reused),  1 FFMA2 (packed pair, fma.rn.f32x2),
 *   2 MUFU (lg2.approx),  3 DFMA (fp64),  4 FFMA whose three source registers are all distinct.
 * lane_ops_per_second_out (HOST) receives scalar results per second (an FFMA2 counts two; x 2 = flop/s for
 * the FMA kinds); milliseconds_out (HOST, may be NULL) the timed launch's duration.  Uses the default stream
 * of the current device and waits for it.  Errors: ANTS_ERR_INVALID, ANTS_ERR_CUDA, ANTS_ERR_NOMEM.
 */
int ants_probe_throughput(int32_t kind, int32_t iters, double *lane_ops_per_second_out, double *milliseconds_out);

#ifdef __cplusplus
}
#endif
#endif /* ANTS_RECON_H */
