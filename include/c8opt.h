/*
 * c8opt.h -- C-ABI boundary of the B200-native optical photon path.
 *
 * The path (arxiv 2309.15861, Baack & Alameddine, ICRC2023; cited as
 * PAPER.md:<line>; "R<n>" = a reading listed in DESIGN.md §2):
 *
 *   charged-particle track segment
 *     -> Cherenkov photons   (Frank-Tamm yield PAPER.md:43-45, homogeneous step
 *                             PAPER.md:47, cone generated downward and rotated by
 *                             the 180-degree Rodrigues matrix PAPER.md:49-73)
 *     -> fluorescence photons (constant yield x energy loss, positions uniform
 *                             along the track, isotropic PAPER.md:29-35, or
 *                             beamed toward a telescope PAPER.md:39)
 *     -> straight-line propagation with the optical-path arrival time and an
 *        optional transmission weight (R8, R17)
 *     -> telescope-sphere intersection (BASELINE.json north_star, R10)
 *     -> per-telescope tally, or compacted 28-byte photon-bunch records.
 *
 * All of it runs in hand-written CUDA kernels for sm_100a.  There is no CPU
 * fallback: without a CUDA device every entry point that needs one returns
 * C8OPT_ERR_CUDA.
 *
 * Conventions
 *   - plain C types only; "host" / "device" is stated for every pointer.
 *   - return value: 0 = OK, negative = error code below; the message of the
 *     last error of a context is available from c8opt_last_error().
 *   - units: metres, nanoseconds, nanometres (wavelength), g/cm^2 (depth), MeV.
 *   - geometry: flat atmosphere, z up = altitude above sea level (R9).
 *   - one context per host thread; calls on one context must not overlap.
 *   - a context belongs to the CUDA device that was current when it was created;
 *     every entry point makes that device current for its own duration and
 *     restores the caller's device before it returns.
 */
#ifndef C8OPT_H
#define C8OPT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define C8OPT_OK              0
#define C8OPT_ERR_ARGUMENT   (-1)  /* null pointer, bad size, non-monotone layers, ...   */
#define C8OPT_ERR_CUDA       (-2)  /* CUDA runtime error or no sm_100 device             */
#define C8OPT_ERR_CAPACITY   (-3)  /* photon-output region overflowed (records dropped)  */

#define C8OPT_MAX_LAYERS      8
#define C8OPT_MAX_TELESCOPES  4096

#define C8OPT_PROC_CHERENKOV     1u   /* bit 0 of c8opt_run_params.processes */
#define C8OPT_PROC_FLUORESCENCE  2u   /* bit 1 */
#define C8OPT_MODE_TALLY   0u
#define C8OPT_MODE_OUTPUT  1u
/* Ground-plane radial profile (section 3.1 "Intensity & Timing Profile", Fig. 3a / 3b): every bunch
 * that crosses the observation level z = h_obs going down is binned by its distance r from the shower core
 * (c8opt_set_ground_histogram); a bin holds {n, sum w, sum w t} with the arrival time of R8 on that plane and the
 * transmission weight of R17.  Telescopes are not consulted and none are needed (R26). */
#define C8OPT_MODE_GROUND_HIST 2u
/* c8opt_run_params.flags.  CULL: segment culling (Fig. 2 :63-65) in its exact, conservative form:
 * a Cherenkov segment whose emission cone provably misses every telescope sphere -- for every telescope k,
 * | angle(d, c_k - p_mid) - theta_c | > asin(R_k / D) + asin((L/2) / D), D = |c_k - p_mid| - L/2 -- skips the
 * photon loop.  Tallies and records are identical with and without it; the skipped bunches still count as
 * generated and are reported in counters[C8OPT_CNT_CULLED]; C8OPT_CNT_UPWARD then covers propagated bunches only. */
/* c8opt_run_params.fl_beam_telescope = C8OPT_BEAM_ARRAY: PAPER.md:39 for several telescopes ("an emission area is
 * defined which includes all telescopes involved"; "the required scaling factor is calculated and applied to the total
 * number of photons").  Per segment, the emission is uniform in the cone about the line from the segment midpoint to
 * the centre of the sphere holding every telescope sphere (centre of the bounding box of the telescope centres,
 * R_b = max |c_k - centre| + R_k), sin(alpha) = (R_b + L/2) / D; the photon NUMBER is mu (1 - cos alpha) / 2 and the
 * bunches keep weight mu'/n_b; segments inside that sphere emit isotropically, unscaled.  fl_beam_halfangle_rad is
 * not used (R28). */
#define C8OPT_BEAM_ARRAY   (-2)
#define C8OPT_FLAG_CULL    1u
/* REFRACT: the refraction corrections of PAPER.md:77 ("straight line propagation followed by the application of
 * correction factors which changes the arrival angle, position, and timing") in the first-order planar-Snell reading
 * DESIGN.md R27: on the plane of the telescope centre the arrival point moves by
 *   dr = tan(theta0) / cos^2(theta0) [eta(e_z) (e_z - c_z) - kappa (T(c_z) - T(e_z))]   along the horizontal flight
 * direction and the direction turns by dtheta = tan(theta0) (eta(e_z) - eta(c_z)); the sphere test and the record
 * use the corrected point and direction; the arrival time (optical path, R8) changes only to second order and stands. */
#define C8OPT_FLAG_REFRACT 2u
/* CUT_CENTRE / CUT_TELESCOPES: the paper's own angular particle cut (section 1.2.1, Fig. 2 :63-65; DESIGN.md
 * R29): "calculate the angle difference between the currently handled particles' flight direction and the vector to the
 * experiment center.  For higher precision, the minimum angle to each individual telescope can be used."  A Cherenkov
 * segment whose direction is more than c8opt_run_params.cut_angle_rad (the paper recommends 6 degrees) off the vector
 * from its midpoint to the experiment centre (centre of the bounding box of the telescope centres) -- or, with
 * CUT_TELESCOPES, off the vector to every telescope centre -- is not handled: no photon is drawn.  Unlike CULL this cut
 * is LOSSY (that is the paper's trade; its Fig. 2 is the lost light against the cut angle): tallies and records are those
 * of the kept segments.  The bunches of a cut segment still count as generated and are reported in
 * counters[C8OPT_CNT_CULLED].  Fluorescence is never cut.  Both flags set = CUT_TELESCOPES. */
#define C8OPT_FLAG_CUT_CENTRE      4u
#define C8OPT_FLAG_CUT_TELESCOPES  8u

typedef struct c8opt_ctx c8opt_ctx;   /* opaque, owned by the library */

/* One atmosphere layer: column depth T(h) = a + b exp(-h / c) [g/cm^2] for
 * h >= h_lo (layer 0 also covers h < h_lo of layer 0).  Density is -dT/dh.
 * (BASELINE.json configs[1] "T(h)=a_i+b_i*exp(-h/c_i)"; R18.) */
typedef struct { double h_lo_m, a_gcm2, b_gcm2, c_m; } c8opt_layer;

/* Atmosphere descriptor (host memory, copied by c8opt_create_atmosphere).
 * Refractivity n(h) - 1 = eta0 * rho(h) / rho0.  tau is the optional vertical
 * optical-depth table tau(h, lambda) from altitude h down to the observation
 * level, row-major [tau_nh][tau_nl], bilinear, clamped at the edges (R17);
 * tau == NULL or tau_nh == 0 means no absorption. */
typedef struct {
    int32_t     n_layers;                       /* 1 .. C8OPT_MAX_LAYERS, h_lo ascending */
    c8opt_layer layers[C8OPT_MAX_LAYERS];
    double      eta0, rho0_gcm3, h_obs_m;
    int32_t     tau_nh, tau_nl;
    double      tau_h0_m, tau_dh_m, tau_l0_nm, tau_dl_nm;
    const float *tau;                           /* host */
} c8opt_atmosphere_desc;

/* One track segment, 48 bytes ("steps ... a couple of meters").
 * (dx,dy,dz) is the unit direction (re-normalised in fp64; off unity by more
 * than 1e-3 => the segment is counted invalid and emits nothing), gamma the
 * Lorentz factor (> 1), charge in units of e, dE the energy loss over the
 * segment (used by fluorescence only), flags bit 0 = muon label (ignored). */
typedef struct {
    float x0, y0, z0, t0_ns;
    float dx, dy, dz, length_m;
    float gamma, charge, dE_MeV;
    uint32_t flags;
} c8opt_segment;

/* Run parameters (host memory, read during the call). */
typedef struct {
    uint64_t seed;                 /* Philox key = (seed[31:0], seed[63:32])  (R20)        */
    uint32_t processes;            /* C8OPT_PROC_* bits                                     */
    uint32_t mode;                 /* C8OPT_MODE_TALLY, C8OPT_MODE_OUTPUT or C8OPT_MODE_GROUND_HIST */
    double   lam1_nm, lam2_nm;     /* Cherenkov band (PAPER.md:45 integral over lambda)     */
    double   bunch_size;           /* B: n_b = ceil(mu / B) bunches of weight mu / n_b (R1) */
    double   fl_yield_per_MeV;     /* constant fluorescence yield (R13)        */
    double   fl_lam1_nm, fl_lam2_nm;
    int32_t  fl_beam_telescope;    /* -1 isotropic; k >= 0 beam toward telescope k (R14);
                                      C8OPT_BEAM_ARRAY beam at the whole array (R28)        */
    uint32_t flags;                /* C8OPT_FLAG_* bits                                     */
    double   fl_beam_halfangle_rad;
    double   cut_angle_rad;        /* C8OPT_FLAG_CUT_*: the angular particle cut, in [0, pi] */
    double   cauchy_b_nm2;         /* b >= 0 [nm^2] of n(lambda, h) - 1 = eta(h) (1 + b / lambda^2); 0: n does not depend on
                                      lambda.  > 0 (the Frank-Tamm integrand with n(lambda); R30): the
                                      yield is the integral over the band (16-interval Simpson in 1 / lambda, cut at the
                                      threshold), every photon leaves at the Cherenkov angle of its own wavelength and carries
                                      sin^2(lambda) / <sin^2> as a weight factor.  Runs on kernel instances of its own (the
                                      general photon loop: about 3.6 x the time of the plain run on configs[1]); not with
                                      C8OPT_FLAG_CULL, not in C8OPT_MODE_GROUND_HIST.  Air in the band 300-600 nm: b ~ 5.7e3 nm^2 */
} c8opt_run_params;

/* Optional outputs of one propagate call; every pointer is DEVICE memory owned
 * by the caller and may be NULL (all NULL / out == NULL in plain tally mode).
 *   records      : photon-output mode; 7 floats per record {x, y, cos_x, cos_y,
 *                  t, lambda, weight}: x, y on the horizontal plane through the
 *                  telescope centre, relative to the centre (R11).  Telescope k
 *                  owns records [tel_offset[k], tel_offset[k] + tel_capacity[k]);
 *                  the library keeps one cursor per telescope in the context
 *                  (cleared by c8opt_reset_tallies) so consecutive calls append.
 *   ids          : parallel to records; (segment id << 25) | (process tag << 24)
 *                  | photon index, for validation.
 *   counts       : uint32[n][2], bunches n_b emitted by segment i for the
 *                  Cherenkov (tag 0) and fluorescence (tag 1) process.
 * Record order inside a telescope region is unspecified (R22). */
typedef struct {
    float          *records;
    const uint64_t *tel_offset;      /* device, [n_tel], in records */
    const uint64_t *tel_capacity;    /* device, [n_tel], in records */
    uint64_t       *ids;
    uint32_t       *counts;
} c8opt_output;

typedef struct { uint64_t hits; double sum_w; double sum_wt; } c8opt_tally;

/* One radial bin of the ground-plane profile: bunches, sum of weights, sum of weight x arrival time [ns].
 * Photon density = sum_w / (pi (r_hi^2 - r_lo^2)); mean arrival time = sum_wt / sum_w; the paper masks bins with
 * fewer than 50 photons -- left to the caller. */
typedef struct { uint64_t n; double sum_w; double sum_wt; } c8opt_hist_bin;

/* indices into the counters[8] array of c8opt_read_tallies */
enum {
    C8OPT_CNT_SEGMENTS = 0, C8OPT_CNT_GENERATED = 1, C8OPT_CNT_UPWARD = 2, C8OPT_CNT_HITS = 3,
    C8OPT_CNT_RECORDS = 4, C8OPT_CNT_DROPPED = 5, C8OPT_CNT_INVALID = 6, C8OPT_CNT_CULLED = 7
};

/* Validate the descriptor, build the layer / transmission tables and upload
 * them to the current CUDA device.  *out receives a new context.
 * Errors: ARGUMENT (null, n_layers out of range, h_lo not ascending, c <= 0,
 * rho0 <= 0, bad tau shape), CUDA. */
int c8opt_create_atmosphere(const c8opt_atmosphere_desc *desc, c8opt_ctx **out);

/* Replace the telescope set: xyzr is HOST float[n][4] = centre and radius of
 * each sphere (BASELINE.json north_star "telescopes' spheres").  Builds the
 * ground-plane candidate grid used when n is large and clears the tallies.
 * Errors: ARGUMENT (n < 1 or > C8OPT_MAX_TELESCOPES, radius <= 0, non-finite). */
int c8opt_add_telescopes(c8opt_ctx *ctx, const float *xyzr, int32_t n);

/* Generate, propagate, intersect and tally / write the photons of n segments
 * (DEVICE array d_seg) with global ids first_segment_id + i.  Asynchronous on
 * `cuda_stream` (a cudaStream_t; NULL = default stream) in every mode: the call
 * only enqueues work (kernel launches and, in photon-output mode, one small
 * device-to-device copy of tel_capacity into the context), allocates nothing
 * and never waits for the device; it accumulates into the context's tallies
 * and counters, so many batches may precede one read.  out->tel_offset /
 * tel_capacity must stay valid until the enqueued work has run.
 * Random stream (R20): Philox4x32-10, key = seed.  A fluorescence
 * photon j of segment S draws the block with counter (j, S[31:0], S[63:32], 1);
 * the Cherenkov photons 2k and 2k + 1 share the block with counter
 * (k, S[31:0], S[63:32], 0) -- words (r0, r1) for the even one, (r2, r3) for the
 * odd one.  The stream is a function of (seed, segment id, photon index) only:
 * results do not depend on how segments are batched.
 * Errors: ARGUMENT (null, no telescopes, bad params, output mode without
 * records / offsets), CUDA. */
int c8opt_propagate_segments(c8opt_ctx *ctx, const c8opt_segment *d_seg, uint64_t n,
                             uint64_t first_segment_id, const c8opt_run_params *params,
                             const c8opt_output *out, void *cuda_stream);

/* Same path with the segments in HOST memory (pinned memory makes the copies
 * asynchronous): the segment table is cut into chunks (a small first one, then
 * doubling up to a quarter of the table) whose host->device copy overlaps the
 * kernel of the previous chunk on two internal streams; returns after all work
 * is enqueued, ordered after prior work on `cuda_stream`, and `cuda_stream`
 * waits for it (also when an error is returned half way).  out->counts, if
 * given, is still DEVICE memory.  Needs three device staging buffers of one
 * chunk each: allocated by c8opt_reserve_host_staging, else by the first call
 * that needs them (that call then synchronises the internal streams once). */
int c8opt_propagate_segments_host(c8opt_ctx *ctx, const c8opt_segment *h_seg, uint64_t n,
                                  uint64_t first_segment_id, const c8opt_run_params *params,
                                  const c8opt_output *out, void *cuda_stream);

/* Create the internal streams and allocate the three device staging buffers of
 * c8opt_propagate_segments_host for tables of up to max_segments segments
 * (3 x 48 bytes x min(max(max_segments / 4, 32 Ki), 1 Mi), rounded to whole
 * tiles), so that no later call allocates.  Errors: CUDA. */
int c8opt_reserve_host_staging(c8opt_ctx *ctx, uint64_t max_segments);

/* Synchronise with all work enqueued on the context and copy the results to
 * HOST memory: host_out[n_tel] tallies, counters[8] (may be NULL),
 * host_tel_count[n_tel] = records written per telescope (may be NULL).
 * Returns C8OPT_ERR_CAPACITY if any record was dropped (results are still
 * copied); ARGUMENT if n_tel differs from the telescope count. */
int c8opt_read_tallies(c8opt_ctx *ctx, c8opt_tally *host_out, int32_t n_tel,
                       uint64_t *counters, uint64_t *host_tel_count);

/* Configure (n_bins in 1 .. 1024) or drop (n_bins == 0) the ground-plane radial profile: n_bins equal bins of
 * width r_max_m / n_bins about the core (core_x_m, core_y_m) on the observation level of the atmosphere; bunches
 * landing at r >= r_max_m are counted as overflow.  Allocates n_bins + 1 device bins, zeroed (and zeroed again by
 * c8opt_reset_tallies).  Synchronises the device.  Errors: ARGUMENT, CUDA. */
int c8opt_set_ground_histogram(c8opt_ctx *ctx, double core_x_m, double core_y_m, double r_max_m, int32_t n_bins);

/* Wait for the device and copy the profile accumulated by the C8OPT_MODE_GROUND_HIST calls since the last reset to
 * HOST memory: host_out[n_bins]; *overflow (may be NULL) = bunches beyond r_max; counters[8] (may be NULL) as in
 * c8opt_read_tallies with HITS = bunches that reached the plane.  Errors: ARGUMENT (n_bins mismatch), CUDA. */
int c8opt_read_ground_histogram(c8opt_ctx *ctx, c8opt_hist_bin *host_out, int32_t n_bins, uint64_t *overflow, uint64_t *counters);

/* Zero tallies, counters and the per-telescope record cursors (asynchronous
 * on `cuda_stream`). */
int c8opt_reset_tallies(c8opt_ctx *ctx, void *cuda_stream);

void c8opt_destroy(c8opt_ctx *ctx);

/* Message of the last error on this context (or of the last failed
 * c8opt_create_atmosphere when ctx == NULL).  Never NULL. */
const char *c8opt_last_error(const c8opt_ctx *ctx);

/* Number of kernels launched by this context so far (for bench.py's
 * gpu_launches). */
uint64_t c8opt_launch_count(const c8opt_ctx *ctx);

/* ---- the entry point that allocates nothing --------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the tally-mode pass (the same kernels as c8opt_propagate_segments with C8OPT_MODE_TALLY) with
 * no context and no allocation.  What the context path keeps in cudaMalloc'ed memory -- the counters and tallies the
 * kernel accumulates into, and the telescope tables -- lives in ONE file-scope `static __device__` array of
 * C8OPT_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit); its stated
 * limit is C8OPT_STATIC_MAX_TELESCOPES telescopes.  The call makes no cudaMalloc / cudaFree / cudaMallocHost and no
 * allocating library call; it enqueues a set-up kernel (tables written, accumulators zeroed: the array keeps the last
 * call's contents), the propagate kernel(s) and a kernel that writes the results, all on `cuda_stream`, and returns
 * without synchronising.  The first call on a device also looks up the array's address and raises the kernels'
 * shared-memory limit (once per device, the CURRENT device is used).
 *   atmosphere   HOST, as for c8opt_create_atmosphere, except that atmosphere->tau is ignored:
 *   d_tau        DEVICE, the transmission table tau[tau_nh][tau_nl] (shape / axes from `atmosphere`), or NULL for none;
 *                the caller's memory, read by the kernels
 *   xyzr, n_tel  HOST, as for c8opt_add_telescopes; 1 <= n_tel <= C8OPT_STATIC_MAX_TELESCOPES
 *   d_seg, n, first_segment_id, params   as for c8opt_propagate_segments; params->mode must be C8OPT_MODE_TALLY
 *   d_tallies_out    DEVICE, [n_tel] c8opt_tally, written (not accumulated into)
 *   d_counters_out   DEVICE, [8] uint64 in the order of C8OPT_CNT_* (RECORDS = DROPPED = 0), or NULL
 * Every call shares the one array per device: calls that overlap on the GPU (different streams, or two processes'
 * worth of threads on one device) RACE; order them on one stream or with events.  Results equal the context path's
 * up to the order of the floating-point atomics.  Errors: ARGUMENT (also: too many telescopes, a mode other than
 * tally; message from c8opt_last_error(NULL)), CUDA. */
#define C8OPT_STATIC_MAX_TELESCOPES 8
#define C8OPT_STATIC_SCRATCH_BYTES 1024
int c8opt_tally_static(const c8opt_atmosphere_desc *atmosphere, const float *d_tau, const float *xyzr, int32_t n_tel,
                       const c8opt_segment *d_seg, uint64_t n, uint64_t first_segment_id,
                       const c8opt_run_params *params, c8opt_tally *d_tallies_out, uint64_t *d_counters_out,
                       void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* C8OPT_H */
