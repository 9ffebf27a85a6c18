/*
 * spd.h - C ABI of the B200-native single-pulse-detection (SPD) hot path.
 *
 * Method: Adamek & Armour, "Single Pulse Detection Algorithms for Real-time
 * Fast Radio Burst Searches using GPUs" (arXiv:1910.08324).  Citations are
 * PAPER.md:<line> of the paper text plus the equation / section they fall in.
 *
 * What the library computes, for every DM trial d and time sample n of a
 * de-dispersed plane x[n_dm][n_t] (row-major float32, time contiguous):
 *
 *   X_L[n]   = sum_{j=0}^{L-1} x[d, n+j]                       eq. (2)
 *   SNR_L[n] = (X_L[n] - L mu_d) / (sqrt(L) sigma_d)           eq. (4),(5) PAPER.md:69,87-91
 *   Y[d,n]   = max_{L in B} SNR_L[n],  W[d,n] = index of that L eq. (12)
 *
 * over a (possibly incomplete, "lossy") set of boxcar widths B,
 * with long boxcars built from partial sums of shorter ones (eq. 15,
 * PAPER.md:284 eq. 16) and never summed directly, followed by a threshold /
 * peak-candidate stage.
 *
 * Conventions:
 *   - windows are start-aligned: index n is the FIRST sample of the boxcar (eq. 2);
 *   - valid windows only: widths with n + L > n_t are skipped; if no width fits,
 *     Y = -inf and W = -1;
 *   - widths are visited in ascending order with a strict '>' update
 *     (PAPER.md:287), so the smallest width wins exact ties;
 *   - W is the INDEX into the plan's ascending, de-duplicated width table
 *     (spd_plan_get_widths), not the width itself.
 *
 * Every function is thread-safe with respect to distinct plans.  No function
 * throws, exits or synchronises the device unless stated.  All functions
 * returning int return SPD_OK (0) or a negative spd_status; a human-readable
 * message for the calling thread's last error is in spd_last_error_string().
 * There is NO CPU fallback: on a machine without an sm_100 device every
 * compute entry point fails with SPD_ERR_UNSUPPORTED_DEVICE.
 * The library reads no environment variable: kernel choice and work split are plan flags
 * (spd_plan_create_ex) and plan options (spd_plan_set_option).
 *
 * Output-visible artefact of the streaming-tree kernels: the width index rides in the 5 low
 * mantissa bits of the SNR while the maximum is taken, so out_snr differs from the exact float32
 * product by up to 31 ulp (3.7e-6 relative, inside the 1e-4 tolerance of the method's parity
 * rule).  The warp-per-stream kernel (spd_plan_info.tree_kernel == 2) stores those 5 bits as they
 * are - the low mantissa bits of out_snr then equal 31 - out_width; the block-per-stream kernel
 * (tree_kernel == 1) and the any-width-set kernels store them cleared / untouched.
 */
#ifndef SPD_B200_SPD_H_
#define SPD_B200_SPD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPD_VERSION 200

typedef enum spd_status {
    SPD_OK = 0,
    SPD_ERR_INVALID_ARG = -1,        /* NULL pointer, bad size, bad width set */
    SPD_ERR_UNSUPPORTED_DEVICE = -2, /* no CUDA device, or not compute capability 10.x */
    SPD_ERR_ALLOC = -3,              /* host or device allocation failed */
    SPD_ERR_CUDA = -4                /* a CUDA runtime call or kernel launch failed */
} spd_status;

/* Width-set kinds of spd_width_set_generate. */
typedef enum spd_width_kind {
    SPD_WIDTHS_ALL = 0,       /* 1..max_width: the "ideal SPD algorithm" */
    SPD_WIDTHS_POW2 = 1,      /* {1,2,4,...} <= max_width: decimation-in-time set, Alg. 3 */
    SPD_WIDTHS_BOXDIT = 2,    /* eq. (14) PAPER.md:216 with D = 2; param = L_max per iteration */
    SPD_WIDTHS_IGRID = 3,     /* eq. (18) / Table 1; param = depth d */
    SPD_WIDTHS_GEOMETRIC = 4  /* round(r^j), r = param / 1000 (> 1); this project's addition */
} spd_width_kind;

/* Boxcar-separation kinds of spd_separation_generate (the paper's decimated grids). */
typedef enum spd_grid_kind {
    SPD_GRID_EVERY_SAMPLE = 0, /* L_s = 1 for every width */
    SPD_GRID_DIT = 1,          /* Alg. 3: width 2^i at every 2^i-th sample */
    SPD_GRID_BOXDIT = 2,       /* Alg. 1, D = 2: the widths of iteration i (eq. 14, param = L_max)
                                  at every 2^i-th sample ("6,8,10,12 at every second point") */
    SPD_GRID_IGRID = 3         /* param = P layers: the widths of step 2^i at every (2^i / P)-th sample */
} spd_grid_kind;

/* Plan creation flags (spd_plan_create_ex). */
#define SPD_FLAG_FORCE_GENERIC 0x1u     /* use the any-width-set kernels even where a streaming tree applies */
#define SPD_FLAG_BLOCK_TREE 0x2u        /* widths {2^k}: keep the block-per-stream kernel where the warp-per-stream
                                           kernel (9 <= K <= 14 widths, tensor-memory delay lines) would be chosen */
#define SPD_FLAG_GENERIC_WORKSPACE 0x4u /* any-width-set path: use the device-workspace kernels even where the
                                           shared-memory tile kernel applies */
#define SPD_FLAG_WIDTH_U8 0x8u          /* out_width is uint8 [n_dm][n_t] instead of int32 (SURVEY.md sec. 8(f) row f4,
                                           "compact width index": 9 B per sample instead of 12); 255 stands for -1.
                                           SPD_PATH_DYADIC_TREE plans only (else SPD_ERR_INVALID_ARG) */

/* Plan options (spd_plan_set_option). */
#define SPD_OPT_SEGMENTS_PER_ROW 1 /* streaming trees: value >= 1 cuts every DM row into that many independent
                                      streams (each replays its look-ahead once); value 0 restores the automatic
                                      split (warp-per-stream kernel: one piece of the plane's steps per resident warp) */
#define SPD_OPT_HOST_ROWS_PER_BLOCK 2 /* spd_run_host / spd_run_host_candidates: DM rows per staged row block
                                         (value >= 1); value 0 restores the automatic choice (about 256 MiB of rows).
                                         Frees the staging buffers; the next host call allocates them again */

/* Which kernels a plan dispatches to (spd_plan_info.path). */
#define SPD_PATH_DYADIC_TREE 1 /* streaming partial-sum tree, widths {1,2,4,...,2^(K-1)} */
#define SPD_PATH_IGRID_TREE 3  /* the same streaming tree for widths {2^k} U {3 * 2^m} (IGRID depth 1, eq. 18) */
#define SPD_PATH_GENERIC 2     /* any width set: per-row running partial sums, staged per tile in shared memory */
#define SPD_PATH_GRID 4        /* any width set with a boxcar separation per width (spd_plan_create_grid) */

typedef struct spd_plan spd_plan; /* opaque */

/* One detection of the candidate stage (reading A9: the paper only names
 * "peak-finding").  t is the start sample of the boxcar. */
typedef struct spd_candidate {
    int32_t dm;        /* DM-trial (row) index */
    int32_t t;         /* time sample, start-aligned */
    float snr;         /* Y[dm, t] */
    int32_t width_idx; /* W[dm, t] */
} spd_candidate;

typedef struct spd_plan_info {
    int64_t n_dm, n_t;
    int32_t n_widths, max_width;
    int32_t path;               /* SPD_PATH_* */
    int32_t launches_per_run;   /* kernels one spd_run enqueues */
    int32_t threads_per_block;  /* of the dominant kernel */
    int32_t blocks;             /* grid size of the dominant kernel */
    int32_t chunk;              /* time samples per streaming step (dyadic tree), else 0 */
    int32_t segments_per_row;   /* independent streams per DM row (dyadic tree), else 0 */
    int64_t smem_bytes;         /* dynamic shared memory per block of the dominant kernel */
    int64_t workspace_bytes;    /* plan-owned device workspace */
    int64_t activity_bytes;     /* size of the activity map of spd_run_flagged (multiple of 128) */
    int32_t activity_block;     /* time samples of one row covered by one byte of that map */
    int32_t activity_per_row;   /* bytes of that map per DM row */
    int32_t tree_kernel;        /* streaming trees: 1 = one block per stream, 2 = one warp per stream (tensor-memory
                                   delay lines; max_width 256 .. 8192); grid plans that run on the latter: 2; else 0 */
    int32_t piece_chunks;       /* warp-per-stream kernel: steps per piece when the plane's steps are cut, in
                                   row-major order, into one piece per resident warp (pieces may span rows;
                                   segments_per_row is then 0); else 0 */
    int32_t width_bytes;        /* bytes per element of out_width: 4, or 1 with SPD_FLAG_WIDTH_U8 */
    uint32_t flags;             /* the SPD_FLAG_* bits the plan was created with */
} spd_plan_info;

/*
 * spd_width_set_generate - write an ascending width set into out[0..cap).
 *   kind/param : see spd_width_kind.  max_width >= 1 caps every member
 *                (reading A7: max_width is L_end, an upper bound).
 *   out        : HOST array of cap int32 (may be NULL when cap == 0 to query the size).
 *   n_out      : HOST, receives the number of widths of the set (even if > cap).
 * Returns SPD_ERR_INVALID_ARG for unknown kind, bad param, or cap too small
 * (n_out is still written in the last case).
 */
int spd_width_set_generate(int32_t kind, int32_t param, int32_t max_width,
                           int32_t* out, int32_t cap, int32_t* n_out);

/*
 * spd_plan_create - describe one problem: plane shape, width set B, L_end.
 *   out        : HOST, receives the plan (caller owns; free with spd_plan_destroy).
 *   n_dm, n_t  : plane is n_dm rows (DM trials) x n_t time samples, 1 <= n_t <= 2^31-1.
 *   width_set  : HOST array of n_widths boxcar widths in samples (copied, sorted
 *                ascending, de-duplicated).  Error if empty, any width < 1,
 *                any width > max_width, or more than 32768 distinct widths.
 *   max_width  : L_end; must satisfy max_width <= n_t.
 * The plan owns small device tables, the workspace of spd_row_stats and - only for a
 * SPD_PATH_GENERIC plan whose max_width exceeds what a shared-memory tile holds (about
 * 45 000 samples) - a workspace of n_dm*(n_t+1) doubles; spd_plan_info.workspace_bytes
 * reports the total.  Uses the current CUDA device.
 */
int spd_plan_create(spd_plan** out, int64_t n_dm, int64_t n_t,
                    const int32_t* width_set, int32_t n_widths, int32_t max_width);

/* Same, with SPD_FLAG_* bits. */
int spd_plan_create_ex(spd_plan** out, int64_t n_dm, int64_t n_t,
                       const int32_t* width_set, int32_t n_widths, int32_t max_width,
                       uint32_t flags);

/*
 * spd_separation_generate - boxcar separation L_s of each width of a set, by the paper's schedules.
 *   widths : HOST array of n_widths widths (>= 1); out: HOST array of n_widths int32.
 * Returns SPD_ERR_INVALID_ARG for an unknown kind, a bad param, or (SPD_GRID_DIT) a width
 * that is not a power of two.
 */
int spd_separation_generate(int32_t kind, int32_t param, const int32_t* widths, int32_t n_widths, int32_t* out);

/*
 * spd_plan_create_grid - a plan whose width k is evaluated only at the time samples that are
 * multiples of separations[k] (the paper's lossy grids - "wider pulses ...
 * at every D^(i) point"; sensitivity eq. (27)-(31)).
 *   width_set   : HOST, n_widths widths, STRICTLY ascending, each in [1, max_width];
 *   separations : HOST, n_widths powers of two that do not decrease with the width.
 * spd_run / spd_run_flagged / spd_run_host on such a plan write one merged full-resolution
 * plane: out_snr[d,n] = max over the widths whose grid contains n (and whose window fits,
 * reading A3), out_width the index of that width; -inf / -1 where no width's grid contains n
 * (only if separations[0] > 1).  Limits: max_width <= 45057, n_widths <= 1024.  A set {1, 2, 4, ..., 2^(K-1)}
 * with 9 <= K <= 14, and the IGRID depth-1 set {2^k} U {3 * 2^m} over the same range when the two widths of an
 * octave share a separation (SPD_GRID_IGRID), run on the warp-per-stream tree kernel
 * (spd_plan_info.tree_kernel == 2), where the keys of a level are formed on its grid points only.  The BoxDIT
 * algorithm itself (Alg. 1) - the widths of SPD_WIDTHS_BOXDIT with L_max = 4, 8, 16 or 32 (the
 * last iteration may be cut by max_width) on the separations of SPD_GRID_BOXDIT with the same L_max, at most 11
 * iterations and 256 widths, n_t % 4 == 0 - runs on a streaming kernel of its own (spd_boxdit.cu: all iterations
 * of a chunk in one block, decimated series and longest boxcars in shared memory; spd_plan_info.threads_per_block
 * == 256, chunk == 4096).  Other sets run on a shared-memory tile kernel (threads_per_block == 1024).
 * spd_plan_info.path is SPD_PATH_GRID.  Errors as spd_plan_create plus the conditions above.
 *
 * spd_plan_create_grid_ex: the same with creation flags; SPD_FLAG_FORCE_GENERIC keeps the plan on the tile kernel
 * (no tree, no BoxDIT kernel); the other flags are refused.
 */
int spd_plan_create_grid(spd_plan** out, int64_t n_dm, int64_t n_t,
                         const int32_t* width_set, const int32_t* separations, int32_t n_widths,
                         int32_t max_width);
int spd_plan_create_grid_ex(spd_plan** out, int64_t n_dm, int64_t n_t,
                            const int32_t* width_set, const int32_t* separations, int32_t n_widths,
                            int32_t max_width, uint32_t flags);

/* Frees the plan and everything it owns.  NULL is allowed. */
void spd_plan_destroy(spd_plan* plan);
/* The same under north_star's name (spd_plan_create / spd_run / spd_destroy). */
void spd_destroy(spd_plan* plan);

/*
 * spd_plan_set_option - change one SPD_OPT_* setting of a plan; call it between runs (not while a
 * run of this plan is being enqueued from another thread).  Returns SPD_ERR_INVALID_ARG for an
 * unknown option, a value out of range, or an option that does not apply to the plan's path.
 */
int spd_plan_set_option(spd_plan* plan, int32_t option, int64_t value);

/* Copies the plan's ascending width table to out[0..*n) (HOST); *n receives the count.
 * out may be NULL to query the count. */
int spd_plan_get_widths(const spd_plan* plan, int32_t* out, int32_t* n);

/* Fills *info (HOST). */
int spd_plan_get_info(const spd_plan* plan, spd_plan_info* info);

/*
 * spd_run - the hot path on DEVICE buffers.
 *   plane      : DEVICE, float32 [n_dm][n_t] row-major, 16-byte aligned, read only.
 *   mean, sigma: DEVICE, float32 [n_dm]; per-DM mu(x) and sigma(x) of eq. (5).
 *                sigma > 0 and finite inputs are preconditions (not checked).
 *   out_snr    : DEVICE, float32 [n_dm][n_t], fully overwritten with Y.
 *   out_width  : DEVICE, int32 [n_dm][n_t] (uint8 [n_dm][n_t] for a plan created with SPD_FLAG_WIDTH_U8),
 *                fully overwritten with W.
 *   cuda_stream: a cudaStream_t (NULL = default stream).  The call only
 *                enqueues work; it never synchronises.
 * Buffers are owned by the caller and must not alias.  A SPD_PATH_DYADIC_TREE
 * plan is read-only during the call (concurrent runs on different streams are
 * allowed); a SPD_PATH_GENERIC plan with a workspace (see spd_plan_create) runs one call
 * at a time.
 */
int spd_run(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
            float* out_snr, void* out_width, void* cuda_stream);

/*
 * spd_find_candidates - threshold + 1-D peak stage (row a8; reading A9):
 * (d, n) is reported iff Y[d,n] >= threshold and Y[d,n] > Y[d,n-1] and
 * Y[d,n] >= Y[d,n+1] (row ends compare against -inf).
 *   out_snr, out_width : DEVICE planes produced by spd_run.
 *   list      : DEVICE array of `capacity` spd_candidate; order unspecified.
 *   n_found   : DEVICE int64; receives the number of peaks found, which may
 *               exceed capacity (overflow: only the first `capacity` appends are stored).
 * Asynchronous on cuda_stream.
 */
int spd_find_candidates(const spd_plan* plan, const float* out_snr, const void* out_width,
                        float threshold, spd_candidate* list, int64_t capacity,
                        int64_t* n_found, void* cuda_stream);

/*
 * spd_run_flagged - spd_run with row a8's threshold test fused into the same pass.
 * Besides Y and W it fills the caller's activity map: byte [d * activity_per_row + b]
 * is non-zero if any Y[d, n] with b * activity_block <= n < (b+1) * activity_block may
 * reach `threshold` (it is zero only if none does), so the candidate stage can skip the
 * rest of the plane.  The plane is still read once and Y, W written once.
 *   threshold : candidate threshold in SNR units (the value later given to
 *               spd_find_candidates_flagged, or any lower one).
 *   activity  : DEVICE, uint8 [spd_plan_info.activity_bytes], 16-byte aligned, fully overwritten.
 * Other arguments, asynchrony and aliasing rules as spd_run.  A SPD_PATH_GENERIC plan
 * marks every block active.
 */
int spd_run_flagged(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                    float* out_snr, void* out_width, float threshold, uint8_t* activity,
                    void* cuda_stream);

/*
 * spd_find_candidates_flagged - spd_find_candidates restricted to the blocks marked in
 * `activity` (written by spd_run_flagged on the same out_snr with a threshold <= this
 * one).  Same rule, same outputs; samples of unmarked blocks are never candidates
 * because their Y is below the threshold.
 */
int spd_find_candidates_flagged(const spd_plan* plan, const float* out_snr, const void* out_width,
                                const uint8_t* activity, float threshold, spd_candidate* list,
                                int64_t capacity, int64_t* n_found, void* cuda_stream);

/*
 * spd_row_stats - per-DM mean and standard deviation of the plane, the inputs of eq. (4)/(5)
 * (sec. 4.6.2: Chan et al. streaming algorithm with point-wise outlier
 * rejection).  Pass 0 uses every sample of a row; each of the n_reject_passes further passes
 * uses the samples with |x - mean| <= clip_sigma * sigma of the previous pass (float32
 * comparison).  sigma is the population standard deviation (ddof 0).  With
 * n_reject_passes == 0 this is the plain per-row mean / sigma of reading A6.
 *   plane       : DEVICE, float32 [n_dm][n_t] (any alignment; 16-byte aligned rows are faster).
 *   clip_sigma  : rejection threshold in sigmas (> 0 when n_reject_passes > 0; the paper's
 *                 comparison used 2).
 *   mean, sigma : DEVICE, float32 [n_dm], overwritten.  A row whose samples are all rejected
 *                 keeps its previous estimate.
 * Asynchronous on cuda_stream; uses a plan-owned workspace (one call at a time per plan).
 * Each pass reads the plane once.
 */
int spd_row_stats(const spd_plan* plan, const float* plane, float clip_sigma, int32_t n_reject_passes,
                  float* mean, float* sigma, void* cuda_stream);

/*
 * spd_width_sigma - standard deviation per boxcar width measured on the plane (SURVEY.md sec. 8(f1),
 * "we calculate the standard deviation only for boxcar filters of width that are equal to
 * a powers of two.  We then interpolate ... for all intermediate boxcar widths"; reading A17).
 *   plane   : DEVICE [n_dm][n_t] float32.
 *   mean    : DEVICE [n_dm] float32, the per-row mean (e.g. from spd_row_stats); used as the shift of
 *             the variance sums only.
 *   sigma_w : DEVICE [n_dm][n_widths] float32, written: sigma of the sums of 2^j consecutive samples
 *             (population standard deviation over the floor(n_t / 2^j) aligned groups) at widths
 *             2^j, linear in the width in between, sqrt(width) beyond the last level with two groups.
 * Asynchronous on cuda_stream; uses a plan-owned workspace (one call per plan at a time).
 */
int spd_width_sigma(const spd_plan* plan, const float* plane, const float* mean, float* sigma_w,
                    void* cuda_stream);

/*
 * spd_run_sigma_w - spd_run with SNR_L = (X_L - L mean) / sigma_w[d][L's index] (eq. 4, PAPER.md:69,
 * with the measured sigma(X_L) of spd_width_sigma in place of eq. 5's sqrt(L) sigma).
 * For every plan except SPD_PATH_GENERIC plans on the device-workspace kernels (max_width above about 45 000, or
 * SPD_FLAG_GENERIC_WORKSPACE) and SPD_FLAG_WIDTH_U8 plans, which return SPD_ERR_INVALID_ARG.  Other arguments
 * (alignment included) as spd_run.
 */
int spd_run_sigma_w(const spd_plan* plan, const float* plane, const float* mean, const float* sigma_w,
                    float* out_snr, void* out_width, void* cuda_stream);

/*
 * spd_run_host - the same hot path on HOST buffers (end-to-end entry point):
 * copies row blocks of the plane to the device, runs the kernels and copies
 * Y and W back, overlapping copies and kernels on internal streams.
 *   plane, out_snr, out_width : HOST (pinned memory recommended), shapes as spd_run.
 *   mean, sigma               : HOST float32 [n_dm].
 * Blocks until the results are in out_snr / out_width.  Any plan; device staging
 * buffers are allocated on first use and kept in the plan (hence the non-const plan).
 * On an error in the middle of the run the internal streams are drained before returning,
 * so no copy into the caller's buffers is in flight afterwards.
 */
int spd_run_host(spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                 float* out_snr, void* out_width);

/*
 * Output separated by iteration (eq. 12: "We have chosen to separate the output by iteration,
 * that is the output for ith iteration is Y^i[n] = max_{L in B^i} SNR(X^i_L[n])", with W^i the width that
 * produced it; Y^i has N / D^(i) samples).  For a plan with boxcar separations (spd_plan_create_grid) an
 * ITERATION is a run of consecutive widths that share one separation s: BoxDIT iteration i (s = 2^i, the widths
 * of eq. 14), one width per iteration on the DIT grid, the widths of one step of IGRID with P layers.  Point m
 * of iteration i's plane is sample n = s m of the row, m < n_points = ceil(n_t / s):
 *     Y^i[d][m] = max over the iteration's widths L with s m + L <= n_t of SNR_L[s m],  W^i[d][m] = its index
 * in the plan's width table (-inf / -1 where none fits, reading A3).  spd_run's merged plane (reading A16) is
 * the maximum of these over the iterations whose grid holds a sample.
 *
 * spd_plan_get_iterations: HOST arrays of cap entries (each may be NULL); *n_iter receives the count (<= 32).
 * spd_run_iterations: out_snr_iter (float32) and out_width_iter (int32) are DEVICE buffers holding the
 *   iterations' planes one after the other, iteration i as [n_dm][n_points[i]] row-major at element offset
 *   n_dm * (n_points[0] + ... + n_points[i-1]); plane, mean, sigma as spd_run (eq. 5's sqrt(L) sigma).
 *   Asynchronous on cuda_stream.  Any grid plan, one pass over the plane and one launch for all iterations: BoxDIT
 *   plans (Alg. 1's widths on Alg. 1's grids) on the BoxDIT streaming kernel, whose levels are the iterations;
 *   every other grid on the shared-memory tile kernel of the any-width-set path.
 * Both return SPD_ERR_INVALID_ARG for a plan without separations.
 */
int spd_plan_get_iterations(const spd_plan* plan, int32_t cap, int32_t* n_iter, int32_t* first_width,
                            int32_t* n_widths, int32_t* separation, int64_t* n_points);
int spd_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                       float* out_snr_iter, int32_t* out_width_iter, void* cuda_stream);

/*
 * spd_row_stats_static - spd_row_stats for callers that may not allocate (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): no plan, and the call enqueues kernels and one memset on
 * cuda_stream and nothing else - no cudaMalloc, cudaFree or allocating library routine, on the first call
 * or later.  Same kernels, same arithmetic and the same work split rule as spd_row_stats (PAPER.md:720-726,
 * reading A14): results agree with it to rounding, and exactly when both cut a row into the same parts.
 *   plane            : DEVICE float32 [n_dm][n_t], row-major (16-byte aligned with n_t % 4 == 0 takes the
 *                      vectorised loads; any alignment is accepted).
 *   mean, sigma      : DEVICE float32 [n_dm], written (also read between the rejection passes).
 *   clip_sigma, n_reject_passes : as spd_row_stats (0 <= n_reject_passes <= 64; 0 = all samples, reading A6).
 * The scratch (partial moments per row part, per-row state) is a fixed array in the library's device image,
 * SPD_STATIC_SCRATCH_BYTES (1.7 MiB), which every GPU that loads the library holds until exit.  Limits:
 * n_dm <= SPD_STATIC_MAX_ROWS, else SPD_ERR_INVALID_ARG with a message naming the limit (n_t is unlimited:
 * rows are cut into at most SPD_STATIC_MAX_PARTIALS / n_dm parts).  All calls on a device share that one
 * array: it keeps the last call's contents (what must start at zero is cleared by the call itself), and two
 * calls that overlap on the GPU - different streams without an ordering between them - race on it; serialise
 * them (one stream, or events).  Asynchronous; SPD_ERR_UNSUPPORTED_DEVICE without an sm_100 device.
 */
#define SPD_STATIC_MAX_ROWS 8192
#define SPD_STATIC_MAX_PARTIALS 65536
#define SPD_STATIC_SCRATCH_BYTES (24 * SPD_STATIC_MAX_PARTIALS + 24 * SPD_STATIC_MAX_ROWS)
int spd_row_stats_static(const float* plane, int64_t n_dm, int64_t n_t, float clip_sigma,
                         int32_t n_reject_passes, float* mean, float* sigma, void* cuda_stream);

/*
 * spd_row_stats_converge - spd_row_stats "repeated until convergence": rejection
 * passes go on, per DM row, until one changes neither the mean nor sigma by more than
 * rel_tol * sigma(previous pass), or max_reject_passes are done (1 <= max_reject_passes <= 64,
 * rel_tol >= 0).  The test runs on the device; a row that has converged is skipped by the later
 * passes (its plane samples are not read again), so over-provisioning max_reject_passes costs
 * kernel launches only.
 *   n_passes : DEVICE int32 [n_dm] (may be NULL): rejection passes done for each row.
 * Other arguments and conventions as spd_row_stats.
 */
int spd_row_stats_converge(const spd_plan* plan, const float* plane, float clip_sigma, int32_t max_reject_passes,
                           float rel_tol, float* mean, float* sigma, int32_t* n_passes, void* cuda_stream);

/*
 * spd_cluster_candidates - 2-D (DM x time) peak stage over the 1-D candidates (SURVEY.md sec. 8(f)
 * row f4; the paper names it only: "candidates are selected using a peak-finding algorithm",
 * PAPER.md:708, 742).  Reading A18 (this project's definition): candidate (d, n) with best width
 * L = widths[width_idx] is kept iff no sample of the window |d' - d| <= dm_radius, |n' - n| <= L
 * (clipped to the plane) has a larger out_snr and none that comes earlier in (d, n) order has an
 * equal one.
 *   out_snr   : DEVICE plane written by spd_run*.
 *   list_in   : DEVICE, the candidates of spd_find_candidates(_flagged); n_in : DEVICE int64, their
 *               count as that call wrote it (values above capacity_in are clamped to it).
 *   dm_radius : >= 0, half-height of the window in DM trials.
 *   list_out  : DEVICE array of capacity_out spd_candidate (must not alias list_in); n_out : DEVICE
 *               int64, receives the number kept (may exceed capacity_out: overflow as spd_find_candidates).
 * Asynchronous on cuda_stream; order of list_out unspecified.
 */
int spd_cluster_candidates(const spd_plan* plan, const float* out_snr, const spd_candidate* list_in,
                           const int64_t* n_in, int64_t capacity_in, int32_t dm_radius, spd_candidate* list_out,
                           int64_t capacity_out, int64_t* n_out, void* cuda_stream);

/*
 * spd_run_host_candidates - end-to-end entry point that returns what a pipeline consumes: the
 * candidate list.  Row blocks of the HOST plane go to the device, every block runs the hot path with
 * the fused threshold test and the 1-D candidate stage (rows a1-a8), the 2-D peak stage runs over
 * the whole list (row f4; skipped when dm_radius < 0), and only the list comes back.
 *   plane, mean, sigma : HOST, as spd_run_host (pinned memory recommended).
 *   list      : HOST array of `capacity` spd_candidate, in unspecified order; n_found : HOST int64,
 *               the number found, which may exceed capacity (then only `capacity` are stored; with
 *               the 2-D stage an overflow of the 1-D list makes the result incomplete - n_1d, if not
 *               NULL, receives the 1-D count so that the caller can tell).
 * Needs the whole plane's out_snr on the device when dm_radius >= 0 (windows cross row blocks):
 * 4 B per sample of device memory, allocated on first use and kept; dm_radius < 0 needs two row
 * blocks only.  Blocks until the list is in host memory.
 */
int spd_run_host_candidates(spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                            float threshold, int32_t dm_radius, spd_candidate* list, int64_t capacity,
                            int64_t* n_found, int64_t* n_1d);

/* Message describing the calling thread's most recent error ("" if none). */
const char* spd_last_error_string(void);

/* Library version (SPD_VERSION). */
int spd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPD_B200_SPD_H_ */
