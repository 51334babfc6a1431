/*
 * epo.h -- C ABI of the B200-native hot path of EPO (Edge-based Pose Optimization, arxiv 2607.00579).
 *
 * The library evaluates, for every selected directed image pair (s -> t), the edge-based reprojection
 * loss of the paper (Eq. 6-8) and its analytic gradient w.r.t. both cameras' 6-DoF
 * poses, reduces them per camera, and runs the first-order optimisation loop of Alg. 2
 * with Adam on se(3) increments and the paper's pose-change stopping rule
 * entirely on the device.  Every step runs in hand-written CUDA kernels
 * for sm_100a; there is no CPU fallback: without a CUDA device every compute entry point returns
 * EPO_ERR_CUDA.
 *
 * Conventions
 *   poses     world-to-camera [R|t], row-major 3x4, x_cam = R X_w + t
 *   K         (fx, fy, cx, cy) per view; pixel (u,v) is the sample position (no half-pixel offset)
 *   depth     z-depth along the optical axis
 *   gradient  w.r.t. a left perturbation T_c <- Exp(eps_c) T_c, eps = (v, w), translation part first
 *   pairs     (source, target): edge pixels of `source` are projected into `target`  (Eq. 8)
 *
 * Pointers.  Every array argument may be a HOST or a DEVICE pointer (detected with
 * cudaPointerGetAttributes; device pointers must belong to cfg.device).  The caller owns every array
 * it passes; the library copies inputs during the call and never retains caller pointers.  The context
 * owns all device memory it allocates and frees it in epo_destroy.
 * Streams.  All work is enqueued on cfg.stream.  Calls that return data through HOST pointers
 * synchronise that stream before returning; calls given only DEVICE output pointers do not.
 * Errors.  Every function returns an epo_status; nothing throws or aborts.  On error the context is
 * left unchanged (epo_set_views / epo_set_pairs are all-or-nothing); epo_last_error gives a
 * context-owned, NUL-terminated description valid until the next call on that context.
 * Threads.  One context per thread at a time; no global state (device memory comes from a per-context
 * pool; the device's default memory pool and its attributes are never touched).
 * Determinism.  Edge lists, distance fields, pair lists, loss, gradient and every iteration of epo_step
 * are bit-reproducible run to run: all reductions run in a fixed order, without atomics on values.
 */
#ifndef EPO_H_
#define EPO_H_

#include <stdint.h>

#if defined(__GNUC__)
#define EPO_API __attribute__((visibility("default")))
#else
#define EPO_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct epo_ctx epo_ctx;

typedef enum {
  EPO_OK = 0,
  EPO_ERR_INVALID_ARG = 1,   /* NULL required pointer, bad size, non-finite intrinsics, bad pair index ... */
  EPO_ERR_BAD_STATE = 2,     /* call order: set_pairs before set_views, loss_grad/step before both        */
  EPO_ERR_OUT_OF_MEMORY = 3,
  EPO_ERR_CUDA = 4,          /* any CUDA runtime failure, including "no device"                           */
  EPO_ERR_UNSUPPORTED = 5
} epo_status;

typedef struct {
  int32_t n_views, width, height;   /* one resolution per context (all images resized to width 518) */
  float   huber_delta;              /* Huber threshold; 1.0 (paper silent: DESIGN.md reading S1)            */
  float   clamp_start, clamp_end;   /* lambda: 10 -> 6 ...                                                  */
  int32_t clamp_steps;              /* ... linearly over the first 1000 steps               */
  float   lr_max;                   /* 3e-3                                                  */
  int32_t warmup_steps, max_steps;  /* 25, 2000: linear warm-up then cosine decay           */
  float   beta1, beta2, adam_eps;   /* 0.9, 0.999, 1e-8 (reading S10)                       */
  float   eps1, eps2;               /* 0.5, 0.1 degrees                                      */
  int32_t w1, w2;                   /* 25, 50 steps                                          */
  int32_t smooth_window;            /* 1: moving average of width w; 0: raw  */
  int32_t early_stop;               /* 1: epo_step stops at phase 2; 0: phase is tracked but never stops    */
  int32_t dtf_format;               /* 0: fp32 distance fields; 1: fp16 fields (BASELINE.json config 4)    */
  int32_t e_max;                    /* 0: keep all edge pixels; >0: keep entries floor(j n / e_max) (S6)    */
  float   z_min;                    /* 1e-6: depths and projected z at or below it are invalid             */
  int32_t device;                   /* CUDA device ordinal                                                  */
  void*   stream;                   /* cudaStream_t (NULL = legacy default stream)                          */
  int32_t pair_budget;              /* M of the stochastic viewgraph sub-sampling: when
                                       the pair list has more than M pairs, every iteration of epo_step evaluates
                                       a fresh uniform random subset of M pairs.  0 (default) = off: all pairs
                                       every step, as BASELINE.json's configs fix the list.  Paper default 1024. */
  uint64_t subsample_seed;          /* seed of that draw: pair p (position in the list given to epo_set_pairs)
                                       gets, at optimiser step s, the key = output number s * 2^32 + p + 1 of
                                       SplitMix64(subsample_seed); the subset is the M pairs with the smallest
                                       (key, p).  A pure function of (seed, s, p): reproducible, no host draw.  */
  int32_t stop_rule;                /* second-stage stopping rule: 0 (default) pose-based, Eq. 9-10 with w2 / eps2;
                                       1 loss-based (the variant of Tab. 7): the relative loss change
                                       |L_s - L_{s-1}| / |L_{s-1}| stays below eps_loss for w_loss consecutive steps.
                                       The first stage (phase 0 -> 1) is pose-based in both.                        */
  int32_t w_loss;                   /* 100                                                           */
  float   eps_loss;                 /* 5e-4                                                          */
  int32_t joint_phase;              /* 0 (default): epo_step optimises the poses only.  1: also the joint phase's variables
                                       (PAPER.md:64, 78-87): a focal scale per camera, f = f0 (1 + gamma) (Eq. 4), from the
                                       first iteration, and the affine depth Z = Z0 alpha + beta (Eq. 5) of every listed
                                       edge pixel in iterations that start in phase >= 1; AdamW with the loop's learning
                                       rate and weight_decay towards the identity.  An iteration is then three launches:
                                       the fused kernel (which also emits the joint derivatives), the per-camera
                                       reduction (+ gamma), the per-pixel depth update.  May be combined with pair_budget. */
  float   weight_decay;             /* 0.01                                                          */
  void*   mem_pool;                 /* cudaMemPool_t all device memory of the context is taken from (stream-ordered, on
                                       cfg.stream).  NULL (default): the context creates a private pool and destroys it
                                       in epo_destroy.  A caller-owned pool may be shared by consecutive contexts so
                                       that a new one reuses the blocks of a destroyed one; it must outlive them.   */
} epo_config;

/* Fill *cfg with the paper's hyper-parameters (n_views/width/height = 0, device 0, stream NULL). */
EPO_API epo_status epo_config_default(epo_config* cfg);

/* Create a context.  Requires n_views >= 2, 2 <= width,height <= 65535 (16-bit pixel coordinates). */
EPO_API epo_status epo_create(const epo_config* cfg, epo_ctx** out);

/* Free everything the context owns.  NULL-safe. */
EPO_API void epo_destroy(epo_ctx* ctx);

/*
 * Edge extraction ("the edge map E_i via the Canny edge detector [4]"; Alg. 1 l.6):
 * images [N][H][W] 8-bit grey -> edges [N][H][W] u8 (1 = edge, 0), ready for epo_set_views.  Canny's scheme in integer
 * arithmetic: binomial 5x5 smoothing (replicate border, rounded), Sobel 3x3, squared L2 magnitude, non-maximum
 * suppression in four direction sectors, hysteresis with thresholds low <= high on the gradient magnitude (strict:
 * a candidate has |g| > low, a strong one |g| > high; 0 <= low <= high <= 1442).  Border pixels are never edges.
 * The paper states no parameters; the caller chooses the thresholds.  Host or device pointers; N, W, H are the
 * context's.  Synchronises the stream (the hysteresis is iterated until nothing changes).
 */
EPO_API epo_status epo_extract_edges(epo_ctx* ctx, const uint8_t* images, int32_t low, int32_t high, uint8_t* edges);

/* The same from colour images, as the paper extracts its edges from the RGB frames: rgb [N][H][W][3]
 * 8-bit interleaved -> grey by the BT.601 luma in 8-bit fixed point, Y = (77 R + 150 G + 29 B + 128) >> 8 (the paper
 * states no conversion: DESIGN.md reading C7; a grey pixel keeps its value), then epo_extract_edges. */
EPO_API epo_status epo_extract_edges_rgb(epo_ctx* ctx, const uint8_t* rgb, int32_t low, int32_t high, uint8_t* edges);

/*
 * Load the initial estimate G = {K_i, P_i, Z_i} (Eq. 1) and the edge maps E_i
 * (PAPER.md:62), and run the one-time preprocessing (Alg. 1 l.6-7):
 *   - edge-pixel compaction: per view, the list of (u, v, Z) with edges != 0 and finite Z > z_min, in
 *     raster order (v ascending, then u), optionally sub-sampled to e_max entries;
 *   - exact Euclidean distance transform DTF_i (distance in pixels to the nearest pixel with
 *     edges != 0; W+H everywhere if the view has none), fp32 = correctly rounded sqrt of the exact
 *     integer squared distance; optionally rounded (RNE) to fp16.
 * K [N][4]; poses [N][12]; depth [N][H][W] fp32; edges [N][H][W] u8 (non-zero = edge).
 * Resets poses, Adam moments, step counter, phase and traces; keeps no pair list (call epo_set_pairs).
 */
EPO_API epo_status epo_set_views(epo_ctx* ctx, const float* K, const float* poses, const float* depth,
                         const uint8_t* edges);

/*
 * Viewgraph estimation by exhaustive cycle-consistent reprojection (Eq. 2, 117, 380-384, 396) from the
 * CURRENT poses, the intrinsics and the depth maps given to epo_set_views.  For every ordered pair (i, j) the grid of
 * source pixels u = stride/2 + a stride, v = stride/2 + b stride with a usable depth (finite, > z_min) is projected
 * into view j (must land in front of it and inside the image), lifted there with view j's depth at the nearest
 * pixel, and projected back; a point is consistent if its round trip ends less than tau pixels from where it
 * started.  The unordered pair {i, j} is valid if in BOTH directions at least min_frac of the usable points are
 * consistent (paper: tau = 3.0, min_frac = 0.125; the grid stride is not stated, 8 is this library's default).
 *   pairs     [capacity][2] out (nullable when capacity = 0): directed pairs (i, j), (j, i) for valid i < j, ascending;
 *             ready for epo_set_pairs.  Host or device pointer.
 *   n_pairs   out (host): number of directed pairs found; if it exceeds capacity the call fails with
 *             EPO_ERR_INVALID_ARG after setting it, and writes no pairs.
 *   counts    [N][N][2] out, nullable: (consistent, usable) of the cycle i -> j -> i (0, 0 on the diagonal).
 * Synchronises the stream.  Does not change the context (call epo_set_pairs with the result).
 * Depth: always the maps Z0 given to epo_set_views.  With cfg.joint_phase = 1 the refined depth (Z0 alpha + beta) exists
 * only at the listed edge pixels, not on the dense grid this test samples, so it is NOT used here; the current poses are.
 */
EPO_API epo_status epo_build_viewgraph(epo_ctx* ctx, int32_t grid_stride, float tau, float min_frac, int32_t* pairs,
                                       int64_t capacity, int64_t* n_pairs, int32_t* counts);

/*
 * Set the viewgraph as a list of DIRECTED pairs [P][2] = (source, target), P >= 1,
 * indices in [0, N), source != target; duplicates are kept (they weigh twice).  Builds the canonical
 * order (ascending (target, source), stable), the per-target and per-source incidence lists and the
 * work list of the fused kernel.  Resets the optimiser (Adam / AdamW moments, step counter, phase and traces)
 * and nothing else: the CURRENT poses (and joint variables) stay, so a viewgraph re-estimated from refined poses
 * can be installed without losing them.  epo_reset rewinds to the initial poses.
 * Synchronises the stream even when `pairs` is a DEVICE pointer (the exception to the rule at the top of this file): the
 * list is copied to the host, validated there, and the work-item length of the fused kernel is chosen on the host.
 * With cfg.pair_budget > 0 the list may hold at most 524,288 pairs (128 CTAs x 4096 pairs of the selection kernel, which
 * must all be resident at once); a longer list is refused with EPO_ERR_UNSUPPORTED.  Without sub-sampling the only limit
 * is memory.
 */
EPO_API epo_status epo_set_pairs(epo_ctx* ctx, const int32_t* pairs, int64_t n_pairs);

/*
 * One evaluation at the CURRENT poses with clamp `lambda`:
 *   pair_loss[p]  = sum_valid H_delta(min(d, lambda)) / n_valid   (0 if n_valid = 0; Alg. 3 l.11-12)
 *   loss          = mean over the P directed pairs                 (Eq. 6; = 1/2 Eq. 6 for symmetric lists)
 *   grad[c]       = d loss / d eps_c, (v, w) order, n_valid held fixed
 * loss [1] required; pair_loss [P], pair_valid [P] (user pair order) and grad [N][6] are nullable.
 * Does not change poses or optimiser state.
 */
EPO_API epo_status epo_loss_grad(epo_ctx* ctx, float lambda, float* loss, float* pair_loss, int32_t* pair_valid,
                         float* grad);

/*
 * Joint-phase gradients at the CURRENT poses (Eq. 4-5; "in the subsequent joint phase,
 * optimization is extended to include the depth maps"), same loss, same clamp, n_valid held fixed:
 *   g_logf [N]         d loss / d ln f_c, both focal lengths of camera c scaled together (Eq. 4: f = f0 (1 + gamma), so
 *                      d loss / d gamma_c = g_logf[c] / (1 + gamma_c)), as target and as source of its pairs
 *   g_depth [N][H][W]  d loss / d Z_c(u, v) at the edge pixels of the lists (0 elsewhere); with Eq. 5, Z = Z0 alpha + beta:
 *                      d loss / d alpha = Z0 g_depth, d loss / d beta = g_depth
 *   loss [1]           nullable: the loss of this evaluation
 * Evaluates all pairs (no sub-sampling), in ONE pass of the fused kernel; every edge pixel's pairs are then summed in a
 * fixed order (no atomics: bit-reproducible).  Does not change poses, variables or optimiser state (the loop that
 * optimises f and Z is cfg.joint_phase = 1, see epo_step).
 */
EPO_API epo_status epo_loss_grad_joint(epo_ctx* ctx, float lambda, float* loss, float* g_logf, float* g_depth);

/*
 * Run up to n_iters iterations of Alg. 2 on the device without host synchronisation between them:
 *   lambda_s -> loss + gradient -> Adam (lr_s: PAPER.md:121) -> T_c <- Exp(eps_c) T_c
 *   -> theta95^s (Eq. 9-10, 95th percentiles) -> Converged tests (phase 0 -> 1 -> 2).
 * Iterations stop early when the step counter reaches max_steps or, if early_stop, when phase 2 is
 * reached.  iters_done / phase (0, 1, or 2 = second convergence reached) are nullable; host pointers
 * there make the call synchronise.
 * With cfg.pair_budget = M > 0 and more than M pairs, iteration s evaluates the fresh uniform random subset of M
 * pairs that epo_get_pair_subset(ctx, s, ...) reports, drawn by a device kernel inside the loop; loss
 * and gradient are then means over those M pairs.  epo_loss_grad always evaluates the whole list.
 */
EPO_API epo_status epo_step(epo_ctx* ctx, int32_t n_iters, int32_t* iters_done, int32_t* phase);

/* Current poses, [N][12] fp32 (rounded from the fp64 device state) / fp64 (exact). */
EPO_API epo_status epo_get_poses(epo_ctx* ctx, float* poses);
EPO_API epo_status epo_get_poses_f64(epo_ctx* ctx, double* poses);

/* Replace the current poses ([N][12] fp32; NULL = the poses given to epo_set_views) and reset Adam
 * moments, step counter, phase and traces.  Preprocessing and pair lists are kept. */
EPO_API epo_status epo_reset(epo_ctx* ctx, const float* poses);

/*
 * Checkpoint / resume of the optimisation (Alg. 2: everything the loop carries from one iteration to the
 * next).  The blob holds the current poses (fp64), the Adam moments, the step counter, phase and stop flags, the theta95
 * and loss traces, and -- cfg.joint_phase = 1 -- gamma, alpha, beta with their AdamW moments, the current intrinsics and
 * points.  It does NOT hold views, distance fields or pair lists: restore into a context that was given the SAME
 * epo_config, epo_set_views and epo_set_pairs inputs (sizes are checked -- views, resolution, max_steps, joint_phase, pair
 * and edge-pixel counts --, contents are the caller's responsibility).  After epo_set_state the context continues exactly
 * where the exporting one stood: the following iterations are bit-identical to those the exporter would have run.
 *   epo_get_state_size  bytes [1] out (host)
 *   epo_get_state       blob: host or device pointer, capacity >= that size (else EPO_ERR_INVALID_ARG)
 *   epo_set_state       blob as written by epo_get_state of this library version; a blob from another problem or
 *                       configuration is refused with EPO_ERR_INVALID_ARG and the context is left unchanged
 * Both copy on cfg.stream and synchronise it.  The layout is private to the library version (header-checked), native
 * endianness; not an interchange format.
 */
EPO_API epo_status epo_get_state_size(epo_ctx* ctx, int64_t* bytes);
EPO_API epo_status epo_get_state(epo_ctx* ctx, void* blob, int64_t capacity);
EPO_API epo_status epo_set_state(epo_ctx* ctx, const void* blob, int64_t bytes);

/* Joint-phase variables (cfg.joint_phase = 1), all nullable, host or device pointers, fp64: gamma [N]; alpha and beta
 * as [N][H][W] maps (1 and 0 off the edge lists).  The current intrinsics are K0 (1 + gamma), the current depth of a
 * listed edge pixel is Z0 alpha + beta. */
EPO_API epo_status epo_get_joint_variables(epo_ctx* ctx, double* gamma, double* alpha, double* beta);

/* ---- introspection (used by the parity tests and the benchmark) ------------------------------- */
/* The subset of the pair list that iteration `step` of epo_step evaluates (stochastic viewgraph sub-sampling,
 * PAPER.md:465-474, 500; see epo_config.pair_budget): flags [P] in the caller's pair order, 1 = evaluated.  All 1
 * when sub-sampling is off or the list is not longer than the budget.  Computed by the loop's own device kernel. */
EPO_API epo_status epo_get_pair_subset(epo_ctx* ctx, int32_t step, uint8_t* flags /* [P] */);
EPO_API epo_status epo_get_edge_counts(epo_ctx* ctx, int32_t* offsets /* [N+1] exclusive prefix sums */);
EPO_API epo_status epo_get_edge_list(epo_ctx* ctx, int32_t view, uint16_t* uv /* [E][2] (u,v) */, float* z /* [E] */);
EPO_API epo_status epo_get_dtf(epo_ctx* ctx, int32_t view, float* dtf /* [H][W]; fp16 fields are widened */);
EPO_API epo_status epo_get_pair_order(epo_ctx* ctx, int32_t* canonical_pairs /* [P][2] */, int32_t* perm /* [P]:
                              index in the user list of the k-th canonical pair */);
/* loss (at the poses before update s) and theta95 of steps first .. first+count-1 (<= steps done) */
EPO_API epo_status epo_get_trace(epo_ctx* ctx, int32_t first, int32_t count, float* loss, float* theta95);
/* attempted reprojections per evaluation = sum over pairs of the source's edge count */
EPO_API epo_status epo_get_work(epo_ctx* ctx, int64_t* reprojections_per_eval, int64_t* kernel_launches_so_far);

/* Measurement hook (bench.py "roofline"): launch ONLY the fused loss+gradient kernel `reps` times on
 * cfg.stream at the current poses, each launch bracketed by CUDA events recorded on that stream; if
 * flush_l2, a buffer larger than the L2 is overwritten before each launch (outside the events).
 * Returns the mean and minimum launch duration in milliseconds (host pointers, nullable). Synchronises. */
EPO_API epo_status epo_time_loss_grad_kernel(epo_ctx* ctx, float lambda, int32_t reps, int32_t flush_l2,
                                             float* ms_mean, float* ms_min);

/* Measurement hook (bench.py "roofline", the gather ceiling; SURVEY.md 8(d) micro-benchmarks g1 / g2, north_star): the
 * fused kernel's tap stream replayed with NOTHING else.  One launch of the kernel's `record` instantiation writes the
 * texel coordinates of every sample's 2x2 footprint (4 bytes per sample; not valid: a marker) to a scratch buffer; the
 * timed launches then run the same grid (one CTA per work item, same passes and lanes), read those 4 bytes and issue
 * one four-texel gather per valid sample from the same atlas, summing the codes in integers -- no position arithmetic,
 * no square-root table, no loss.  Their duration is what the L1TEX / L2 path needs for this workload's gathers.
 * Arguments and results as for epo_time_loss_grad_kernel.  Allocates and frees its scratch; does not touch the
 * context's state. */
EPO_API epo_status epo_time_gather_ceiling(epo_ctx* ctx, float lambda, int32_t reps, int32_t flush_l2,
                                           float* ms_mean, float* ms_min);

/*
 * Distance transform of ONE edge map without any device-memory allocation (the a-P2 / a-P3 kernels of epo_set_views:
 * PAPER.md:378-379 Alg. 1 l.7, "exact L2 distance transform"; result bit-identical to epo_get_dtf's fp32 field).
 *
 * Who needs it.  epo_set_views takes its work buffers from a memory pool, i.e. it allocates.  Two kinds of caller cannot
 * accept that: (1) a process whose HBM is already owned by its own allocator -- an inference server or a training job
 * that reserved everything at start-up -- where a cudaMalloc from a library either fails or steals the block the host
 * program was about to ask for; (2) a loop with a per-frame deadline, because cudaMalloc and cudaFree synchronise the
 * device.  This call needs no context and allocates nothing, ever: its only work buffer (the row pass's
 * int32 [height][width]) is an array compiled into libepo.so, EPO_EDT_NO_ALLOC_MAX_PIXELS entries = 2 MiB, that every
 * GPU which loads the library carries until the process exits.
 *
 *   d_edges  [height][width] u8, DEVICE pointer, non-zero = edge          (input, caller-owned, read only)
 *   d_dtf    [height][width] fp32, DEVICE pointer: distance in pixels to the nearest edge pixel, width + height
 *            everywhere if there is none                                   (output, caller-owned, fully overwritten)
 *   stream   cudaStream_t of the CURRENT device (NULL = legacy default stream); the two kernels are enqueued on it and the
 *            call returns without synchronising -- d_dtf is ready when that stream reaches this point
 *   err      nullable, err_len bytes: receives a NUL-terminated description when the result is not EPO_OK
 * Runs on the calling thread's current device (it never switches devices); both pointers must belong to it.
 * Limits.  width * height <= EPO_EDT_NO_ALLOC_MAX_PIXELS (the paper's 518 x 392 frames use 39 % of it); anything larger is
 * refused with EPO_ERR_UNSUPPORTED and nothing is launched.  2 <= width, height <= 65535 as for epo_create.
 * First call on each device: looks up that device's address of the built-in array (and, as for any CUDA library, the
 * driver loads the kernels then).  Make that first call during start-up, before the stream is ever put into capture mode;
 * later calls only launch.
 * Sharing.  There is one array per GPU, shared by every call, thread and stream of the process, and it still holds the
 * previous call's row distances.  Nothing has to be cleared (each call overwrites the part it reads before reading it),
 * but two calls that can run at the same time on one GPU -- different streams, or different threads -- overwrite each
 * other's rows and both results are garbage: put them on one stream or order them with events.
 */
#define EPO_EDT_NO_ALLOC_MAX_PIXELS (512 * 1024)
EPO_API epo_status epo_edt_no_alloc(const uint8_t* d_edges, int32_t width, int32_t height, float* d_dtf, void* stream,
                                    char* err, int32_t err_len);

EPO_API const char* epo_last_error(const epo_ctx* ctx);
EPO_API const char* epo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EPO_H_ */
