/*
 * optflow.h -- C-ABI of liboptflow.so: the dense optical-flow solve of arxiv/paper_1306_2461
 * (Gautier & Aider, "Real-time planar flow velocity measurements using an optical flow algorithm
 * implemented on GPU"), written from scratch as CUDA kernels for NVIDIA B200 (sm_100a).
 *
 * The method (sec. 2.4): a local, iterative, gradient-based, windowed sum-of-squared-
 * differences registration of the Lucas-Kanade family, one vector per pixel, solved by Gauss-Newton
 * iterations coarse-to-fine over an image pyramid from a zero initial guess.  The step list is
 * BASELINE.json:5; every point the paper leaves open follows the readings D1..D23 in DESIGN.md.
 *
 * Conventions
 *   - images: H rows x W columns, row-major, dense (pitch == width); pixel (x,y) = (column,row).
 *   - flow (u,v) in pixels per frame pair with  I2(x+u, y+v) ~= I1(x,y)  (D1).
 *   - "device pointer" = memory of the CUDA device that was current at of_create; "host pointer"
 *     = ordinary host memory.  Streams are cudaStream_t passed as void* (NULL = default stream).
 *   - every int-returning call returns OF_OK (0) or a negative of_status; of_last_error() gives the
 *     text of the calling thread's last failure.  No C++ exception crosses this boundary.
 *   - a handle is not thread-safe; distinct handles are independent.  All scratch belongs to the handle, so only ONE solve of a
 *     handle is in flight at a time: a call on another stream than the previous one is ordered after it (an event wait that the
 *     library enqueues itself); use several handles for concurrent solves.  There is no CPU fallback: without a usable CUDA
 *     device of_create fails.
 *   - alignment: u, v must be 16-byte aligned (the last pass stores vectors), I1, I2 to their element size; a pointer that is
 *     not is rejected with OF_ERR_INVALID_ARG.
 *   - results are bit-reproducible for the same inputs (no atomics in any sum).
 */
#ifndef OPTFLOW_H_
#define OPTFLOW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct of_context *of_handle;

enum of_window { OF_WINDOW_BOX = 0, OF_WINDOW_GAUSSIAN = 1 };
enum of_status { OF_OK = 0, OF_ERR_INVALID_ARG = -1, OF_ERR_ALLOC = -2, OF_ERR_CUDA = -3, OF_ERR_STATE = -4 };
enum of_dtype { OF_DTYPE_F32 = 0, OF_DTYPE_U8 = 1, OF_DTYPE_U16 = 2 };
enum of_stream_mode { OF_STREAM_CONSECUTIVE = 0, OF_STREAM_PAIRS = 1 };

#define OF_MAX_LEVELS 12
#define OF_MAX_WINDOW_RADIUS 16
#define OF_TIMELINE_MAX 4096
#define OF_STATIC_MAX_PIXELS 16777216   /* of_field_minmax_static: largest field, 4096 x 4096 */
#define OF_STATIC_SCRATCH_BYTES 33024   /* its static device array: 256 + 8 * OF_STATIC_MAX_PIXELS / 4096 */

/* ---------------------------------------------------------------------------------------------
 * The three calls named by the north_star (BASELINE.json:5).
 * ------------------------------------------------------------------------------------------- */

/* Create a solver for width x height images ("two inputs to the algorithm, besides image size":
 * n_lev and n_iter; interrogation-window radius).
 *   levels        >= 1, number of pyramid images INCLUDING the base (D3; eq. 1); level
 *                 l+1 has size ((W_l+1)/2, (H_l+1)/2).
 *   window_radius R in [1, OF_MAX_WINDOW_RADIUS]: box of (2R+1)^2 equal weights, or for
 *                 OF_WINDOW_GAUSSIAN a separable Gaussian truncated at R with sigma = R/3 (D11).
 *   iterations    >= 1 Gauss-Newton iterations per level (D16: no convergence test).
 * The coarsest level must be at least (2R+1) x (2R+1).  Allocates all scratch on the current CUDA
 * device (about 12 fp32 planes of the base size); launches no kernel.  Returns NULL on failure. */
of_handle of_create(int width, int height, int levels, int window_radius, int iterations, int window_type);

/* Solve one pair.  I1, I2: device pointers, fp32, dense H x W, read-only.  u, v: device pointers,
 * fp32, dense H x W, write-only (the initial guess is always zero).  Everything is
 * enqueued on `stream`; the call never synchronises and allocates no device memory (the launch sequence is replayed as a CUDA
 * graph: the first call with a new set of pointers captures it, later calls replay it; beyond 64 cached sets the least recently
 * used graph is re-parameterised in place).  Steps enqueued (DESIGN.md
 * "Kernels"): pyramid build of both images, zero field at the coarsest level, then per level
 * coarse-to-fine: x2 flow upsampling, and `iterations` x { warp + gradients + five products +
 * horizontal window sum ; vertical window sum + damped 2x2 solve + in-place (u,v) update }. */
int of_compute(of_handle h, const float *I1, const float *I2, float *u, float *v, void *stream);

/* Destroy; waits for the handle's own streams.  NULL is a no-op. */
void of_destroy(of_handle h);

/* ---------------------------------------------------------------------------------------------
 * Integer camera frames (8-bit camera; BASELINE.json:8-11).  Same as of_compute but
 * I1, I2 are device pointers to dense uint8 / uint16 frames, converted exactly (no scaling, D17)
 * on the device.
 * ------------------------------------------------------------------------------------------- */
int of_compute_u8(of_handle h, const uint8_t *I1, const uint8_t *I2, float *u, float *v, void *stream);
int of_compute_u16(of_handle h, const uint16_t *I1, const uint16_t *I2, float *u, float *v, void *stream);

/* ---------------------------------------------------------------------------------------------
 * Throughput mode: TWO independent pairs in one launch ("the computation of a velocity field is independent of all
 * other computations"; the stream of image pairs).  Pair a is solved with handle ha, pair b with handle hb --
 * two different handles created with the same arguments on the same device, each providing the scratch of its pair -- exactly as
 * of_compute / of_compute_u8 / of_compute_u16 would solve them (dtype = an of_dtype value for all four frames; same pointer rules;
 * both results are bit-identical to the single calls), but by one persistent kernel in which the passes of the two pairs alternate
 * and the grid-wide barrier of one pair is waited for behind a pass of the other (csrc/of_solve_dual.cuh).  What it buys is pairs
 * per second; what it costs is latency: neither field is complete before the launch ends.  Enqueue only, no allocation; both
 * handles count as busy until it ends (a later call on either is ordered after it).  If the handles cannot share a launch (different
 * sizes, parameters or conditioning, a mask, of_set_hoist(1) or of_set_persistent(0) on either), the two pairs are solved one after the other by
 * two ordinary solves, with the same results.  The validity mask of each pair is its handle's (of_get_validity).
 * ------------------------------------------------------------------------------------------- */
int of_compute_dual(of_handle ha, of_handle hb, int dtype, const void *I1a, const void *I2a, float *ua, float *va,
                    const void *I1b, const void *I2b, float *ub, float *vb, void *stream);

/* Text of the calling thread's last error ("" if none).  Never NULL. */
const char *of_last_error(void);

/* Conditioning of the 2x2 solve (D14, D15): relative Levenberg damping lam = eps_rel*tr(G)/2
 * (default 1e-3) and per-iteration increment clamp in pixels (default 3, cf. eq. 1).
 * eps_rel >= 0, max_step_px > 0. */
int of_set_conditioning(of_handle h, float eps_rel, float max_step_px);

/* Local equalisation pre-filter (eq. 2: "mandatory for experimental images"): every frame
 * is replaced by (I - local mean) / local standard deviation over the in-image part of a (2*radius+1)^2
 * box before the pyramid is built; 0 where the local variance is not positive.  Fused with the frame
 * conversion (it replaces that kernel).  radius 0 (default) switches it off; the paper uses 5. */
int of_set_equalisation(of_handle h, int radius);

/* Obstacle mask ("using masks to avoid computations over obstacles or side walls").
 * mask_host: HOST pointer to height rows of row_stride (>= width) bytes, non-zero = fluid, 0 = obstacle;
 * copied and preprocessed by this call (the caller keeps ownership); NULL removes the mask.  A set-up
 * call: it synchronises the device and must not overlap a solve on this handle.  Readings (DESIGN.md
 * M1-M5): an obstacle pixel has zero weight in every window sum and carries no vector (u = v = 0,
 * valid = 0, at every level); a coarse pixel is an obstacle iff all its in-image children are; the
 * images themselves are not altered.  Tiles and tasks that neither hold nor feed a fluid pixel are
 * skipped and the remaining work is re-balanced over the SMs.  Returns OF_OK or an error code. */
int of_set_mask(of_handle h, const uint8_t *mask_host, int row_stride);

/* Replay the per-pair launch sequence as a CUDA graph (default on).  The graph is re-captured when
 * the caller's pointers change. */
int of_set_graph(of_handle h, int enable);

/* Run the whole solve of a pair (all levels, all iterations, flow hand-down) as ONE persistent
 * cooperative kernel whose CTAs alternate the two iteration kernels' passes across a grid barrier
 * (default on: a kernel boundary costs more than a coarse-level pass).  With 0, every pass is its own
 * launch.  Both give bit-identical results. */
int of_set_persistent(of_handle h, int enable);

/* Iterate the coarse pyramid levels in fused form (default on; "coarse-to-fine": a further level
 * should cost ~2 %).  At a level whose image can be cut into at most one tile per SM that fits in shared memory together with its
 * window halo, a CTA forms the products, both window sums and the solve of its tile without leaving the SM and the field is double
 * buffered, so an iteration needs one grid barrier instead of two and the five summed planes of that level stay in shared memory.
 * Every value is formed by the same instructions as in the two-pass form: results are bit-identical with 0 and with
 * of_set_persistent(h, 0).  Levels with an obstacle mask keep the two-pass form.  Synchronises the device (a set-up call). */
int of_set_fused(of_handle h, int enable);

/* Hoist what does not change within a pyramid level out of its iterations (default off).  Ix, Iy are
 * differences of I1 alone (reading D9 of DESIGN.md), so the planes IxIx, IxIy, IyIy -- and their
 * window sums, the 2x2 matrix of the paper's local least-squares problem, PAPER.md:59-63 -- are the
 * same in every iteration of a level; only IxIt, IyIt follow the warped I2.  With 1, the per-iteration
 * product kernel forms and writes all five planes in the first iteration of a level and the two
 * It planes afterwards (60 instead of 72 B per pixel-iteration; SURVEY.md 8(f) note f5).  The
 * arithmetic of every value is unchanged: results are bit-identical to the default.  Off by default
 * because BASELINE.json's north_star states the five-plane form per iteration.  The first call with 1
 * allocates three more planes (the level's window sums a, b, c) on the handle's device.  Applies to the
 * persistent solve kernel; with of_set_persistent(h, 0) every pass forms all five planes.  Returns OF_OK
 * or an error code (OF_ERR_CUDA if the allocation fails; the setting is then unchanged). */
int of_set_hoist(of_handle h, int enable);

/* Validity bytes (1 = tr(G) > 0, D14) of the last iteration at level 0 of the last solve: copies
 * H x W bytes into the device buffer mask_dev, on `stream`. */
int of_get_validity(of_handle h, uint8_t *mask_dev, void *stream);

/* Size of pyramid level `level`. */
int of_level_size(of_handle h, int level, int *width, int *height);

/* Number of kernel launches (graph kernel nodes included) enqueued by the last of_compute* call:
 * persistent mode max(levels-1, 1) (frame conversion fused into the first pyramid step) + 1 (solve); otherwise
 * + levels-1 hand-downs and 2*levels*iterations iteration kernels instead of the solve. */
int of_last_launch_count(of_handle h);

/* Test / profiling hooks.  State is that left by the last of_compute* on this handle.
 * of_get_debug_plane copies one dense fp32 plane of level `level` into out_dev:
 *   which 0,1: pyramid image of I1 / I2;  2,3: final u / v of that level (level 0: the field before
 *   its last iteration);  4..8: the five horizontally summed product planes left by the last
 *   products kernel (valid only for the level it ran on);  9: det = a*c - b^2 (level 0 only). */
int of_get_debug_plane(of_handle h, int level, int which, float *out_dev, void *stream);
/* Run ONE kernel of the iteration, `repeat` >= 1 times back to back, on the handle's internal state
 * of `level` (for per-kernel timing and intermediate parity):
 *   which 0: warp + gradients + products + horizontal sum (K2);  1: vertical sum + solve + update (K3,
 *   in place on the internal field). */
int of_run_step(of_handle h, int level, int which, int repeat, void *stream);

/* Launch ONLY the persistent solve kernel, `repeat` times,
 * on the pyramids left by the last of_compute*; the level-0 result is discarded into scratch.  For
 * timing the dominant kernel with CUDA events and for ncu. */
int of_run_solve(of_handle h, int repeat, void *stream);
/* The same for the two-pair kernel of of_compute_dual (pyramids left by the last solves of ha and hb); fails with OF_ERR_STATE
 * if the handles cannot share a launch.  With the timeline hook on for ha, of_solve_timeline(ha) returns the stamps of that kernel:
 * same positions as for one pair, each pass interval covering the pass of both pairs (the barrier intervals are empty). */
int of_run_solve_dual(of_handle ha, of_handle hb, int repeat, void *stream);

/* Timeline of the persistent solve kernel (profiling hook; the in-kernel analogue of a launch list).
 * While the hook is on, thread 0 of every CTA stores its SM cycle counter, relative to the CTA's start,
 * at every phase boundary (after a CTA-wide barrier; %globaltimer is refreshed too coarsely): start; per level coarse-to-fine { hand-down end, grid barrier end } (not for the
 * coarsest); per iteration { K2 pass end, grid barrier end, K3 pass end, grid barrier end }.
 * Copies the stamps of the last profiled solve to out_host (HOST pointer, may be NULL): those of CTA
 * `cta`, or for cta < 0 the maximum over CTAs (when the last CTA reached each boundary).  Synchronises
 * the device.  Then switches the hook on/off for the following solves.  Returns the number of entries
 * written (0 if the hook was off), or a negative status. */
int of_solve_timeline(of_handle h, int enable, int cta, unsigned long long *out_host, int max_entries);

/* ---------------------------------------------------------------------------------------------
 * Integral quantity of a field on the device (eq. 3: recirculation-bubble surface
 * S_bubble = share of the available vectors with v_x <= T_v, T_v = (min + max)/2 of the mean field; "such
 * an integral value could ... be used as an input in a feedback loop").  All pointers are device pointers
 * to dense H x W arrays; valid_dev (may be NULL = every vector available) is a validity mask as returned
 * by of_get_validity.  Asynchronous on `stream`; integer atomics only, so results are exact.
 * ------------------------------------------------------------------------------------------- */
/* sum_dev += field_dev (running sum for the mean field). */
int of_field_accumulate(of_handle h, float *sum_dev, const float *field_dev, void *stream);
/* out_dev[0] = min, out_dev[1] = max of field_dev over the available vectors (NaN ignored). */
int of_field_minmax(of_handle h, const float *field_dev, const uint8_t *valid_dev, float *out_dev, void *stream);
/* out_dev[0] = number of available vectors with vx <= threshold, out_dev[1] = number of available vectors. */
int of_bubble_count(of_handle h, const float *vx_dev, const uint8_t *valid_dev, float threshold,
                    unsigned long long *out_dev, void *stream);
/* The same two steps with the threshold kept on the device, so that S_bubble of a field needs no host round trip ("this
 * post-processing ... hidden during copy"; eq. 3):
 *   of_bubble_threshold: threshold_dev[0] = T_v = 0.5 * (min + max) / n_fields of sum_dev (the running sum of n_fields fields,
 *                        of_field_accumulate) over the available vectors, formed in fp32;
 *   of_bubble_count_dev: as of_bubble_count with the threshold read from threshold_dev[0]. */
int of_bubble_threshold(of_handle h, const float *sum_dev, int n_fields, const uint8_t *valid_dev, float *threshold_dev, void *stream);
int of_bubble_count_dev(of_handle h, const float *vx_dev, const uint8_t *valid_dev, const float *threshold_dev,
                        unsigned long long *out_dev, void *stream);
/* of_field_minmax for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same result -- out_dev[0] = min, out_dev[1] = max of field_dev[0..n) over the available vectors (valid_dev may
 * be NULL), NaN ignored; the min / max step of eq. 3, PAPER.md:127-131 -- without a handle (of_create allocates) and without any
 * cudaMalloc, cudaFree or allocating library routine.  All pointers are device pointers of the CURRENT device (field_dev, out_dev
 * 4-byte aligned); asynchronous on `stream`; exact and bit-reproducible (integer min / max of per-chunk partials).
 *   Scratch: one file-scope `static __device__` array of OF_STATIC_SCRATCH_BYTES (33 024) bytes in liboptflow.so, held by every
 *   GPU that loads the library until the process exits.  It bounds the size: n > OF_STATIC_MAX_PIXELS (4096 x 4096) is rejected
 *   with OF_ERR_INVALID_ARG and a message that names the limit (as are n == 0 and null / misaligned pointers).
 *   Sharing: every call on a device uses the same array, which keeps the last call's contents; the call clears what must start
 *   at zero itself.  Calls that may OVERLAP on the GPU (different streams with no ordering between them, concurrent host
 *   threads) race on it and give wrong results: order them on one stream or with events.
 *   The first call on each device looks up the array's device address (cudaGetSymbolAddress, no allocation); make that call once
 *   before starting a graph capture. */
int of_field_minmax_static(const float *field_dev, const uint8_t *valid_dev, size_t n, float *out_dev, void *stream);

/* Stand-alone single steps (rows a2, a10 of the scope table), dense device buffers. */
int of_pyramid_down(const float *src, int width, int height, float *dst, void *stream);
int of_upsample_flow(const float *uc, const float *vc, int wc, int hc, float *u, float *v, int width,
                     int height, void *stream);

/* ---------------------------------------------------------------------------------------------
 * Frame pipeline (Fig. 4 schemes; "(5)" in BASELINE.json:5): four pinned host slots,
 * cudaMemcpyAsync on a side stream, events; uploading frame k+1 overlaps solving pair k, and the
 * download of field k overlaps solving pair k+1.
 *   OF_STREAM_CONSECUTIVE: each submitted frame is converted and pyramided once and used as I2 of
 *       pair (k-1,k) and I1 of pair (k,k+1) (scheme 1: "each field computation requires only one
 *       image to be processed"); frame 0 yields no field.
 *   OF_STREAM_PAIRS: each submit carries two frames (I1 then I2, contiguous) = one independent pair.
 * ------------------------------------------------------------------------------------------- */
/* dtype: of_dtype of the frames.  result_on_host != 0: fields are copied to pinned host buffers and
 * of_stream_result returns HOST pointers; else it returns device pointers. */
int of_stream_open(of_handle h, int dtype, int mode, int result_on_host);
/* Pinned host buffer for the next submit (W*H elements, x2 in PAIRS mode); the caller fills it.
 * Blocks until that slot's previous upload has completed.  NULL on error. */
void *of_stream_acquire(of_handle h);
/* Enqueue upload (+ solve + download) of the slot last acquired.  Up to three produced fields may be waiting to be collected
 * (small frames need that depth to keep the GPU busy: a field's way through upload, solve and download takes longer than two
 * solves); returns OF_ERR_STATE if three already are. */
int of_stream_submit(of_handle h);
/* Wait for the oldest uncollected field.  *u, *v point to H x W fp32 (host or device per
 * of_stream_open), valid until the second-next of_stream_result call.  *pair_index (optional)
 * receives its 0-based index.  OF_ERR_STATE if nothing is pending. */
int of_stream_result(of_handle h, const float **u, const float **v, int *pair_index);

/* Validity bytes (H x W, 1 = tr(G) > 0, D14) of the field the last of_stream_result returned: every slot of the result ring has
 * its own plane, written by the last pass of that pair's solve and copied with the field, so the mask belongs to the returned
 * field even while the next pair is being solved (eq. 3 counts "available vectors").  Host pointer if the pipeline
 * was opened with result_on_host, else device pointer; valid as long as the field's pointers. */
int of_stream_result_validity(of_handle h, const uint8_t **valid);
/* Drain and release the pipeline's buffers. */
int of_stream_close(of_handle h);

#ifdef __cplusplus
}
#endif
#endif /* OPTFLOW_H_ */
