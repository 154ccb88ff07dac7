/*
 * jpet.h - C-ABI boundary of the B200 (sm_100a) list-mode MLEM hot path for the two-strip J-PET detector
 * (arXiv:1502.07478; line numbers below are /root/reference/PAPER.md).
 *
 * One MLEM iteration (Eq. 3) is, per event e~_j = (z_u~, z_d~, dl~):
 *   1. direct reconstruction of (tan theta~, y~, z~)  (Eq. 2) and the pixel set E_j whose
 *      centres lie inside the 3-sigma ellipse b C^-1 b <= 9  (App. B :251-269);
 *   2. P(e~_j | i) for i in E_j  (Eq. 7-12, diagonal C) and the denominator
 *      sum_i P(e~_j|i) s(i) rho(i);
 *   3. back-projection  acc(i) += P(e~_j|i) / denominator_j  (Listing 1 line 10);
 *   4. rho_out(l) = rho_in(l) * acc(l) where s(l) > 0, else 0, with s the sensitivity of Eq. 4
 *      (PAPER.md:75-81).  Equivalent to Eq. 5-6 on rho' = s rho.
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  All functions return JPET_OK (0)
 * or a negative error code and never throw; jpet_last_error() gives the text for the calling thread.
 *
 * Conventions
 *   - lengths in mm; image plane (y, z); strips at y = +R (upper, "u") and y = -R (lower, "d"), |z| <= L/2;
 *   - images are float32, row-major [n_y][n_z] (z fastest); pixel (iy, iz) has its centre at
 *       y = (iy - (n_y-1)/2) * pixel,   z = (iz - (n_z-1)/2) * pixel;
 *   - events are float32 [n][3] = (z_u~, z_d~, dl~), C-contiguous; never modified;
 *   - "_dev" pointers are CUDA device pointers on the current device, "_host" pointers are host memory
 *     (pinned memory makes the copies asynchronous; pageable memory works but serialises);
 *   - every buffer is owned by the caller; the library owns only its internal workspace
 *     (sensitivity image, w = s*rho, accumulator replicas, counters, staging buffers), which it grows on
 *     demand and frees in jpet_release();
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer
 *     calls are asynchronous on that stream and never synchronise the device; host-pointer calls return
 *     after their result has landed in the host buffer;
 *   - the library keeps one workspace per CUDA device (the current device of the calling thread selects it) and is
 *     not re-entrant: calls must not overlap in time from several host threads.  Calls on different streams of one
 *     device are ordered by the library (each call waits, on its stream, for the previous call's work), so the
 *     workspace is never used by two streams at once; a3 coefficient, gamma, the sigma_z edge coefficient and the
 *     tuning options are process-wide.
 *   - arithmetic is fp32 (accumulation: fp32 partial sums per work item in shared memory, merged into the image
 *     with fp32 atomics, so the summation order - and the last bits - vary from run to run); the sensitivity
 *     image is evaluated in fp64 and rounded once to fp32.
 */
#ifndef JPET_H
#define JPET_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define JPET_OK 0
#define JPET_E_INVAL (-1)   /* NULL pointer, n < 0, non-positive R/L/sigma/pixel/n_y/n_z, grid reaching |y| >= R
                               (Eq. 4 divides by R -+ y), sigmas so large against R that Eq. 7's square root
                               could go non-positive inside the 3-sigma ellipse, or a sequencing error
                               (accumulate/end without begin) */
#define JPET_E_CUDA (-2)    /* a CUDA call failed (allocation, launch, copy); text in jpet_last_error() */
#define JPET_E_INTERNAL (-3) /* the event kernel met a record it cannot hold (a row piece longer than its register slot, a
                               row count outside the task table): 0 by construction; reported by jpet_get_counters
                               instead of returning a truncated image */

typedef struct { float R; float L; } jpet_geometry;               /* strips y = +-R, |z| <= L/2 */
typedef struct { float sigma_z; float sigma_dl; } jpet_sigmas;    /* C^-1 = diag(1/sz^2, 1/sz^2, 1/sdl^2), gamma = 0
                                                                     (Eq. 12 and PAPER.md:124) */
typedef struct { int32_t n_y; int32_t n_z; float pixel; } jpet_grid;   /* centred on the origin, see above */

/* Sensitivity image, Eq. 4 at every pixel centre, clamped to >= 0 (pixels no LOR through both
 * strips can see).  s_dev: float32 [n_y*n_z], written. */
int jpet_sensitivity(const jpet_geometry *geometry, const jpet_grid *grid, float *s_dev, void *cuda_stream);

/* One MLEM iteration, Eq. 3 = steps 1-4 above.
 *   events_dev : float32 [n][3]; n >= 0 (n == 0 gives rho_out = 0, the empty sum over j)
 *   rho_in_dev : float32 [n_y*n_z], read;  rho_out_dev: float32 [n_y*n_z], written; the two may alias
 * Events with a non-finite component, with no pixel centre inside their ellipse, or with a non-positive
 * denominator are skipped and counted (jpet_get_counters).  Events are processed in internal batches of at
 * most 10^7 (sorted by image sub-tile on the device, then the event kernels) launched back to back on the stream. */
int jpet_mlem_iterate(const float *events_dev, int64_t n, const jpet_geometry *geometry, const jpet_sigmas *sigmas,
                      const jpet_grid *grid, const float *rho_in_dev, float *rho_out_dev, void *cuda_stream);

/* n_iter iterations starting from rho_init_dev (NULL => all ones); n_iter == 0 copies the start image.
 * rho_out_dev may alias rho_init_dev. */
int jpet_reconstruct(const float *events_dev, int64_t n, const jpet_geometry *geometry, const jpet_sigmas *sigmas,
                     const jpet_grid *grid, const float *rho_init_dev, float *rho_out_dev, int32_t n_iter,
                     void *cuda_stream);

/* jpet_mlem_iterate for callers that cannot allocate device memory when they need an iteration.
 * Who that is: a loop with a latency budget (detector monitoring during acquisition) - cudaMalloc and cudaFree hold up
 * every stream of the device while they run, and jpet_mlem_iterate grows its workspace on demand; a plug-in inside a
 * program that has given all device memory to its own pool, where cudaMalloc just fails; a process that is not allowed
 * driver allocations after start-up.  This call makes none: no cudaMalloc, cudaFree or allocating library routine, on
 * any call.  Its scratch (s of Eq. 4, w = s rho, the accumulator, counters) is a fixed array of 3 MiB + 256 bytes compiled
 * into the library; every GPU that loads the library holds that array until the process exits.
 *   - Same arguments, result and skipping rules as jpet_mlem_iterate (Eq. 3, steps 1-4 above; a3 coefficient, gamma and
 *     the sigma_z edge coefficient are honoured, tuning options and "exact_kernel" are not); the caller owns events and
 *     both images, rho_out_dev may alias rho_in_dev; asynchronous on cuda_stream.
 *   - Limits: n_y * n_z <= JPET_NOALLOC_MAX_PIXELS and n <= 2^31 - 1, else JPET_E_INVAL with the limit in the text.
 *   - Every event takes the direct kernel (one warp per event, w read from global memory, red.global.add into the
 *     accumulator) straight from events_dev, unsorted: the slow, simple path - expect a fraction of jpet_mlem_iterate's
 *     rate.  The image differs from jpet_mlem_iterate's by fp32 summation order only.
 *   - The first call on a device looks the array's device address up (cudaGetSymbolAddress) and reads the SM count; make
 *     that first call on each device before any stream capture begins.
 *   - All calls share the one array per device, and it keeps what the last call left in it; each call rewrites or zeroes
 *     every part it reads, so calls one after another (same or different grids) are independent.  Two calls that overlap
 *     on the GPU (different streams without an ordering between them, or two host threads) race on it: order them.
 *     The array is separate from the workspace of the other calls, so those may run concurrently with this one;
 *     jpet_get_counters does not see this call and jpet_release does not free the array. */
#define JPET_NOALLOC_MAX_PIXELS (512 * 512)
int jpet_mlem_iterate_noalloc(const float *events_dev, int64_t n, const jpet_geometry *geometry, const jpet_sigmas *sigmas,
                              const jpet_grid *grid, const float *rho_in_dev, float *rho_out_dev, void *cuda_stream);

/* The same iteration split in three so that a caller can stream event batches (BASELINE config 5):
 *   begin      : w = s * rho_in, accumulators and counters zeroed
 *   accumulate : steps 1-3 for one batch of events (device pointer); any number of calls
 *   end        : step 4 into rho_out_dev (rho_in_dev must hold the same image that was given to begin)
 * begin, accumulate (any number of times), end on one stream is exactly jpet_mlem_iterate. */
int jpet_mlem_begin(const jpet_geometry *geometry, const jpet_sigmas *sigmas, const jpet_grid *grid,
                    const float *rho_in_dev, void *cuda_stream);
int jpet_mlem_accumulate(const float *events_dev, int64_t n_batch, void *cuda_stream);
int jpet_mlem_end(const float *rho_in_dev, float *rho_out_dev, void *cuda_stream);

/* Host-buffer forms (the end-to-end path): events and images live in host memory; the call copies the events
 * to the device in chunks of `chunk_events` (<= 0: library default) on a copy stream that runs ahead of the
 * compute stream, runs the iteration(s) and copies rho back.  Returns when rho_out_host is complete.
 * For n_iter > 1 the events are uploaded once if they fit the staging budget (4 GiB), else once per iteration. */
int jpet_mlem_iterate_host(const float *events_host, int64_t n, const jpet_geometry *geometry,
                           const jpet_sigmas *sigmas, const jpet_grid *grid, const float *rho_in_host,
                           float *rho_out_host, int64_t chunk_events);
int jpet_reconstruct_host(const float *events_host, int64_t n, const jpet_geometry *geometry,
                          const jpet_sigmas *sigmas, const jpet_grid *grid, const float *rho_init_host,
                          float *rho_out_host, int32_t n_iter, int64_t chunk_events);

/* Counters of the most recent iteration on `cuda_stream` (synchronises that stream):
 *   n_evals   = sum_j |E_j|  - unique (event, pixel-centre-inside-ellipse) pairs, the "kernel evaluations"
 *   n_skipped = events skipped as described above
 * Either pointer may be NULL.  Returns JPET_E_INTERNAL if the event kernel flagged a record it could not hold. */
int jpet_get_counters(uint64_t *n_evals_host, uint64_t *n_skipped_host, void *cuda_stream);

/* Counts |E_j| without evaluating the kernel (for evals/s when no iteration has been run).  Synchronises. */
int jpet_count_evals(const float *events_dev, int64_t n, const jpet_geometry *geometry, const jpet_sigmas *sigmas,
                     const jpet_grid *grid, uint64_t *n_evals_host, uint64_t *n_skipped_host, void *cuda_stream);

/* Coefficient of the third component of vector a in Eq. 9.  2 (default) makes a = d e/d theta,
 * consistent with Eq. 8 and Eq. 10; 1 is the equation exactly as printed (reading R5). */
int jpet_set_a3_coef(float k);
float jpet_get_a3_coef(void);

/* Off-diagonal coefficient gamma of the inverse correlation matrix, Eq. 12:
 *   C^-1 = [[1/sigma_z^2, 0, gamma], [0, 1/sigma_z^2, -gamma], [gamma, -gamma, 1/sigma_dl^2]]   [1/mm^2].
 * 0 (default) is the diagonal matrix the paper works with.  Process-wide, takes effect at the next
 * begin / iterate / reconstruct call; those return JPET_E_INVAL when |gamma| > 0.5 / (sqrt(2) sigma_z sigma_dl)
 * (the matrix must stay positive definite and Eq. 7's D positive).  The 3-sigma ellipse does not depend on gamma
 * (b1 = b2 in Eq. 10).  The set call returns JPET_E_INVAL for a non-finite value. */
int jpet_set_gamma(float gamma);
float jpet_get_gamma(void);

/* sigma_z as a function of the hit position (C^-1 "depends on the z~u and z~d ... on the order of 10% from
 * the center (lowest) to the edge (highest)"; the paper gives no functional form - DESIGN.md reading R22):
 *   sigma_z(z) = sigma_z * (1 + eta * min(1, (2 z / L)^2)),   C^-1 = diag(1/sigma_z(z~u)^2, 1/sigma_z(z~d)^2, 1/sigma_dl^2) (+ gamma)
 * per event.  eta = 0 (default) is the constant sigma_z the paper works with; 0.1 is the paper's 10 %.  Process-wide,
 * takes effect at the next begin / iterate / reconstruct / count call; JPET_E_INVAL outside [0, 1]. */
int jpet_set_sigma_z_edge(float eta);
float jpet_get_sigma_z_edge(void);

/* Direct reconstruction (Eq. 2, Fig. 4b): every event is reconstructed to (y~, z~) and counted in the
 * pixel that contains the point (pixel (iy, iz) covers [y_c - pixel/2, y_c + pixel/2) x [z_c - pixel/2, z_c + pixel/2)).
 *   hist_dev       : uint32 [n_y*n_z], INCREMENTED (zero it first for a fresh histogram)
 *   n_outside_host : events whose point falls outside the grid or has a non-finite component (not counted); may be
 *                    NULL; when given the call synchronises the stream, otherwise it is asynchronous. */
int jpet_direct_histogram(const float *events_dev, int64_t n, const jpet_geometry *geometry, const jpet_grid *grid,
                          uint32_t *hist_dev, uint64_t *n_outside_host, void *cuda_stream);

/* Event simulation on the device (the recipe of DESIGN.md section 5, phantom rule
 * PAPER.md:245): event slot i = first + k (k = 0..n-1) is drawn from its own counter-based random stream
 * Philox4x32-10(key = (seed low word, seed high word), counter = (slot low word, slot high word, attempt, block)); a 32-bit
 * output word x becomes the uniform ((x >> 8) + 0.5) 2^-24.  Block 0 of an attempt gives (u0, u1, u2, u3): position, the
 * acceptance draw and the angle; block 1 of the accepted attempt gives the four uniforms of the two Box-Muller pairs
 * (csrc/generator.cuh has the exact order).  Attempt a = 0, 1, ... draws (y, z) uniform in the
 * phantom's bounding rectangle, accepts it with probability intensity / max intensity (first primitive in the list
 * wins), draws theta uniform on (-pi/2, pi/2), keeps the emission if both strips are hit, and smears
 * (z_u, z_d, dl) with N(0, sigma_z), N(0, sigma_z), N(0, sigma_dl) (Box-Muller).  Slot i is therefore the same event
 * whatever n, first or the launch shape.  kind: 0 = ellipse, 1 = box; centre (cy, cz), half sizes (hy, hz) [mm],
 * phi_deg counter-clockwise in the (z horizontal, y vertical) plane.  events_dev: float32 [n][3], written. */
typedef struct { int32_t kind; float cy, cz, hy, hz, phi_deg, intensity; } jpet_primitive;
int jpet_generate_events(const jpet_primitive *phantom_host, int32_t n_primitives, int64_t n, int64_t first,
                         const jpet_geometry *geometry, const jpet_sigmas *sigmas, uint64_t seed, float *events_dev,
                         void *cuda_stream);

/* Multi-GPU event sharding (the paper's CPU scheme - a private rho_new per thread, summed at the
 * end of the iteration, PAPER.md:157 - lifted to devices): every rank runs begin + accumulate over its shard of the
 * events, then the accumulators are summed and every rank finalises.
 *   jpet_mlem_accumulator     device pointer and length of the accumulator of the open iteration (transposed image,
 *                             float32 [n_z][n_y]); valid until the next begin on a different grid or jpet_release -
 *                             for an NCCL all-reduce in place, or for the IPC export below
 *   jpet_mlem_end_peers       step 4 with the accumulator read as the sum of n_peers device buffers (this rank's own
 *                             included, same order on every rank so all ranks get identical bits): the all-reduce
 *                             fused into the finalise kernel over peer (NVLink) mappings.  The caller guarantees that
 *                             every peer has finished its accumulate (a barrier after a stream synchronise) and does
 *                             not start its next begin before all ranks have finished this call.
 *   jpet_ipc_export / open / close   cudaIpc handle (64 bytes) of a device buffer of this process, its mapping in
 *                             another process on the same node, and the unmapping. */
#define JPET_MAX_PEERS 16
int jpet_mlem_accumulator(float **acc_dev, int64_t *n_floats);
int jpet_mlem_end_peers(const float *rho_in_dev, float *rho_out_dev, const float *const *peer_acc_dev, int32_t n_peers,
                        void *cuda_stream);
int jpet_ipc_export(const void *dev_ptr, void *handle64_out);
int jpet_ipc_open(const void *handle64, void **dev_ptr_out);
int jpet_ipc_close(void *dev_ptr);

/* Tuning knobs (do not change results beyond fp32 summation order).  name/value pairs:
 *   "variant"      event-kernel shape id (index into the shape list JPET_SHAPES of csrc/rows_launch.h, see DESIGN.md section 6;
 *                  jpet_plan_describe reports it); -1 = automatic
 *   "force_direct" 1 = skip the shared-memory tiled path: every event goes through the direct kernel
 *                  (w from global memory, red.global.add into the image); 0 = automatic
 *   "chunk"        events per work item of the tiled path; 0 = automatic
 *   "sub_tile_z"   width in pixels of the image sub-tiles the events are sorted by; 0 = automatic.  A forced width whose
 *                  regions do not fit shared memory is not replaced by another: every event then takes the direct kernel
 *                  ("last_tiled" reads 0)
 *   "ctas_per_sm"  cap on resident CTAs per SM for the persistent grid; 0 = automatic
 *   "poly_off"     1 = never evaluate the exponent of Eq. 7 as a polynomial in u (always rsqrt + ex2); 0 = automatic:
 *                  the plan bounds the truncation error and picks degree 3, 4, 5 or the closed form
 *   "degree_classes_off"  1 = one degree for all events; 0 (default) = when the plan's degree is 4 or 5, the sort tests every
 *                  event against its own truncation bound and the events that pass are walked with the degree-3
 *                  polynomial (a second launch of the same kernel shape; gamma = 0 and constant sigma_z only)
 *   "pdl"          1 (default) = launch the kernels of an iteration with programmatic stream serialisation (each starts
 *                  with griddepcontrol.wait: only launch latency overlaps the previous kernel); 0 = plain launches
 *   "time_kernel"  1 = bracket each tiled event-kernel launch with CUDA events on its stream; the summed duration of
 *                  the launches of the last iteration (one per batch of events) is then read with
 *                  jpet_get_option("last_kernel_ns") (synchronises on the last one), their number with
 *                  "last_kernel_launches"
 *   "stage_bytes"  device staging budget of the host-buffer calls (default 4 GiB; 0 = default): events beyond it are
 *                  streamed through a two-slot ring, once per iteration
 *   "exact_kernel" > 0: replace Eq. 7 by the integral it approximates (P = int dtheta/pi N(e~; e(y,z,theta), C)
 *                  over (-pi/2, pi/2)) evaluated with that many trapezoid nodes in tan(theta) over +-8 sigma around the
 *                  integrand's peak, on the same 3-sigma pixel set; every event takes the direct kernel (a diagnostic mode,
 *                  ~50x slower); 0 (default) = Eq. 7
 * jpet_get_option also answers "last_variant", "last_variant_low" (the degree-3 shape of the second degree class, -1 if
 * there is one class), "last_tiled", "last_smem_bytes" (what the last iteration used) and
 * "last_overflow" (row pieces that did not fit their register slot: 0 by construction; synchronises the device).
 * Returns JPET_E_INVAL for an unknown name or a value out of range. */
int jpet_set_option(const char *name, int64_t value);
int64_t jpet_get_option(const char *name);

/* Number of kernels this library has launched since load (for bench.py's gpu_launches). */
uint64_t jpet_launch_count(void);

/* Frees the internal workspace (device and pinned host memory).  Safe to call at any time between calls. */
void jpet_release(void);

/* Text of the last error on the calling thread ("" if none).  The pointer stays valid until the next call. */
const char *jpet_last_error(void);

/* Host-side plan of the event kernel for a problem (no GPU needed; for tests and tuning): the kernel shape and the
 * tiling that jpet_mlem_begin would choose with the current options, a3 coefficient and gamma.
 *   out[0] shape id              out[1] degree of the exponent polynomial (0 = closed form rsqrt + ex2)
 *   out[2] warps per event       out[3] event groups per CTA       out[4] / out[5] pixel capacity of piece A / B
 *   out[6] HS (rows of a region) out[7] WZ (columns of a region)   out[8] / out[9] sub-tile Sy / Sz
 *   out[10] / out[11] halo Hy / Hz                                 out[12] events per work item
 *   out[13] dynamic shared memory per CTA [bytes]                  out[14] 1 = tiled (0: every event on the direct kernel)
 *   out[15] / out[16] smallest / largest ellipse row count of the task table (0, 0: no table)
 *   out[17] (when n_out >= 18) shape id of the degree-3 instance for the events of the second degree class, -1 if none
 * n_out = number of int64 slots the caller provides (>= 17).  task_table_host (may be NULL) receives up to
 * table_cap 32-bit words of the task table [(row count - out[15]) * 32 * out[2] + lane]: piece A in bits 0-15, piece B
 * in bits 16-31; a 16-bit entry: bits 0-7 row, 8-9 part, 10-11 log2(parts), bit 15 valid (csrc/task_table.h).
 * Returns the number of table words (>= 0), or a negative error code. */
int64_t jpet_plan_describe(const jpet_geometry *geometry, const jpet_sigmas *sigmas, const jpet_grid *grid, int64_t *out,
                           int32_t n_out, uint32_t *task_table_host, int64_t table_cap);

/* Name of an event-kernel shape id ("" if out of range); the pointer is static. */
const char *jpet_shape_name(int32_t shape);

/* ABI version of this header: bumped whenever a signature changes. */
int jpet_abi_version(void);
#define JPET_ABI_VERSION 2

#ifdef __cplusplus
}
#endif
#endif /* JPET_H */
