/*
 * dm.h -- C ABI of the B200-native multi-mode difference-map (DM) iteration.
 *
 * What it computes: Section II of arXiv:1808.10375, eqs. (1)-(7):
 * for every view j and mode pair (k,l) the exit wave psi_jkl = P_k * O_l|window (eq. 2,
 * PAPER.md:43) is updated by eq. (3) with the constrained Fourier
 * transform of eq. (4), then the object is updated by eq. (6)
 * (PAPER.md:60), the probe by eq. (5), and one row of convergence errors
 * (eq. (7)) is appended.  Readings of everything the paper leaves open
 * (order of the updates, beta, regularisers, FFT convention, error definitions) are the
 * table "Readings" in DESIGN.md; this header only states argument meaning.
 *
 * Conventions
 *   - every pointer says HOST or DEV.  DEV = device memory of the current CUDA device,
 *     owned by the caller (PyTorch in this repo); the library never frees or reallocates
 *     caller memory and allocates no device memory itself: all state lives in the
 *     workspace the caller lends with dm_plan_set_workspace.
 *   - complex arrays are interleaved float pairs (re,im) = complex64, row-major.
 *       probe   c64 [K][N][N]          object  c64 [L][obj_h][obj_w]
 *       psi     c64 [n_views][K][L][N][N]
 *       intensities f32 [n_views][N][N], zero frequency (DC) at index [0][0], never fftshifted
 *   - positions int32 [n_views][2] = (y0,x0): top-left corner of view j's N x N object
 *     window; probe pixel (ry,rx) meets object pixel (y0+ry, x0+rx).  Integer pixels only.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Work is enqueued
 *     asynchronously unless the function says "syncs".
 *   - no exception, abort or exit crosses this boundary: every call returns a dm_status.
 *     dm_last_error(plan) gives a text for the last non-OK status of that plan.
 *     Asynchronous device faults surface as DM_ERR_CUDA at the next syncing call.
 *   - thread safety: one plan may be used from one host thread at a time.
 */
#ifndef DM_B200_H
#define DM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dm_plan dm_plan; /* opaque, owned by the library */

typedef enum {
    DM_OK = 0,
    DM_ERR_INVALID_ARG = 1,   /* null pointer, non-positive size, value out of range        */
    DM_ERR_OUT_OF_BOUNDS = 2, /* a view window is not inside [0,obj_h) x [0,obj_w)          */
    DM_ERR_UNSUPPORTED = 3,   /* N not in {64,128,256,512}, K*L > 8, odd obj_w              */
    DM_ERR_NO_DATA = 4,       /* dm_iterate / getters before dm_set_data                    */
    DM_ERR_WORKSPACE = 5,     /* workspace missing, too small, misaligned, error table full */
    DM_ERR_CUDA = 6           /* a CUDA runtime call failed; text in dm_last_error          */
} dm_status;

typedef enum {
    DM_PARAM_BETA = 0,        /* beta of eq. (3), in [0,1]; default 1.0                      */
    DM_PARAM_ALPHA_OBJ = 1,   /* relative inertial factor a_O >= 0 of eq. (6); default 1e-3  */
    DM_PARAM_ALPHA_PROBE = 2, /* relative inertial factor a_P >= 0 of eq. (5); default 1e-3  */
    DM_PARAM_EPS_F = 3,       /* zero guard in eq. (4): scale = amp/sqrt(S+eps); default 1e-30 */
    DM_PARAM_PATH = 4,        /* 0 = auto (default), 1 = force the staged (L2-scratch) path,
                                 2 = force the fused shared-memory path (DM_ERR_UNSUPPORTED at
                                 dm_set_data if N > 128), 3 = force the register-resident
                                 path (DM_ERR_UNSUPPORTED at dm_set_data unless N = 128),
                                 4 = force the view-pipelined warp-FFT path (any N; the
                                 default for N >= 256)                                       */
    DM_PARAM_LAG = 5,         /* path 4: views between the row, column and inverse-row phases
                                 of one view (integer >= 1; 0 = derive from the task counts,
                                 default).  Sizes the scratch ring: set before
                                 dm_plan_set_workspace (INVALID_ARG afterwards)              */
    DM_PARAM_PRECISION = 6    /* 0 = FP32 / complex64 (default, the tuned paths); 1 = FP64 /
                                 complex128 validation mode: the whole iteration in the
                                 paper's own precision with plain kernels and
                                 the definition's summation orders -- for long free-running
                                 comparisons, not for speed.  Inputs and getters stay
                                 float32 / complex64 (converted at the boundary); the error
                                 table is f64 either way.  Needs a larger workspace: set
                                 before dm_plan_set_workspace (INVALID_ARG afterwards)       */
} dm_param;

/* Build the plan (HOST only, no CUDA call): validates, copies `positions` (HOST,
 * int32 [n_views][2]), builds the scan-window table and the per-object-tile coverage
 * lists (step S0 of DESIGN.md; r_j of eq. (2)).
 * Errors: INVALID_ARG (null, sizes <= 0), UNSUPPORTED (N, K*L, odd obj_w),
 * OUT_OF_BOUNDS (first offending view is named in dm_last_error of a NULL plan).    */
dm_status dm_plan_create(dm_plan **out, int N, int n_views, int K, int L, int obj_h, int obj_w,
                         const int32_t *positions);

/* Set a parameter.  Must precede dm_set_data (INVALID_ARG afterwards or out of range). */
dm_status dm_plan_set_param(dm_plan *plan, dm_param which, double value);

/* Bytes of device workspace the plan needs (psi, sqrt(I), P/O double buffers, tables,
 * partial sums, error table, L2 scratch of the staged path).  Asks the current CUDA
 * device for its SM count (the reduction geometry and the persistent grids follow it;
 * without a device the B200's 148 is assumed).                                        */
dm_status dm_plan_workspace_bytes(dm_plan *plan, size_t *bytes);

/* Lend the workspace: DEV pointer, 256-byte aligned, >= dm_plan_workspace_bytes.  Borrowed
 * until dm_plan_destroy; contents are the library's.                                   */
dm_status dm_plan_set_workspace(dm_plan *plan, void *dev, size_t bytes);

/* Load a problem: stores sqrt(I) (in the spectrum layout of the kernels),
 * copies P0 and O0, sets psi_jkl = P0_k * O0_l|window, freezes the absolute regularisers
 * from P0/O0 (reading A8), uploads the tables and clears the error table.
 * intensities DEV f32 [n_views][N][N] (>= 0, not validated on the device),
 * probe0 DEV c64 [K][N][N], object0 DEV c64 [L][obj_h][obj_w].  Work is enqueued on `stream`;
 * the caller's buffers may be released once that stream work has completed.  The FIRST call
 * on a workspace (and the first after a change of path or precision) also uploads the integer
 * tables and twiddles from pageable host memory and SYNCS `stream` (up to three times) while
 * doing so; later calls on the same workspace are fully asynchronous.                    */
dm_status dm_set_data(dm_plan *plan, const float *intensities, const float *probe0,
                      const float *object0, void *stream);

/* Run n_iter >= 0 DM iterations (psi update eq. 3/4, object eq. 6, probe eq. 5, errors
 * eq. 7), async on `stream`, no host synchronisation inside.  Appends n_iter error rows. */
dm_status dm_iterate(dm_plan *plan, int n_iter, void *stream);

/* Copy the current probe / object / psi to caller DEV buffers (async on `stream`).      */
dm_status dm_get_probe(const dm_plan *plan, float *out_dev, void *stream);
dm_status dm_get_object(const dm_plan *plan, float *out_dev, void *stream);
dm_status dm_get_psi(const dm_plan *plan, float *out_dev, void *stream);

/* Error table: row it = [eps_F, eps_psi, eps_P[0..K), eps_O[0..L)] as f64 (DESIGN.md
 * reading A10; eq. (7)).  Copies min(rows, max_rows) rows to out_host (HOST) and SYNCS
 * the device.                                                                          */
dm_status dm_get_errors(const dm_plan *plan, double *out_host, int max_rows, int *rows_written);

/* Parity hook (teacher forcing): overwrite probe / object / psi from DEV buffers; NULL =
 * keep.  Does not touch sqrt(I), the frozen regularisers or the error table.           */
dm_status dm_set_state(dm_plan *plan, const float *probe_dev, const float *object_dev,
                       const float *psi_dev, void *stream);

/* Integer tables of step S0 (HOST outputs, no CUDA call), compared bit-exactly with the
 * oracle's.  Window table: int32 [n_views][3] = (y0, x0, y0*obj_w + x0).               */
dm_status dm_get_window_table(const dm_plan *plan, int32_t *out_host);
/* Coverage lists: for every tile_h x tile_w object tile (row-major), the ascending list of
 * views whose window intersects it, as CSR.  Call once with tile_ptr_host = tile_views_host
 * = NULL to get tile_h, tile_w and nnz; then with arrays of n_tiles+1 and nnz entries.   */
dm_status dm_get_coverage(const dm_plan *plan, int *tile_h, int *tile_w, int32_t *tile_ptr_host,
                          int32_t *tile_views_host, int64_t *nnz);

/* The frozen absolute regularisers (alpha_obj, alpha_probe) computed by dm_set_data, as
 * f64[2] to HOST.  SYNCS.                                                              */
dm_status dm_get_alphas(const dm_plan *plan, double *out_host2);

/* Mode diagnostics (a probe mode is kept while its "contribution ... to the total
 * intensity is larger than at least 1%"): the power fraction of every mode of the current
 * state, out_host[k] = sum_r |P_k|^2 / sum_k sum_r |P_k|^2 (k < K) followed by the same for the
 * object modes, out_host[K + l]; f64[K + L] to HOST; 0/0 := 0.  Fixed-order FP64 sums.  SYNCS THE
 * DEVICE (cudaDeviceSynchronize) first, so it sees the state of whatever stream dm_iterate ran on, then
 * runs its two small kernels on the default stream and syncs again: a diagnostic, not a hot-path call.  */
dm_status dm_get_mode_power(const dm_plan *plan, double *out_host);

/* End-to-end entry with HOST buffers (what a beamline caller with data in host memory
 * does): copies intensities / probe0 / object0 HOST->DEV into a staging
 * area inside the workspace, runs dm_set_data + n_iter iterations, copies probe and object
 * DEV->HOST, and SYNCS.  out_probe_host / out_object_host may be NULL.  Needs the
 * workspace (which includes the staging area).  The intensities travel in 8 chunks on an
 * internal copy stream while the set-up kernels that do not need them (psi = P0*O0, the
 * frozen regularisers) run on `stream`; pass pinned host memory for the copies to be
 * asynchronous.  Results are bit-identical to the device-pointer calls.                 */
dm_status dm_solve_host(dm_plan *plan, const float *intensities_host, const float *probe0_host,
                        const float *object0_host, int n_iter, float *out_probe_host,
                        float *out_object_host, void *stream);

/* Which path dm_iterate runs for this plan: 1 staged, 2 fused, 3 register-resident,
 * 4 view-pipelined warp-FFT, 64 FP64 validation mode
 * (valid after dm_set_data);
 * and how many kernels one iteration launches (the bench's gpu_launches claim).           */
dm_status dm_plan_info(const dm_plan *plan, int *path, int *launches_per_iter);

/* Launch geometry the kernels of this plan run with (test / measurement aid; HOST output, no
 * CUDA call).  The parity tests assert through it that they reach the loop shapes of the
 * full-size launches.  Writes min(n_out, DM_GEOMETRY_FIELDS) int32 values:
 *   [0] psi-update path (as dm_plan_info)      [1] SM count the grids were sized for
 *   [2] probe update (eq. (5)): CTAs along the view axis   [3] views summed by each of them
 *   [4] object update (eq. (6)): longest coverage list     [5] list entries per batch
 *   [6] path 3: persistent CTAs   [7] CTAs per view   [8] most views one of their groups takes
 *   [9] path 4: scratch ring slots    [10] phase lag (views)   [11] persistent CTAs   [12] warps per CTA
 *   [13] path 3: 1 = the CTAs of a view meet at a software barrier in L2, 0 = hardware cluster
 * [6]-[8], [11] and [13] are valid after dm_set_data (they come from occupancy queries).          */
#define DM_GEOMETRY_FIELDS 14
dm_status dm_plan_geometry(const dm_plan *plan, int32_t *out_host, int n_out);

/* Per-phase device timing (measurement aid of bench.py; off by default).  When on, dm_iterate
 * records CUDA events on `stream` around the four phases of every iteration (psi update S1-S6,
 * object S7, probe S8, error row S9), for at most 4096 iterations between two reads.
 * dm_get_phase_ms SYNCS, writes the summed milliseconds per phase to out_ms4 (HOST f32[4]) and
 * the number of iterations they cover to *iters, and resets the accumulation.            */
dm_status dm_plan_set_profiling(dm_plan *plan, int on);
dm_status dm_get_phase_ms(dm_plan *plan, float *out_ms4, int *iters);

/* Measurement aid (no plan needed): the roofline denominators of DESIGN.md measured on the current
 * device with plain streaming kernels ("FP32 peak").  scratch_dev = DEV buffer of
 * scratch_bytes >= 512 MiB (>> L2; contents destroyed), 16-byte aligned.  Writes min(n_out,
 * DM_PEAK_FIELDS) f64 to out_host (HOST) and SYNCS:
 *   [0] FP32 lane-operations/s with scalar FFMA     [1] the same with packed FFMA2 (fma.rn.f32x2)
 *   [2] HBM read-only GB/s   [3] HBM copy GB/s (read + write bytes)   [4] L2-resident read GB/s (32 MiB)
 *   [5] shared-memory read GB/s (conflict-free 128-bit)   [6] SM count
 * One FMA counts as ONE lane-operation: an FFT butterfly is mostly adds, so the FP32 bound of the psi
 * update is lane-operations / [0], not flops / (2 x [0]).  Errors: INVALID_ARG, WORKSPACE, CUDA.        */
#define DM_PEAK_FIELDS 7
dm_status dm_measure_peaks(void *scratch_dev, size_t scratch_bytes, double *out_host, int n_out, void *stream);

/* Test hook, HOST only, no CUDA call: runs the kernels' own FFT pass code (the same
 * __host__ __device__ functions the kernels inline: radix butterflies, twiddle table,
 * swizzled tile addressing, digit-reversal map) single-threaded on the host for one
 * N x N frame and returns the spectrum in natural order.  in/out HOST c64 [N][N].       */
dm_status dm_host_fft2(int N, const float *in_host, float *out_host, int inverse);
/* Same hook for a named psi-update path: 1/2 = the shared-memory tile passes above, 3 = the
 * register-resident 128 x 128 transform (csrc/dm_regfft.cuh: register passes, both exchange
 * layouts, spectrum-layout table) emulated thread by thread, phase by phase.  N = 128 only
 * for path 3 (UNSUPPORTED otherwise).                                                    */
dm_status dm_host_fft2_path(int N, int path, const float *in_host, float *out_host, int inverse);

/* Probe update without a workspace and without any allocation: eq. (5), PAPER.md:58,
 *   P_k(r) = (alpha P_old_k(r) + sum_j sum_l conj(O_l(r + r_j)) psi_jkl(r)) / (alpha + sum_j sum_l |O_l(r + r_j)|^2),
 * the same two-stage reduction dm_iterate runs as its step S8 (FP32 partial sums over contiguous view
 * chunks, j ascending and l ascending inside; chunk-ascending FP64 second stage; P_new = P_old where the
 * denominator is 0), for a caller that holds psi, O and P itself.
 * For whom: every other call of this header needs a workspace the caller allocates.  A caller that may not
 * allocate -- a plug-in in an application whose own pool took all device memory at start-up, a measurement-time
 * loop in which cudaMalloc / cudaFree are forbidden because they stall every stream of the device and may fail
 * -- has nowhere to put the partial sums.  Here they go into a fixed array of DM_NOALLOC_SCRATCH_BYTES that is
 * part of the library image: the CUDA driver places it on each GPU that loads the library and keeps it until the
 * process exits.  The call itself performs no cudaMalloc / cudaFree and uses no allocating library routine.
 *   positions_dev  DEV int32 [n_views][2] = (y0, x0); NOT validated (they are device data): every window must
 *                  lie inside the object, as dm_plan_create would have checked
 *   object_dev     DEV c64 [L][obj_h][obj_w]        psi_dev  DEV c64 [n_views][K][L][N][N], 16-byte aligned
 *   probe_old_dev  DEV c64 [K][N][N]                probe_new_dev  DEV c64 [K][N][N] (out; must not alias probe_old_dev)
 *   alpha_probe    the ABSOLUTE regulariser (>= 0), e.g. dm_get_alphas()[1] of a plan, or 0 for the literal quotient
 *   err_text_host  HOST char[err_text_bytes] or NULL: receives the text of a non-OK status (there is no plan to ask)
 * Limit: N * N * (8 K + 4) bytes (one chunk of partial sums) must fit the array, else DM_ERR_WORKSPACE with both
 * sizes in the text; within the limit, fewer chunks fit for larger N * N * K, which costs parallelism, not
 * correctness (the FP32 summation order, hence the last bits, follows the chunk count).  Other errors:
 * INVALID_ARG (null, sizes < 1, alpha < 0), UNSUPPORTED (N, K * L > 8), OUT_OF_BOUNDS (object smaller than a
 * window), CUDA.  Async on `stream`.
 * First call on each device: looks up the device address of the array (cudaGetSymbolAddress, once per device,
 * with that device current) and the SM count; make that call outside any stream capture.
 * Sharing: all calls on a device use the same array, which keeps the previous call's contents (nothing in it
 * needs clearing: a call overwrites every slot it later reads).  Calls that overlap on the GPU (two streams,
 * two host threads) race on it: serialise them.                                                              */
#define DM_NOALLOC_SCRATCH_BYTES (16u << 20)
dm_status dm_probe_update_noalloc(int N, int n_views, int K, int L, int obj_h, int obj_w,
                                  const int32_t *positions_dev, const float *object_dev, const float *psi_dev,
                                  const float *probe_old_dev, float alpha_probe, float *probe_new_dev, void *stream,
                                  char *err_text_host, size_t err_text_bytes);

const char *dm_status_string(dm_status s);
const char *dm_last_error(const dm_plan *plan); /* plan may be NULL: last create error */
void dm_plan_destroy(dm_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* DM_B200_H */
