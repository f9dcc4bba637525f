/*
 * vmat.h - C ABI of libvmat: the beamlet-price step of the pricing problem of the
 * column-generation VMAT optimiser of arXiv 1503.01721, on one NVIDIA B200 (sm_100a).
 *
 *   x --> d = D x --> (F, g = dF/dd) --> p = D^T g --> per control point, per MLC leaf row,
 *                                                      the minimum-price contiguous opening
 *
 * Citations are lines of /root/reference/PAPER.md ("L43" = line 43) with the section or
 * equation they fall in; "C1".."C14" are the readings listed in DESIGN.md.
 *
 * Conventions for every call
 *   - `dev` pointers are CUDA device memory of the current device, `host` pointers are host
 *     memory.  The library never allocates or frees a vector it is handed: the caller owns
 *     every argument before and after the call.  The handle owns only the two matrix layouts
 *     and its scratch.
 *   - Compute calls enqueue work on `stream` (a cudaStream_t passed as void*, NULL = the legacy
 *     default stream) and return without synchronising.  Scalars (F, best_angle) land in device
 *     memory.  One evaluation may be in flight per handle at a time (the handle holds scratch).
 *   - Return value: VMAT_OK (0) or a negative vmat_status; no exception or abort crosses the
 *     ABI; on failure the outputs are unspecified and *out handles are left untouched.
 *     vmat_last_error() gives a thread-local message for the last failure.
 *   - Results are deterministic run to run: canonical storage order, fixed reduction order,
 *     no floating-point atomics anywhere.
 *   - Values are FP32, indices int32, nnz and row pointers int64 at the boundary (Table 2,
 *     L198-L202: 12 B/nnz COO, 8 B/nnz CSR).  Inside the handle a layout stores its secondary indices
 *     either as int32 (8 B per entry, the paper's format) or as a u16 offset from a per-32-entry base
 *     (6.125 B per entry); see vmat_ddc_create_ex.
 */
#ifndef VMAT_H
#define VMAT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum vmat_status {
    VMAT_OK = 0,
    VMAT_ERR_INVALID_ARG = -1,   /* NULL pointer, negative size, non-monotone offsets, ...        */
    VMAT_ERR_INDEX_RANGE = -2,   /* a COO voxel / beamlet index outside [0,n)                     */
    VMAT_ERR_DUPLICATE   = -3,   /* the same (voxel, beamlet) pair twice (C14)                    */
    VMAT_ERR_OOM         = -4,   /* device or host allocation failed                              */
    VMAT_ERR_CUDA        = -5,   /* any other CUDA runtime error (message in vmat_last_error)     */
    VMAT_ERR_NONFINITE   = -6    /* a COO value is NaN or +-Inf                                   */
} vmat_status;

/* Opaque handle: owns CSR(D) (voxel rows, for D x), CSR(D^T) (beamlet rows, for D^T g; the
 * paper's GPU format, L121), the offset tables and scratch. */
typedef struct vmat_ddc vmat_ddc;

typedef struct vmat_ddc_info {
    int64_t n_voxels, n_beamlets, nnz, n_angles, n_leaf_rows;
    int64_t bytes_csr_d;        /* 8*nnz + 8*(n_voxels+1): plain CSR(D) in the paper's format (Table 2)  */
    int64_t bytes_csr_dt;       /* 8*nnz + 8*(n_beamlets+1)                                             */
    int64_t bytes_device_total; /* everything the handle holds on the device                            */
    int64_t n_dose_blocks;      /* segments (one warp each) of the dose kernel                          */
    int64_t max_leaf_row_len;   /* longest leaf row, in beamlets                                        */
    int64_t max_voxel_row_nnz, max_beamlet_row_nnz;
    int64_t index_bits_d, index_bits_dt;     /* 16 or 32: index encoding chosen for each layout          */
    int64_t padded_d, padded_dt;             /* stored entries incl. pads (multiples of 32), >= nnz      */
    int64_t bytes_stream_d;     /* bytes vmat_dose streams per call: values + indices (+ bases) of the
                                   padded entries + int64 row starts + the int32 segment table           */
    int64_t bytes_stream_dt;    /* bytes vmat_price streams per call: the same for D^T (no segment table) */
    int64_t tiles_d, tiles_uniform_d;        /* u16 layouts: 256-entry tiles, and those stored with ONE base     */
    int64_t tiles_dt, tiles_uniform_dt;      /* (span <= 65535) instead of one per 32-entry group; 0 for int32   */
    int64_t grid_dose, grid_price;           /* CTAs the dose and the price kernel are launched with (bench.py checks
                                                a stored ncu capture against them before quoting its DRAM traffic)  */
    int64_t sm_affine_dose, sm_affine_price; /* 1: the kernel draws its items from per-SM queues (vmat_ddc_set_schedule) */
} vmat_ddc_info;

/* A0 ingest / layout build (D arrives as COO - values, voxel (row) index,
 * beamlet (column) index, equal length, any order - and is converted to CSR "at the
 * initialization stage").  Builds both layouts on the device, rows in canonical order (sorted by
 * the secondary index).
 *   coo_*               host OR device pointers, length nnz (detected with cudaPointerGetAttributes);
 *                       the caller may free them when the call returns.
 *   angle_col_offset    host [n_angles+1]: beamlets of control point a are columns [off[a], off[a+1])
 *                       (the angle blocks D = [D_1 ... D_A] of L119); off[0] = 0, off[n_angles] = n_beamlets.
 *   angle_row_offset    host [n_angles+1]: MLC leaf rows of control point a.
 *   leafrow_col_offset  host [n_leaf_rows+1], n_leaf_rows = angle_row_offset[n_angles]: beamlets of a
 *                       leaf row, left to right; leaf rows do not straddle control points.
 * Synchronous (returns after the build finished).  Validates index ranges, finiteness, duplicates
 * and offset tables.  Empty rows, empty columns and nnz = 0 are legal. */
int vmat_ddc_create(vmat_ddc **out, int32_t n_voxels, int32_t n_beamlets, int64_t nnz,
                    const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                    int32_t n_angles, const int32_t *angle_col_offset, const int32_t *angle_row_offset,
                    const int32_t *leafrow_col_offset, void *stream);

/* Same, with the index encoding of the two layouts chosen by the caller:
 *   index_bits = 32  int32 secondary indices, 8 B per stored entry (the paper's CSR, Table 2);
 *   index_bits = 16  u16 offsets from one int32 base per group of 32 stored entries, 6.125 B per entry; a
 *                    group whose indices would span more than 65535 is closed early and padded, so any
 *                    matrix can be stored;
 *   index_bits = 0   per layout, 16 if that is at least 5 % smaller than 32, else 32 (what
 *                    vmat_ddc_create does).
 * Results are deterministic for a given setting.  Across settings they are bit-identical whenever no group
 * had to be closed early (always when the layout's secondary dimension is <= 65536); otherwise the pads
 * shift entries between the lanes' partial sums and the FP32 results differ by summation order only. */
int vmat_ddc_create_ex(vmat_ddc **out, int32_t n_voxels, int32_t n_beamlets, int64_t nnz,
                       const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                       int32_t n_angles, const int32_t *angle_col_offset, const int32_t *angle_row_offset,
                       const int32_t *leafrow_col_offset, int32_t index_bits, void *stream);

/* Frees the layouts and scratch.  NULL is a no-op. */
int vmat_ddc_destroy(vmat_ddc *h);

int vmat_ddc_info_get(const vmat_ddc *h, vmat_ddc_info *info /* host, out */);

/* Test/debug: copies one layout to host arrays.  which = 0: CSR(D) (rows = voxels, idx = beamlets),
 * which = 1: CSR(D^T) (rows = beamlets, idx = voxels).  ptr [rows+1], idx/val [nnz] in canonical CSR order
 * (the grouping, padding, tile interleave and index encoding of the device layout are undone); idx = val = NULL copies the row pointers only.
 * Synchronous. */
int vmat_ddc_export_csr(const vmat_ddc *h, int which, int64_t *ptr, int32_t *idx, float *val /* host, out */);

/* A1 forward dose d = D x, d_i = sum_j D_ij x_j ("repeated forward dose
 * calculation", L27).  x dev [n_beamlets] in, d dev [n_voxels] out.
 * The handle is const for the caller but holds scratch the launch writes (the reordered copy of x, the work-queue
 * counters of the persistent schedule): as for every compute call, ONE launch per handle may be in flight at a time;
 * two streams must be ordered with an event.  Overlapping launches give wrong or stale outputs without an error;
 * vmat_ddc_set_schedule puts the queue counters back in order afterwards. */
int vmat_dose(const vmat_ddc *h, const float *x, float *d, void *stream);

/* A2 objective and gradient (Eq. (1); Eq. (4)):
 *   F   = sum_i w_over[s_i] max(0, d_i - T[s_i])^2 + w_under[s_i] max(0, T[s_i] - d_i)^2
 *   g_i = dF/dd_i = 2 w_over[s_i] max(0, d_i - T[s_i]) - 2 w_under[s_i] max(0, T[s_i] - d_i)
 * with s_i = voxel_struct[i] (C9).  Sign: the paper's g is -grad F and its price pi is maximised;
 * here g = +grad F, p = -pi is minimised - identical selections (C1).  w_over = omega+ (overdose),
 * w_under = omega- (C10).
 *   d dev [n_voxels] in; voxel_struct dev u8 [n_voxels]; T, w_over, w_under dev [n_struct], n_struct <= 256;
 *   g dev [n_voxels] out; F dev double [1] out (FP64 sum in a fixed order). */
int vmat_objective_grad(const vmat_ddc *h, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                        const float *T, const float *w_over, const float *w_under,
                        float *g, double *F, void *stream);

/* A2 once more, for callers that cannot allocate device memory: no handle, no cudaMalloc / cudaFree, no allocating
 * library routine, neither in this call nor before it.  Meant for code that runs where an allocation is forbidden or
 * impossible: a host application that gave the whole GPU to its own memory pool at start-up, a latency-bound control
 * loop that must stay clear of the driver's allocation lock (cudaMalloc may wait for the whole device), a plug-in whose
 * host forbids driver allocations once it is initialised.  vmat_objective_grad does not fit them because its scratch lives in a vmat_ddc, and vmat_ddc_create allocates.
 *   Arguments and results are those of vmat_objective_grad with n_voxels passed in place of the handle; F and g are
 * bit-identical to vmat_objective_grad's.  Works on the current device; enqueues two kernels on `stream`.
 *   Scratch: the per-block FP64 partial sums of F sit in an array compiled into the library (256 KiB; every GPU that
 * loads libvmat.so holds it until the process exits).  Hence the limit: n_voxels <= VMAT_OBJECTIVE_STATIC_MAX_VOXELS,
 * beyond it the call returns VMAT_ERR_INVALID_ARG and vmat_last_error() names the limit.
 *   First call on a device: looks up the array's device address (cudaGetSymbolAddress, no allocation) and keeps it.
 * Make that first call outside any stream capture, e.g. once at start-up with n_voxels = 0.
 *   Sharing: all calls on a device, from every thread and stream, use the same array.  Calls that follow one another on
 * one stream are fine - each call overwrites every slot it later reads, so nothing has to be cleared and leftovers of
 * an earlier call are never seen.  Two calls whose kernels may run at the same time (different streams, no event between
 * them) race on the array and return a wrong F; order them yourself. */
#define VMAT_OBJECTIVE_STATIC_MAX_VOXELS (1 << 23)
int vmat_objective_grad_static(int32_t n_voxels, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                               const float *T, const float *w_over, const float *w_under,
                               float *g, double *F, void *stream);

/* A3 beamlet prices p = D^T g, p_j = sum_i D_ij g_i (Eq. (3); "Pi = D^T g", L121; one warp per
 * beamlet row as in L127).  g dev [n_voxels] in, p dev [n_beamlets] out.  One launch per handle in flight at a time
 * (the work-queue counters and, in the fused calls, the leaf-row tickets belong to the handle; see vmat_dose). */
int vmat_price(const vmat_ddc *h, const float *g, float *p, void *stream);

/* Contract check for the objective arguments of every call that takes them: voxel_struct dev u8 [n_voxels] must hold
 * ids < n_struct (they index T / w_over / w_under; the compute calls do not re-check them on the device: an id
 * beyond n_struct reads past the tables).  Synchronous.  Returns VMAT_ERR_INDEX_RANGE if an id is out of range,
 * VMAT_ERR_INVALID_ARG for n_struct outside 1..256. */
int vmat_check_structure_ids(const uint8_t *voxel_struct, int32_t n_voxels, int32_t n_struct, void *stream);

/* A4 + A5 aperture selection without interdigitation (L133): for every MLC leaf row the contiguous
 * opening [L,R) (beamlet columns within the row, 0 <= L <= R <= n_row; C8) minimising the summed
 * price, the closed opening (value 0, L = R = 0) included (C4); then per control point the sum of its
 * rows' best prices, and the control point with the smallest sum.
 * Arithmetic (C5, C6): S_0 = 0, S_{c+1} = S_c + (double)p[j0+c] left to right in FP64; candidates all
 * 0 <= L <= R <= n with V = S_R - S_L; the result is the smallest candidate in the order (V, L, R).
 *   p dev [n_beamlets] in; angle_mask dev u8 [n_angles] or NULL (1 = occupied control point: its rows
 *   stay closed, angle_price = +inf; C7);
 *   L, R dev int32 [n_leaf_rows]; row_price dev double [n_leaf_rows]; angle_price dev double [n_angles]
 *   (sum in row order, FP64); best_angle dev int32 [1]: smallest control point attaining the minimum
 *   among unoccupied ones, or -1 when that minimum is >= 0 (no improving aperture, L56). */
int vmat_select_apertures(const vmat_ddc *h, const float *p, const uint8_t *angle_mask,
                          int32_t *L, int32_t *R, double *row_price, double *angle_price,
                          int32_t *best_angle, void *stream);

/* One whole price evaluation A1 -> A5 with the fused kernels: (dose + objective/gradient) then
 * (price + row opening) then aperture price.  Same arguments and outputs as the four calls above;
 * every output vector is written (d, g, p included). */
int vmat_price_eval(const vmat_ddc *h, const float *x,
                    const uint8_t *voxel_struct, int32_t n_struct,
                    const float *T, const float *w_over, const float *w_under,
                    const uint8_t *angle_mask,
                    float *d, float *g, double *F, float *p,
                    int32_t *L, int32_t *R, double *row_price, double *angle_price,
                    int32_t *best_angle, void *stream);

/* A3 -> A5 with the fused kernels, from a gradient the caller already holds: (price + row opening), aperture price.
 * This is the second half of vmat_price_eval; the angle-sharded multi-GPU path (NEXT-4) calls it after the
 * all-reduce of the dose.  Arguments as for vmat_price and vmat_select_apertures. */
int vmat_price_select(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p, int32_t *L, int32_t *R,
                      double *row_price, double *angle_price, int32_t *best_angle, void *stream);

/* End-to-end variant with HOST buffers: copies x (host, ideally pinned, [n_beamlets]) to the device,
 * runs vmat_price_eval on device scratch owned by the handle, copies F, L, R, row_price, angle_price
 * and best_angle back to the host arrays, and synchronises the stream before returning.
 * The objective tables (voxel_struct, T, w_over, w_under, angle_mask) are device pointers as above. */
int vmat_price_eval_host(vmat_ddc *h, const float *x_host,
                         const uint8_t *voxel_struct, int32_t n_struct,
                         const float *T, const float *w_over, const float *w_under,
                         const uint8_t *angle_mask,
                         double *F_host, int32_t *L_host, int32_t *R_host, double *row_price_host,
                         double *angle_price_host, int32_t *best_angle_host, void *stream);

/* The same end-to-end call, pipelined over two slots so that the host <-> device copies of one evaluation overlap the
 * kernels of the other: _submit enqueues, for slot 0 or 1, the copy of x_host (pinned host memory) on a copy-in
 * stream, the evaluation on `stream`, and the copies of the results into the host buffers on a copy-out stream, and
 * returns at once; _wait blocks until that slot's host outputs are complete.  A slot must be waited for before it
 * is submitted again; x_host and the output buffers of a slot belong to the library between _submit and _wait.
 * The objective arguments are device pointers as in vmat_price_eval.  Results are identical to vmat_price_eval_host. */
int vmat_price_eval_host_submit(vmat_ddc *h, int32_t slot, const float *x_host,
                                const uint8_t *voxel_struct, int32_t n_struct,
                                const float *T, const float *w_over, const float *w_under,
                                const uint8_t *angle_mask,
                                double *F_host, int32_t *L_host, int32_t *R_host, double *row_price_host,
                                double *angle_price_host, int32_t *best_angle_host, void *stream);
int vmat_price_eval_host_wait(vmat_ddc *h, int32_t slot);

/* Aperture dose vector DA(A_k) = sum_{j in A_k} D_:j (Eq. (5)) of the aperture given by the
 * openings [L,R) of the leaf rows of control point `angle`: DA = D 1_A, on the device (the paper did
 * this on the CPU from COO, L137).  L, R dev int32 [n_leaf_rows] (as written by the selection);
 * x_scratch dev [n_beamlets] (overwritten with the indicator); DA dev [n_voxels] out.
 * Only the beamlet rows of that control point are read (layout D^T); their entries are summed per voxel in 64-bit
 * fixed point (exact, order-free), so DA is deterministic and within one FP32 rounding of the exact sum. */
int vmat_aperture_dose(const vmat_ddc *h, int32_t angle, const int32_t *L, const int32_t *R,
                       float *x_scratch, float *DA, void *stream);

/* ------------------------------------------------------------------------------------------------------
 * NEXT-3: aperture selection under MLC hardware constraints.
 *
 * MLC geometry, once per handle: leafrow_pos0 host int32 [n_leaf_rows] = physical column (in beamlet widths, on
 * the control point's own grid) of the first beamlet of every leaf row (ignored for rows without beamlets).  The
 * field range of a control point is [Pmin, Pmax] = [min pos0, max pos0 + n] over its non-empty rows and may span
 * at most 254 beamlet widths (255 leaf positions); the longest leaf row is bounded by the SM's shared memory ((n+1)^2 table entries of
 * 10 bytes: about 145 beamlets on B200).  Returns VMAT_ERR_INVALID_ARG beyond either.  Synchronous. */
int vmat_ddc_set_leaf_geometry(vmat_ddc *h, const int32_t *leafrow_pos0);

/* A4 + A5 with constraints.  A leaf row has a state (a, b), a <= b: the physical positions of its two leaf ends;
 * row-local L = a - pos0, R = b - pos0 (C8).  Open states (a < b) lie inside the row's beamlets, 0 <= L < R <= n;
 * a closed pair (a == b, value 0) may be parked anywhere in the control point's field range, so for a closed row
 * L = R may be negative or exceed n (rows without beamlets count from Pmin).  Readings C22-C24:
 *   interdigitation != 0: adjacent rows r, r+1 of a control point must satisfy a_r <= b_{r+1} and a_{r+1} <= b_r
 *       (L135: "L_{k,irow} <= min{R_{k,irow-1}, R_{k,irow+1}}", for every row, closed ones included);
 *   windows (L66: apertures "compatible with those chosen" at neighbouring control points): L_lo[r] <= L <= L_hi[r],
 *       R_lo[r] <= R <= R_hi[r]; each of the four dev int32 [n_leaf_rows] arrays may be NULL (no bound).
 * Per control point the aperture minimising the summed price over ALL feasible combinations of row states is
 * returned (the paper enumerates them; here a row-by-row recursion with exact minima): value of a state V = S_R -
 * S_L as in vmat_select_apertures (C6), aperture price = V_last + (... + (V_1 + V_0)).  Ties: the last row takes its
 * smallest optimal state in (a, b) order, every earlier row the smallest state attaining the minimum it feeds.  A
 * control point without a feasible combination (or occupied, angle_mask) gets price +inf and L = R = 0.  Unlike
 * vmat_select_apertures an aperture is reported even when its price is >= 0; best_angle is -1 then.
 * Outputs as vmat_select_apertures; bit-identical to the oracle on the same FP32 p.  Asynchronous. */
int vmat_select_apertures_constrained(vmat_ddc *h, const float *p, const uint8_t *angle_mask, int32_t interdigitation,
                                      const int32_t *L_lo, const int32_t *L_hi, const int32_t *R_lo,
                                      const int32_t *R_hi, int32_t *L, int32_t *R, double *row_price,
                                      double *angle_price, int32_t *best_angle, void *stream);

/* Leaf-travel windows (L66: candidate apertures "need to be compatible with those chosen" at neighbouring control
 * points, through s_k <= S^U_{k,k+1}(A_k, A_{k+1}); PAPER.md does not define S^U - reading C25): a leaf end moves at
 * most max_leaf_travel beamlet widths per control-point step.  For every leaf row of every UNOCCUPIED control point
 * k (angle_mask[k] == 0) the nearest occupied control point k' on either side of k within k's arc bounds both leaf
 * ends of the same leaf row: |a_k - a_k'| <= max_leaf_travel |k - k'|, likewise b.  Writes the windows row-local,
 * -2^30 / +2^30 where nothing binds (all rows of occupied control points).
 *   angle_mask dev u8 [n_angles]; L, R dev int32 [n_leaf_rows]: openings of the occupied control points (row-local);
 *   arc_angle_offset host int32 [n_arcs+1], n_arcs <= 16: control points of every arc, each arc with one MLC (the
 *   same number of leaf rows at all its control points);  L_lo .. R_hi dev int32 [n_leaf_rows] out.
 * Needs vmat_ddc_set_leaf_geometry.  Asynchronous. */
int vmat_leaf_windows(const vmat_ddc *h, const uint8_t *angle_mask, const int32_t *L, const int32_t *R, int32_t n_arcs,
                      const int32_t *arc_angle_offset, int32_t max_leaf_travel, int32_t *L_lo, int32_t *L_hi,
                      int32_t *R_lo, int32_t *R_hi, void *stream);

/* ------------------------------------------------------------------------------------------------------
 * NEXT-2: the master problem (MP), Eq. (6)-(10) L70-L101 and the four BB steps of L139.
 * With the apertures chosen so far and their dose vectors DA(A_k) (Eq. (5)), find fluence rates
 * y_k in [y_lo_k, y_hi_k] (Eq. (6): R^L/S^U_k and R^U/S^L_k, supplied by the caller) minimising F(z),
 * z = sum_k DA(A_k) y_k, by the Barzilai-Borwein iteration: step sizes Eq. (7) and Eq. (8) alternately,
 * subspace step rule Eq. (9)/(10), three stopping rules (L101).  Readings C15-C20 of DESIGN.md:
 * g_A = +dF/dy and y <- y - delta g_A; a variable at its lower (upper) bound with g_A > 0 (< 0) is held and
 * its gradient entry zeroed; y is clipped into the box after every update; first step = exact line minimiser
 * of the current quadratic piece; iteration 1, 3, .. use Eq. (7), 2, 4, .. Eq. (8), the previous delta is kept
 * when <s,t> <= 0; z is recomputed as DA y every iteration.
 * The handle owns a dense copy of the aperture dose vectors in blocks of 32 apertures, voxel-major inside a block
 * (float [ceil(max_apertures / 32)][n_voxels rounded up to 16][32], max_apertures <= 384: one voxel's 32 coefficients
 * of a block are one 128-byte line; rows of voxels no aperture reaches are never read) and the FP64 iteration state; y persists between solves (warm start, as in the
 * column-generation loop L56).  All sums are FP64 in a fixed order: results are deterministic. */
typedef struct vmat_mp vmat_mp;
int vmat_mp_create(vmat_mp **out, int32_t n_voxels, int32_t max_apertures, void *stream);
int vmat_mp_destroy(vmat_mp *h);
/* Forgets every aperture (the storage is kept).  Enqueued on `stream`, like every other call. */
int vmat_mp_reset(vmat_mp *h, void *stream);
/* Appends aperture k = current count: DA dev float [n_voxels] (e.g. from vmat_aperture_dose), its starting
 * fluence rate y0 (clipped into the box) and bounds.  Asynchronous: the three scalars travel through a pinned
 * staging buffer of the handle. */
int vmat_mp_add_aperture(vmat_mp *h, const float *DA, double y0, double y_lo, double y_hi, void *stream);
/* Overwrites the fluence rates of the current apertures (y_host host double [count]); clipped by the solve. */
int vmat_mp_set_fluence(vmat_mp *h, const double *y_host, void *stream);
int vmat_mp_size(const vmat_mp *h, int32_t *n_apertures, int32_t *max_apertures /* host, out, may be NULL */);
/* Voxels that at least one of the current apertures reaches (a non-zero in their row of the aperture dose matrix), as
 * of the last solve.  Only these rows are read by the BB passes (4 m n_reached bytes per iteration); the dose of the
 * others is 0 whatever y, and their constant terms of Eq. (1) are added to F once per solve. */
int vmat_mp_reached_voxels(const vmat_mp *h, int32_t *n_reached /* host, out */);
/* Launch geometry of the solve kernel for m apertures on this handle's device: CTAs of the grid and the number of
 * voxel rows the whole grid takes per step of the grid-stride loop of a pass (parity tests size their cases with it so that
 * the loop's steady state is reached).  Either output may be NULL. */
int vmat_mp_pass_geometry(const vmat_mp *h, int32_t m, int32_t *n_cta, int32_t *rows_per_grid_step /* host, out */);
/* Runs the BB iteration from the handle's current y until a stopping rule fires (tested at the top of every
 * iteration, in this order):  reason 1 "stationary": every entry of g_A is 0 after the subspace rule;
 * 2 "objective": it >= 5 and |F(j) - F(j-1)| <= eps_F |F(j-1)| for the five latest j;  3 "step": it >= 1 and
 * max_k |y_k(it) - y_k(it-1)| <= eps_y;  4: it == max_iter.  The iterate at which the rule fired is returned.
 *   voxel_struct, T, w_over, w_under: the objective, as for vmat_objective_grad (device pointers);
 *   z dev float [n_voxels] out or NULL: the dose z = DA y of the returned iterate;
 *   y_host double [count], F_host, n_iter_host, reason_host: host, out, each may be NULL.
 * The whole iteration runs in ONE cooperative kernel launch (one persistent CTA per SM; the stopping rules are
 * evaluated on the device); the call synchronises the stream once, at the end, to return the host outputs. */
int vmat_mp_solve(vmat_mp *h, const uint8_t *voxel_struct, int32_t n_struct, const float *T, const float *w_over,
                  const float *w_under, int32_t max_iter, double eps_F, double eps_y, float *z, double *y_host,
                  double *F_host, int32_t *n_iter_host, int32_t *reason_host, void *stream);
/* Trace of the last solve: F_hist host double [n_iter + 1] (objective at iterate 0 .. n_iter), delta_hist host
 * double [n_iter] (step size used to leave iterate it); either may be NULL. */
int vmat_mp_history(const vmat_mp *h, double *F_hist, double *delta_hist);

/* The column-generation loop (Figure 1(a)): start with z = 0 and no apertures; repeat { PP1: g =
 * dF/dz, p = D^T g;  PP2: best opening per leaf row of the unoccupied control points, best control point; stop if
 * none has a negative price;  Eq. (5): its aperture dose vector;  MP: fluence rates of all apertures so far (BB,
 * warm-started, the new aperture at 0 clipped into [y_lo, y_hi]) } until max_apertures.  Every step runs on the
 * device; `mp` is reset first and holds the apertures afterwards (capacity >= max_apertures).  Neighbour
 * compatibility of apertures (L50-L54, L66) is not modelled (C7, C21): every aperture gets the bounds [y_lo, y_hi].
 *   z dev float [n_voxels] out: final dose;  L, R dev int32 [n_leaf_rows] out: openings of the chosen control
 *   points, 0 elsewhere;  host outputs (each but n_apertures_host may be NULL): n_apertures_host [1];
 *   angles_host int32 [max_apertures] (control point of aperture k, in the order chosen);  y_host double
 *   [max_apertures];  F_hist_host double [max_apertures + 1] (F(0), then F after every master problem);
 *   aperture_price_host double [max_apertures] (price of aperture k when chosen, < 0);  mp_iters_host int32
 *   [max_apertures];  stop_host [1]: 0 = no improving aperture left, 1 = max_apertures reached.  Synchronous. */
int vmat_column_generation(vmat_ddc *h, vmat_mp *mp, const uint8_t *voxel_struct, int32_t n_struct, const float *T,
                           const float *w_over, const float *w_under, int32_t max_apertures, double y_lo, double y_hi,
                           int32_t mp_max_iter, double eps_F, double eps_y, float *z, int32_t *L, int32_t *R,
                           int32_t *n_apertures_host, int32_t *angles_host, double *y_host, double *F_hist_host,
                           double *aperture_price_host, int32_t *mp_iters_host, int32_t *stop_host, void *stream);

/* The same loop with the pricing problem under hardware constraints (NEXT-3): interdigitation != 0 applies
 * inside every new aperture, max_leaf_travel >= 0 (with n_arcs, arc_angle_offset as for vmat_leaf_windows; < 0 =
 * off) keeps every new aperture reachable from the occupied control points next to it (C25).  With both off this
 * is vmat_column_generation.  The loop also stops (stop 0) when the best feasible aperture has a price >= 0.  Closed
 * rows of a chosen aperture report their parked position in L = R. */
int vmat_column_generation_ex(vmat_ddc *h, vmat_mp *mp, const uint8_t *voxel_struct, int32_t n_struct, const float *T,
                              const float *w_over, const float *w_under, int32_t max_apertures, double y_lo, double y_hi,
                              int32_t mp_max_iter, double eps_F, double eps_y, int32_t interdigitation,
                              int32_t max_leaf_travel, int32_t n_arcs, const int32_t *arc_angle_offset, float *z,
                              int32_t *L, int32_t *R, int32_t *n_apertures_host, int32_t *angles_host, double *y_host,
                              double *F_hist_host, double *aperture_price_host, int32_t *mp_iters_host,
                              int32_t *stop_host, void *stream);

/* NEXT-4 (angle shards): the A5 rule across column blocks, on the device.
 * vmat_best_pair: this block's candidate as a pair of doubles {aperture price, control point in GLOBAL numbering}
 *   from the outputs of vmat_price_select / vmat_price_eval on the block (angle_price dev double [n_angles of the
 *   block], best_angle dev int32 [1], local numbering); {0.0, -1.0} when the block has no improving aperture.
 * vmat_merge_best: the rule of A5 over n such pairs (dev double [n][2], e.g. all-gathered over the ranks): smallest
 *   price, ties -> smallest control point, none below 0 -> {0.0, -1.0}; result in best dev double [2].
 * Both enqueue one tiny kernel on `stream`; nothing comes to the host. */
int vmat_best_pair(const vmat_ddc *h, const double *angle_price, const int32_t *best_angle, int32_t angle_lo,
                   double *pair, void *stream);
int vmat_merge_best(const double *pairs, int32_t n, double *best, void *stream);

/* Profiling hook for bench.py's roofline: four CUDA events (cudaEvent_t passed as void*, any may be NULL)
 * that every following vmat_price_eval / vmat_price_eval_host on this handle records on its stream:
 * ev[0] just before and ev[1] just after the dose(+objective) kernel, ev[2] just before and ev[3] just
 * after the price(+row opening) kernel.  Pass NULL for `ev` to clear.  The events stay owned by the caller. */
int vmat_ddc_set_profile_events(vmat_ddc *h, void *const *ev /* host [4] or NULL */);

/* Work distribution of the two streaming kernels (vmat_dose, vmat_price and every fused call).
 *   sm_affine = 1   persistent kernels, SM count x resident CTAs per SM; the items (4 voxel segments; 8 beamlet rows)
 *                   are cut into one contiguous queue per SM with equal stored bytes, and a CTA draws from the queue of
 *                   the SM it runs on, then from the next non-empty one: the CTAs resident on an SM work on
 *                   neighbouring items, whose gathers of x / g overlap.
 *   sm_affine = 0   one CTA per item, in the order the hardware dispatches them.
 *   sm_affine = -1  (what vmat_ddc_create sets) per kernel, 1 where the layout has >= 16 items per resident CTA of
 *                   >= 64 KB each, else 0; vmat_ddc_info.sm_affine_dose / _price say which.
 * Every output is bit-identical under all settings (an item's sums have a fixed order).  Takes effect from the
 * next launch; not to be called while a launch on this handle is in flight.  Also zeroes the queue counters (they reset
 * themselves after every completed launch; this repairs them after an aborted or overlapping one) and waits for that:
 * synchronises the legacy default stream. */
int vmat_ddc_set_schedule(vmat_ddc *h, int32_t sm_affine);

/* Thread-local, static storage; never NULL. */
const char *vmat_last_error(void);

/* Number of kernels the last compute call on this thread launched (bench.py's gpu_launches). */
int vmat_last_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* VMAT_H */
