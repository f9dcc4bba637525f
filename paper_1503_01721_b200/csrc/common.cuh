// common.cuh - handle layout, error plumbing and load helpers shared by the libvmat kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <limits.h>
#include <vector>
#include <atomic>
#include "../../include/vmat.h"
#include "smqueue.cuh"
// items a CTA takes per visit to its SM's queue (smqueue.cuh): one atomic per chunk.  Measured on B200 (config 3, dose
// kernel): 1: 2.81 ms, 2: 2.88, 4: 2.94, 8: 3.02 - a CTA that keeps several consecutive items to itself takes them
// away from the CTAs beside it, which is the sharing the queues exist for.
#ifndef VMAT_DOSE_QUEUE_CHUNK
#define VMAT_DOSE_QUEUE_CHUNK 1
#endif
#ifndef VMAT_PRICE_QUEUE_CHUNK
#define VMAT_PRICE_QUEUE_CHUNK 1
#endif
constexpr int DOSE_QUEUE_CHUNK = VMAT_DOSE_QUEUE_CHUNK, PRICE_QUEUE_CHUNK = VMAT_PRICE_QUEUE_CHUNK;

// ------------------------------------------------------------------ error plumbing
void vmat_set_error(const char *fmt, ...);
extern thread_local int g_vmat_launches;

#define VMAT_CUDA(call)                                                                     \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            vmat_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? VMAT_ERR_OOM : VMAT_ERR_CUDA;        \
        }                                                                                   \
    } while (0)

#define VMAT_LAUNCH_CHECK()                                                                 \
    do {                                                                                    \
        ++g_vmat_launches;                                                                  \
        cudaError_t e_ = cudaGetLastError();                                                \
        if (e_ != cudaSuccess) {                                                            \
            vmat_set_error("%s:%d: kernel launch -> %s", __FILE__, __LINE__, cudaGetErrorString(e_)); \
            return VMAT_ERR_CUDA;                                                           \
        }                                                                                   \
    } while (0)

// Resident CTAs per SM of a persistent kernel on the handle's device, asked once per (kernel instance, device) - not
// once per process: a process may hold handles on GPUs (or MIG slices) of different size.  `table` is the calling
// template instance's own static array, zero-initialised; a racing first call asks twice and stores the same value.
constexpr int VMAT_MAX_DEVICES = 64;
template <typename Kernel>
static inline int vmat_resident_ctas(Kernel kernel, int threads, int device, std::atomic<int> *table)
{
    const bool cached = device >= 0 && device < VMAT_MAX_DEVICES;
    int o = cached ? table[device].load(std::memory_order_relaxed) : 0;
    if (o > 0) return o;
    int cur = device;
    cudaGetDevice(&cur);
    if (cur != device) cudaSetDevice(device);                 // the occupancy query answers for the current device
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kernel, threads, 0) != cudaSuccess) { o = 0; cudaGetLastError(); }
    if (cur != device) cudaSetDevice(cur);
    o = o > 0 ? o : 1;
    if (cached) table[device].store(o, std::memory_order_relaxed);
    return o;
}

// ------------------------------------------------------------------ one matrix layout on the device
// A layout is a PADDED, GROUPED CSR (spmv.cuh): the rows are cut into segments (one warp each), every
// segment starts at a multiple of 32 padded positions and is a whole number of 32-entry groups.
//   narrow (index_bits 16): val f32[P], off u16[P], base i32[P/32]: secondary index = base[group] + off
//   wide   (index_bits 32): val f32[P], idx i32[P]                 (the paper's 8 B/nnz format, Table 2)
// ptr holds the canonical (unpadded) row pointers, pptr the padded position of each row's first entry.
struct PackedLayout {
    int32_t n_rows = 0;
    int64_t nnz = 0;          // real entries
    int64_t P = 0;            // padded entries (multiple of 32)
    int index_bits = 32;      // 16 or 32
    int64_t n_tiles = 0, n_tiles_uniform = 0;   // narrow: full tiles, and those with one base for all 8 groups
    int64_t *ptr = nullptr;   // [n_rows+1] canonical row pointers
    int64_t *pptr = nullptr;  // [n_rows+1] padded row starts; pptr[n_rows] = P
    float *val = nullptr;     // [P (+pad)]
    void *sec = nullptr;      // narrow: uint16_t off[P (+pad)];  wide: int32_t idx[P (+pad)]
    int32_t *base = nullptr;  // narrow: [P/32 (+pad)];           wide: unused (NULL)
    int32_t n_sec = 0;        // size of the secondary dimension (length of the vector the product gathers from)
    int64_t bytes() const     // device bytes of the streams a product reads (values + indices + padded row starts)
    {
        return index_bits == 16 ? 6 * P + 4 * (P / 32) + 8 * ((int64_t)n_rows + 1)
                                : 8 * P + 8 * ((int64_t)n_rows + 1);
    }
};

// Device view handed to the kernels.
//
// Checked build (`python -m paper_1503_01721_b200.build --force -DVMAT_CHECKED`; compute-sanitizer is not available on
// the B200 pool this was developed on): the view also carries the layout's extent, and every stream access and every
// gathered index of the kernels that walk a layout (k_dose, k_price, k_aperture_scatter) is asserted against it -
// pads, tails after the last full tile and early-closed groups included.  A violation traps the kernel and the next
// CUDA call returns cudaErrorAssert, which fails whatever test is running.  The normal build compiles none of it.
struct MatView {
    const float *val;
    const void *sec;
    const int32_t *base;
#ifdef VMAT_CHECKED
    int64_t P;               // stored entries
    int32_t n_sec;           // valid secondary indices are [0, n_sec)
#endif
};
#ifdef VMAT_CHECKED
#include <assert.h>
static inline MatView view_of(const PackedLayout &A) { return MatView{A.val, A.sec, A.base, A.P, A.n_sec}; }
#define VMAT_ASSERT_STREAM(A, first, n) assert((int64_t)(first) >= 0 && (int64_t)(first) + (int64_t)(n) <= (A).P)
#define VMAT_ASSERT_INDEX(A, c) assert((unsigned)(c) < (unsigned)(A).n_sec)
#define VMAT_ASSERT(cond) assert(cond)
#else
static inline MatView view_of(const PackedLayout &A) { return MatView{A.val, A.sec, A.base}; }
#define VMAT_ASSERT_STREAM(A, first, n) ((void)0)
#define VMAT_ASSERT_INDEX(A, c) ((void)0)
#define VMAT_ASSERT(cond) ((void)0)
#endif
// kernel variant for a layout (spmv.cuh: FMT_WIDE 0, FMT_NARROW 1, FMT_NARROW_1BASE 2)
static inline int fmt_of(const PackedLayout &A)
{
    return A.index_bits != 16 ? 0 : (A.n_tiles_uniform == A.n_tiles ? 2 : 1);
}

// ------------------------------------------------------------------ the handle
struct vmat_ddc {
    int32_t n_voxels = 0, n_beamlets = 0, n_angles = 0, n_leaf_rows = 0;
    int64_t nnz = 0;
    PackedLayout D;    // rows = voxels,   secondary index = beamlet   (for d = D x)
    PackedLayout Dt;   // rows = beamlets, secondary index = voxel     (for p = D^T g; the paper's format, L121)
    // Column order of CSR(D) (dose.cu): within a control point the beamlets are renumbered in tiles of 8 columns x all
    // leaf rows, so that the ~8 x 8 patch of beamlets a voxel sees at one control point lies in few 128-byte lines of
    // x.  NULL = identity (every leaf row fits one tile).  D^T, p, x at the boundary keep the caller's numbering.
    int32_t *col_perm = nullptr;            // [n_beamlets] caller's beamlet -> position in x_perm / secondary index of D
    float *x_perm = nullptr;                // [n_beamlets] x in that order, refilled by every dose launch
    std::vector<int32_t> h_col_inv;         // host: position -> caller's beamlet (export undoes the renumbering)
    // offset tables (device)
    int32_t *angle_col_offset = nullptr;    // [n_angles+1]
    int32_t *angle_row_offset = nullptr;    // [n_angles+1]
    int32_t *leafrow_col_offset = nullptr;  // [n_leaf_rows+1]
    int32_t *leafrow_angle = nullptr;       // [n_leaf_rows] control point of each leaf row
    // dose kernel work list: segment i (one warp) covers voxel rows [seg_row[i], seg_row[i+1])
    int32_t *seg_row = nullptr;             // [n_seg+1]
    int32_t n_seg = 0;
    int32_t n_blocks = 0;                   // items of the dose kernel = ceil(n_seg / warps per CTA)
    // SM-affine schedule of the two streaming kernels (smqueue.cuh): per SM one contiguous queue of items with equal
    // stored bytes; per kernel 1: persistent CTAs drawing from them, 0: one CTA per item.  vmat_ddc_set_schedule.
    int sched_dose = 0, sched_price = 0, n_sm = 0;
    int32_t *q_start = nullptr;             // [2][n_sm + 1]: dose items, price items
    uint32_t *q_next = nullptr;             // [2][n_sm + 1] self-resetting counters
    SmQueues queues_dose() const { return SmQueues{q_start, q_next, sched_dose && q_start ? n_sm : 0, DOSE_QUEUE_CHUNK}; }
    SmQueues queues_price() const
    {
        return SmQueues{q_start + n_sm + 1, q_next + n_sm + 1, sched_price && q_start ? n_sm : 0, PRICE_QUEUE_CHUNK};
    }
    double *F_partial = nullptr;            // [n_blocks] per-item objective partials
    int32_t n_obj_blocks = 0;               // blocks of the standalone objective kernel
    double *F_partial_obj = nullptr;        // [n_obj_blocks]
    double *S_scratch = nullptr;            // [n_beamlets + n_leaf_rows + 1] prefix sums of the row selection
    int32_t *beamlet_leafrow = nullptr;     // [n_beamlets] leaf row of each beamlet
    uint32_t *angle_ticket = nullptr;       // [1] ticket of the aperture-price kernel (self-resetting)
    uint32_t *leafrow_done = nullptr;       // [n_leaf_rows] tickets of the fused price+selection kernel (self-resetting)
    std::vector<int32_t> h_angle_row_offset; // host copy
    std::vector<int32_t> h_angle_col_offset; // host copy
    unsigned long long *ad_acc = nullptr;    // [n_voxels] fixed-point accumulators of vmat_aperture_dose
    int ad_shift = 0;                        // its scale: 2^ad_shift
    std::vector<int32_t> h_seg_row;          // host copy of seg_row (export undoes the tile interleave)
    int32_t max_leaf_row_len = 0;
    int64_t max_voxel_row_nnz = 0, max_beamlet_row_nnz = 0;
    int64_t bytes_device = 0;
    int device = 0;
    cudaEvent_t prof_ev[4] = {nullptr, nullptr, nullptr, nullptr};   // vmat_ddc_set_profile_events
    // NEXT-3 (constrained.cu): MLC geometry, set by vmat_ddc_set_leaf_geometry
    int32_t *leafrow_pos0 = nullptr;        // [n_leaf_rows] physical column of each leaf row's first beamlet
    int32_t *angle_pmin = nullptr;          // [n_angles] left end of the control point's field range
    int32_t *angle_wd = nullptr;            // [n_angles] positions in the field range (Pmax - Pmin + 1)
    int32_t *angle_order = nullptr;         // [n_angles] launch order of k_cs_dp: heaviest control points first
    int64_t *row_bp_offset = nullptr;       // [n_leaf_rows+1] start of each leaf row's back pointers in cs_bp
    uint16_t *cs_bp = nullptr;              // back pointers of the row-by-row recursion: per row wd + (n+1)^2
    int32_t cs_max_wd = 0, cs_max_n = 0, cs_max_rows = 0;
    // k_cs_dp runs as two concurrent launches: control points whose longest leaf row is <= CS_SMALL_ROW get a small
    // shared-memory table (several CTAs per SM) on an auxiliary stream, the others the full-size table on the caller's
    int32_t cs_bin_off[3] = {0, 0, 0};      // angle_order[off[b] .. off[b+1]): bin 0 = long rows, bin 1 = short rows
    int32_t cs_bin_tab[2] = {1, 1};         // table dimension (longest row + 1) of each bin
    cudaStream_t cs_aux = nullptr;
    cudaEvent_t cs_fork = nullptr, cs_join = nullptr;
    std::vector<int32_t> h_leafrow_pos0;
    // scratch for the end-to-end host call (allocated on first use)
    float *e2e_x = nullptr, *e2e_d = nullptr, *e2e_g = nullptr, *e2e_p = nullptr;
    int32_t *e2e_L = nullptr, *e2e_R = nullptr, *e2e_best = nullptr;
    double *e2e_row_price = nullptr, *e2e_angle_price = nullptr, *e2e_F = nullptr;
    // the two-slot pipelined host call (vmat_price_eval_host_submit / _wait): per slot the device copy of x and of the
    // results, and the events that order copy-in stream -> caller's stream -> copy-out stream
    struct E2ESlot {
        float *x = nullptr;
        int32_t *L = nullptr, *R = nullptr, *best = nullptr;
        double *row_price = nullptr, *angle_price = nullptr, *F = nullptr;
        cudaEvent_t x_ready = nullptr, done = nullptr, out_ready = nullptr;
        bool in_flight = false;
    } slot[2];
    cudaStream_t e2e_in = nullptr, e2e_out = nullptr;
    bool e2e_sync_ready = false, e2e_slots_ready = false;    // set last: every buffer / stream / event above exists
};

// ------------------------------------------------------------------ tuning constants
// Dose kernel: one warp per segment (a long voxel row, or a run of short rows parked in shared memory).
#ifndef VMAT_DOSE_THREADS
#define VMAT_DOSE_THREADS 128
#endif
#ifndef VMAT_DOSE_SEG_NNZ
#define VMAT_DOSE_SEG_NNZ 512
#endif
#ifndef VMAT_DOSE_MINB
#define VMAT_DOSE_MINB 12
#endif
// Depth of the software pipeline of the tile loop (spmv.cuh: tiles whose stream loads are in flight at once).
// Measured on B200 (config 3): the price kernel is fastest at depth 2 and 6 CTAs/SM (40 registers); the dose kernel at
// depth 1 and 12 CTAs of 4 warps - depth 2 spills at 40 registers in its u16 + per-group-base variant and 10 or 8 CTAs
// lose more than the pipeline gains (profiles/r2_sm_affine.md).
#ifndef VMAT_PRICE_DEPTH
#define VMAT_PRICE_DEPTH 2
#endif
#ifndef VMAT_DOSE_DEPTH
#define VMAT_DOSE_DEPTH 1
#endif
constexpr int DOSE_THREADS = VMAT_DOSE_THREADS;
constexpr int DOSE_SEG_NNZ = VMAT_DOSE_SEG_NNZ;   // a warp's run of short rows holds at most this many padded entries
constexpr int DOSE_MAX_ROWS = 256;                // rows per segment (bounds runs of empty rows)
// Price kernel (CSR-vector, one warp per beamlet row, L127).
#ifndef VMAT_PRICE_THREADS
#define VMAT_PRICE_THREADS 256
#endif
constexpr int PRICE_THREADS = VMAT_PRICE_THREADS;
constexpr int PRICE_WARPS = PRICE_THREADS / 32;
constexpr int SELECT_MAX_ROW = 2048;        // longest leaf row the fused price+select kernel takes

// ------------------------------------------------------------------ load helpers
// Matrix streams are read exactly once per evaluation.  sm_100 has 256-bit global loads
// (SASS LDG.E.256); they carry the L2::evict_first priority, and L1::no_allocate keeps the
// stream out of L1, so the 16-64 GB of matrix data do not wash the gathered vector (x or g,
// <= a few MB) out of the caches.  The address must be 32-byte aligned.
struct Vec8 { uint32_t w[8]; };
__device__ __forceinline__ Vec8 ld_stream_256(const void *p)
{
    Vec8 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]),
                   "=r"(r.w[4]), "=r"(r.w[5]), "=r"(r.w[6]), "=r"(r.w[7]) : "l"(p));
    return r;
}
// 128-bit stream load (eight u16 offsets).  The .L2::evict_first qualifier exists only for .v8.b32, so the
// same priority is given through a cache-hint policy.
struct Vec4 { uint32_t w[4]; };
__device__ __forceinline__ Vec4 ld_stream_128(const void *p)
{
    Vec4 r;
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.b32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ int ld_stream_u16(const uint16_t *p)
{
    unsigned short r;
    asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(r) : "l"(p));
    return (int)r;
}
__device__ __forceinline__ float ld_stream_f(const float *p)
{
    float r;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ int ld_stream_i(const int32_t *p)
{
    int r;
    asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}
// Gathered vector (x or g): read-only path, allocated in L1 with evict-last priority.
__device__ __forceinline__ float ld_gather(const float *p)
{
    float r;
    asm volatile("ld.global.nc.L1::evict_last.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}

// ------------------------------------------------------------------ internal entry points
int vmat_build_layouts(vmat_ddc *h, const int32_t *coo_voxel, const int32_t *coo_beamlet,
                       const float *coo_val, int index_bits, cudaStream_t st);
int vmat_dose_grid(const vmat_ddc *h, bool fuse);      // CTAs of the dose launch (fused or plain)
int vmat_price_grid(const vmat_ddc *h);                // CTAs of the fused price + selection launch
int vmat_launch_dose(const vmat_ddc *h, const float *x, float *d, bool fuse,
                     const uint8_t *voxel_struct, int32_t n_struct, const float *T, const float *w_over,
                     const float *w_under, float *g, double *F, cudaStream_t st);
int vmat_launch_objective(const vmat_ddc *h, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                          const float *T, const float *w_over, const float *w_under, float *g, double *F,
                          cudaStream_t st);
int vmat_launch_price(const vmat_ddc *h, const float *g, float *p, cudaStream_t st);
int vmat_launch_select(const vmat_ddc *h, const float *p, const uint8_t *angle_mask, int32_t *L, int32_t *R,
                       double *row_price, cudaStream_t st);
int vmat_launch_price_select(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p,
                             int32_t *L, int32_t *R, double *row_price, cudaStream_t st, bool skip_occupied = false);
int vmat_launch_price_unoccupied(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p, cudaStream_t st);
int vmat_launch_angle_price(const vmat_ddc *h, const double *row_price, const uint8_t *angle_mask,
                            double *angle_price, int32_t *best_angle, cudaStream_t st);
int vmat_launch_best_pair(const vmat_ddc *h, const double *angle_price, const int32_t *best_angle, int32_t angle_lo,
                          double *pair, cudaStream_t st);
int vmat_launch_merge_best(const double *pairs, int32_t n, double *best, cudaStream_t st);
int vmat_launch_select_constrained(vmat_ddc *h, const float *p, const uint8_t *angle_mask, int interdigitation,
                                   const int32_t *L_lo, const int32_t *L_hi, const int32_t *R_lo, const int32_t *R_hi,
                                   int32_t *L, int32_t *R, double *row_price, double *angle_price, int32_t *best_angle,
                                   cudaStream_t st);
int vmat_launch_leaf_windows(const vmat_ddc *h, const uint8_t *angle_mask, const int32_t *L, const int32_t *R,
                              int32_t n_arcs, const int32_t *arc_angle_offset, int32_t max_leaf_travel, int32_t *L_lo,
                              int32_t *L_hi, int32_t *R_lo, int32_t *R_hi, cudaStream_t st);
