// api.cu - the extern "C" boundary of libvmat (include/vmat.h): argument checks, handle lifetime,
// and the sequencing of the kernels on the caller's stream.  No arithmetic lives here.
#include "spmv.cuh"
#include <stdarg.h>
#include <string.h>
#include <math.h>
#include <stdlib.h>
#include <new>
#include <vector>
#include <algorithm>
#include <utility>

static thread_local char g_err[512] = "";
thread_local int g_vmat_launches = 0;

void vmat_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

#define REQUIRE(cond, msg)                                            \
    do {                                                              \
        if (!(cond)) { vmat_set_error("%s: %s", __func__, msg); return VMAT_ERR_INVALID_ARG; } \
    } while (0)
#define TRY(x) do { int rc_ = (x); if (rc_ != VMAT_OK) return rc_; } while (0)

template <typename T>
static int upload(T **dst, const T *src, int64_t n, int64_t *bytes)
{
    const size_t b = (size_t)(n > 0 ? n : 1) * sizeof(T);
    VMAT_CUDA(cudaMalloc((void **)dst, b));
    *bytes += (int64_t)b;
    if (n > 0) VMAT_CUDA(cudaMemcpy(*dst, src, (size_t)n * sizeof(T), cudaMemcpyHostToDevice));
    return VMAT_OK;
}

// PDL-free, graph-free sequencing: plain launches on the caller's stream.
__global__ void k_aperture_indicator(int n_beamlets, float *__restrict__ x, int row0, int row1,
                                     const int32_t *__restrict__ leafrow_col_offset,
                                     const int32_t *__restrict__ L, const int32_t *__restrict__ R)
{
    // x = indicator of the aperture (Eq. (5): the beamlets within the chosen openings)
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_beamlets) return;
    float v = 0.f;
    if (j >= leafrow_col_offset[row0] && j < leafrow_col_offset[row1]) {
        int lo = row0, hi = row1;                       // leaf row of beamlet j: last row with offset <= j
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (leafrow_col_offset[mid] <= j) lo = mid; else hi = mid;
        }
        const int c = j - leafrow_col_offset[lo];
        v = (c >= L[lo] && c < R[lo]) ? 1.f : 0.f;
    }
    x[j] = v;
}

// ---- Eq. (5) by scatter: DA = sum of the columns of D inside the aperture, read from the beamlet rows of D^T.
// One warp per beamlet of the control point; beamlets outside their row's opening leave at once.  Several
// beamlets reach the same voxel, so the sums go through 64-bit FIXED-POINT atomics: integer addition is exact and
// order-free, hence the result is deterministic and is the correctly rounded sum up to the fixed-point quantum
// 2^-shift (shift chosen at create from max |D_ij| and the beamlets per control point so that no sum overflows:
// quantum < 1e-15 for these matrices).  Touches nnz/n_angles entries instead of streaming all of D (2.7 ms ->
// < 0.1 ms on config 3).
__global__ void k_absmax(const float *__restrict__ val, int64_t n, unsigned *__restrict__ out)
{
    unsigned m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        m = max(m, __float_as_uint(fabsf(val[i])));          // |finite floats| order like their bit patterns
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

template <int FMT>
__global__ void __launch_bounds__(256)
k_aperture_scatter(const int64_t *__restrict__ pptr, MatView A, int j_lo, int j_hi,
                   const int32_t *__restrict__ beamlet_leafrow, const int32_t *__restrict__ leafrow_col_offset,
                   const int32_t *__restrict__ L, const int32_t *__restrict__ R, double scale,
                   unsigned long long *__restrict__ acc)
{
    const int lane = threadIdx.x & 31;
    const int j = j_lo + blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (j >= j_hi) return;
    const int r = beamlet_leafrow[j], c = j - leafrow_col_offset[r];
    if (c < L[r] || c >= R[r]) return;                        // the beamlet is under a leaf
    const int64_t s = pptr[j], e = pptr[j + 1];
    const int nt = (int)((e - s) >> 8);
    auto add = [&](float v, int vox) {
        VMAT_ASSERT_INDEX(A, vox);
        if (v != 0.f) atomicAdd(acc + vox, (unsigned long long)__double2ll_rn((double)v * scale));
    };
    TileCursor<FMT> tc(A, s, lane);
    for (int ti = 0; ti < nt; ++ti, tc.advance()) {
        TileRegs<FMT> t;
        tile_load<FMT>(A, tc, lane, t);
        int vx[8];
        tile_indices<FMT>(A, tc, t, lane, vx);
#pragma unroll
        for (int q = 0; q < 8; ++q) add(__uint_as_float(t.v.w[q]), vx[q]);
    }
    for (int64_t kg = s + (int64_t)nt * TILE; kg < e; kg += GROUP) {
        float v;
        int vox;
        group_entry<FMT>(A, kg, lane, v, vox);
        add(v, vox);
    }
}

__global__ void k_aperture_finish(int n_voxels, const unsigned long long *__restrict__ acc, double inv_scale,
                                  float *__restrict__ DA)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_voxels) DA[i] = (float)((double)(long long)acc[i] * inv_scale);
}

__global__ void k_max_u8(const uint8_t *__restrict__ v, int n, unsigned *__restrict__ out)
{
    unsigned m = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) m = max(m, (unsigned)v[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// n device buffers, committed to their owners only when every one of them could be allocated: after a failure the
// owners are as before (NULL), nothing leaks and *bytes is untouched, so the caller may simply try again later.
static int alloc_all_or_none(void **const *dst, const size_t *bytes_each, int n, int64_t *bytes)
{
    void *tmp[8] = {nullptr};
    size_t total = 0;
    for (int i = 0; i < n; ++i) {
        const cudaError_t e = cudaMalloc(&tmp[i], bytes_each[i]);
        if (e != cudaSuccess) {
            for (int k = 0; k < i; ++k) cudaFree(tmp[k]);
            vmat_set_error("device allocation of %zu bytes failed: %s", bytes_each[i], cudaGetErrorString(e));
            cudaGetLastError();
            return e == cudaErrorMemoryAllocation ? VMAT_ERR_OOM : VMAT_ERR_CUDA;
        }
        total += bytes_each[i];
    }
    for (int i = 0; i < n; ++i) *dst[i] = tmp[i];
    *bytes += (int64_t)total;
    return VMAT_OK;
}
// d, g and p of the end-to-end host calls (shared by the synchronous and the two-slot variant)
static int e2e_alloc_vectors(vmat_ddc *h)
{
    if (h->e2e_d) return VMAT_OK;
    const size_t nv = h->n_voxels > 0 ? h->n_voxels : 1, nb = h->n_beamlets > 0 ? h->n_beamlets : 1;
    void **const dst[] = {(void **)&h->e2e_d, (void **)&h->e2e_g, (void **)&h->e2e_p};
    const size_t sz[] = {nv * 4, nv * 4, nb * 4};
    return alloc_all_or_none(dst, sz, 3, &h->bytes_device);
}

extern "C" {

const char *vmat_last_error(void) { return g_err; }

int vmat_check_structure_ids(const uint8_t *voxel_struct, int32_t n_voxels, int32_t n_struct, void *stream)
{
    REQUIRE(n_struct >= 1 && n_struct <= 256, "n_struct must be in 1..256");
    REQUIRE(n_voxels >= 0 && (voxel_struct || n_voxels == 0), "NULL argument");
    if (n_voxels == 0) return VMAT_OK;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned *d_max = nullptr, h_max = 0;
    VMAT_CUDA(cudaMalloc((void **)&d_max, 4));
    cudaError_t e = cudaMemsetAsync(d_max, 0, 4, st);
    if (e == cudaSuccess) {
        k_max_u8<<<256, 256, 0, st>>>(voxel_struct, n_voxels, d_max);
        e = cudaMemcpyAsync(&h_max, d_max, 4, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_max);
    VMAT_CUDA(e);
    if ((int)h_max >= n_struct) {
        vmat_set_error("vmat_check_structure_ids: structure id %u >= n_struct %d", h_max, n_struct);
        return VMAT_ERR_INDEX_RANGE;
    }
    return VMAT_OK;
}
int vmat_last_launch_count(void) { return g_vmat_launches; }

int vmat_ddc_destroy(vmat_ddc *h)
{
    if (!h) return VMAT_OK;
    void *ptrs[] = {h->D.ptr, h->D.pptr, h->D.val, h->D.sec, h->D.base, h->Dt.ptr, h->Dt.pptr, h->Dt.val, h->Dt.sec,
                    h->Dt.base, h->angle_col_offset,
                    h->angle_row_offset, h->leafrow_col_offset, h->leafrow_angle, h->seg_row, h->F_partial,
                    h->F_partial_obj, h->S_scratch, h->beamlet_leafrow, h->leafrow_done, h->e2e_x, h->e2e_d, h->e2e_g, h->e2e_p, h->e2e_L, h->e2e_R,
                    h->e2e_best, h->e2e_row_price, h->e2e_angle_price, h->e2e_F,
                    h->leafrow_pos0, h->angle_pmin, h->angle_wd, h->row_bp_offset, h->cs_bp, h->ad_acc, h->angle_order,
                    h->col_perm, h->x_perm, h->q_start, h->q_next};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    for (auto &sl : h->slot) {
        for (void *p : {(void *)sl.x, (void *)sl.L, (void *)sl.R, (void *)sl.best, (void *)sl.row_price, (void *)sl.angle_price, (void *)sl.F})
            if (p) cudaFree(p);
        for (cudaEvent_t e : {sl.x_ready, sl.done, sl.out_ready})
            if (e) cudaEventDestroy(e);
    }
    if (h->e2e_in) cudaStreamDestroy(h->e2e_in);
    if (h->e2e_out) cudaStreamDestroy(h->e2e_out);
    if (h->cs_fork) cudaEventDestroy(h->cs_fork);
    if (h->cs_join) cudaEventDestroy(h->cs_join);
    if (h->cs_aux) cudaStreamDestroy(h->cs_aux);
    delete h;
    return VMAT_OK;
}

// Queue q of a kernel (smqueue.cuh) starts at the first item whose first stored entry lies at or beyond q / nq of the
// layout's padded entries.  seg_row != NULL: item = `per` consecutive segments of the dose kernel; NULL: `per` rows.
__global__ void k_queue_starts(int nq, int n_items, int per, int n_units, const int32_t *__restrict__ seg_row,
                               const int64_t *__restrict__ pptr, int64_t P, int32_t *__restrict__ start)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q > nq) return;
    const int64_t target = q == nq ? P : (P / nq) * q;
    int lo = 0, hi = n_items;                                      // smallest item with pos(item) >= target
    if (q == nq) lo = n_items;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const int u = min(mid * per, n_units);
        const int64_t pos = pptr[seg_row ? seg_row[u] : u];
        if (pos >= target) hi = mid; else lo = mid + 1;
    }
    start[q] = lo;
}

static int build_sm_queues(vmat_ddc *h, cudaStream_t st)
{
    int n_sm = 0;
    VMAT_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, h->device));
    h->n_sm = n_sm;
    if (n_sm <= 0) return VMAT_OK;
    const size_t n = 2 * ((size_t)n_sm + 1);
    VMAT_CUDA(cudaMalloc((void **)&h->q_start, n * 4));
    VMAT_CUDA(cudaMalloc((void **)&h->q_next, n * 4));
    h->bytes_device += (int64_t)n * 8;
    VMAT_CUDA(cudaMemsetAsync(h->q_next, 0, n * 4, st));
    const int tb = 64, gb = (n_sm + 1 + tb - 1) / tb;
    k_queue_starts<<<gb, tb, 0, st>>>(n_sm, h->n_blocks, DOSE_THREADS / 32, h->n_seg, h->seg_row, h->D.pptr, h->D.P, h->q_start);
    VMAT_LAUNCH_CHECK();
    k_queue_starts<<<gb, tb, 0, st>>>(n_sm, (h->n_beamlets + PRICE_WARPS - 1) / PRICE_WARPS, PRICE_WARPS, h->n_beamlets,
                                      nullptr, h->Dt.pptr, h->Dt.P, h->q_start + n_sm + 1);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}
// The automatic choice, per kernel.  Measured on B200 (profiles/r2_sm_affine.md): the queues pay where a kernel runs
// many items per resident CTA and an item is long (config 3: 76 KB per dose item, 188 KB per price item, ~100 items
// per CTA: +2.3 % per evaluation, more under the power cap).  With short items the visit to the queue (two block
// barriers and an atomic's round trip to L2) costs more than a fresh CTA from the hardware scheduler (dose items of
// 23 - 55 KB, configs 1 and 2 and the config-4 sweep: -4 %), and with a handful of items per CTA (price kernel of
// configs 1 and 2: 7 and 3) there is nothing to share and the tail is coarser.
static bool sm_affine_pays(int64_t stored_bytes, int64_t n_items, int n_sm, int ctas_per_sm, int64_t min_item_bytes)
{
    if (n_items <= 0 || n_sm <= 0) return false;
    return n_items >= (int64_t)16 * n_sm * ctas_per_sm && stored_bytes / n_items >= min_item_bytes;
}

int vmat_ddc_set_schedule(vmat_ddc *h, int32_t sm_affine)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(sm_affine >= -1 && sm_affine <= 1, "sm_affine must be -1 (automatic), 0 or 1");
    if (sm_affine < 0) {
        h->sched_dose = sm_affine_pays(h->D.bytes(), h->n_blocks, h->n_sm, VMAT_DOSE_MINB, 64 * 1024);
        h->sched_price = sm_affine_pays(h->Dt.bytes(), (h->n_beamlets + PRICE_WARPS - 1) / PRICE_WARPS, h->n_sm, 6, 64 * 1024);
    } else {
        h->sched_dose = h->sched_price = sm_affine;
    }
    // The queue counters reset themselves at the end of every launch that runs to completion (smqueue.cuh).  A launch
    // that was cut short, or two launches that overlapped on this handle against the rule above, leave them non-zero,
    // and every later persistent launch would then find its queues "empty" and write nothing.  No launch is in flight
    // here by contract, so this is the place to put them back to zero.
    if (h->q_next != nullptr) {
        VMAT_CUDA(cudaMemsetAsync(h->q_next, 0, 2 * ((size_t)h->n_sm + 1) * 4, (cudaStream_t)0));
        VMAT_CUDA(cudaStreamSynchronize((cudaStream_t)0));
    }
    return VMAT_OK;
}

int vmat_ddc_create(vmat_ddc **out, int32_t n_voxels, int32_t n_beamlets, int64_t nnz,
                    const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                    int32_t n_angles, const int32_t *angle_col_offset, const int32_t *angle_row_offset,
                    const int32_t *leafrow_col_offset, void *stream)
{
    return vmat_ddc_create_ex(out, n_voxels, n_beamlets, nnz, coo_voxel, coo_beamlet, coo_val, n_angles,
                              angle_col_offset, angle_row_offset, leafrow_col_offset, 0, stream);
}

int vmat_ddc_create_ex(vmat_ddc **out, int32_t n_voxels, int32_t n_beamlets, int64_t nnz,
                       const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                       int32_t n_angles, const int32_t *angle_col_offset, const int32_t *angle_row_offset,
                       const int32_t *leafrow_col_offset, int32_t index_bits, void *stream)
{
    REQUIRE(out != nullptr, "out is NULL");
    REQUIRE(index_bits == 0 || index_bits == 16 || index_bits == 32, "index_bits must be 0 (auto), 16 or 32");
    REQUIRE(n_voxels >= 0 && n_beamlets >= 0 && nnz >= 0 && n_angles >= 0, "negative size");
    REQUIRE(nnz == 0 || (coo_voxel && coo_beamlet && coo_val), "COO pointer is NULL");
    REQUIRE(nnz == 0 || (n_voxels > 0 && n_beamlets > 0), "nnz > 0 with an empty dimension");
    REQUIRE(angle_col_offset && angle_row_offset && leafrow_col_offset, "offset table is NULL");
    REQUIRE(angle_col_offset[0] == 0 && angle_row_offset[0] == 0 && leafrow_col_offset[0] == 0,
            "offset tables must start at 0");
    for (int a = 0; a < n_angles; ++a) {
        REQUIRE(angle_col_offset[a + 1] >= angle_col_offset[a], "angle_col_offset not monotone");
        REQUIRE(angle_row_offset[a + 1] >= angle_row_offset[a], "angle_row_offset not monotone");
    }
    REQUIRE(angle_col_offset[n_angles] == n_beamlets, "angle_col_offset must end at n_beamlets");
    const int32_t n_rows = angle_row_offset[n_angles];
    int32_t max_len = 0;
    for (int r = 0; r < n_rows; ++r) {
        REQUIRE(leafrow_col_offset[r + 1] >= leafrow_col_offset[r], "leafrow_col_offset not monotone");
        max_len = leafrow_col_offset[r + 1] - leafrow_col_offset[r] > max_len
                      ? leafrow_col_offset[r + 1] - leafrow_col_offset[r] : max_len;
    }
    REQUIRE(leafrow_col_offset[n_rows] == n_beamlets, "leafrow_col_offset must end at n_beamlets");
    std::vector<int32_t> row_angle((size_t)(n_rows > 0 ? n_rows : 1), 0);
    for (int a = 0; a < n_angles; ++a) {                 // leaf rows must not straddle control points
        REQUIRE(leafrow_col_offset[angle_row_offset[a]] == angle_col_offset[a],
                "leaf rows straddle a control point boundary");
        for (int r = angle_row_offset[a]; r < angle_row_offset[a + 1]; ++r) row_angle[r] = a;
    }

    vmat_ddc *h = new (std::nothrow) vmat_ddc();
    if (!h) { vmat_set_error("vmat_ddc_create: host allocation failed"); return VMAT_ERR_OOM; }
    h->n_voxels = n_voxels; h->n_beamlets = n_beamlets; h->nnz = nnz;
    h->n_angles = n_angles; h->n_leaf_rows = n_rows; h->max_leaf_row_len = max_len;
    cudaGetDevice(&h->device);
    h->h_angle_row_offset.assign(angle_row_offset, angle_row_offset + n_angles + 1);
    h->h_angle_col_offset.assign(angle_col_offset, angle_col_offset + n_angles + 1);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = VMAT_OK;
    {   // column order of CSR(D): per control point, tiles of COL_TILE columns x all leaf rows (common.cuh)
#ifndef VMAT_COL_TILE
#define VMAT_COL_TILE 8
#endif
        constexpr int COL_TILE = VMAT_COL_TILE;               // 8 floats = one 32-byte sector of x
        std::vector<int32_t> perm((size_t)(n_beamlets > 0 ? n_beamlets : 1), 0);
        bool identity = true;
        for (int a = 0; a < n_angles; ++a) {
            const int ra = angle_row_offset[a], rb = angle_row_offset[a + 1];
            int32_t nxt = angle_col_offset[a], longest = 0;
            for (int r = ra; r < rb; ++r)
                longest = std::max(longest, leafrow_col_offset[r + 1] - leafrow_col_offset[r]);
            for (int c0 = 0; c0 < longest; c0 += COL_TILE)
                for (int r = ra; r < rb; ++r) {
                    const int j0 = leafrow_col_offset[r], n = leafrow_col_offset[r + 1] - j0;
                    for (int c = c0; c < std::min(c0 + COL_TILE, n); ++c) {
                        identity = identity && nxt == j0 + c;
                        perm[j0 + c] = nxt++;
                    }
                }
        }
        // worth a pass over x per dose launch only where leaf rows are several tiles long (max_len = the longest)
        if (!identity && n_beamlets > 0 && max_len >= 4 * COL_TILE) {
            h->h_col_inv.assign((size_t)n_beamlets, 0);
            for (int j = 0; j < n_beamlets; ++j) h->h_col_inv[perm[j]] = j;
            rc = upload(&h->col_perm, perm.data(), (int64_t)n_beamlets, &h->bytes_device);
            if (rc == VMAT_OK) {
                cudaError_t e = cudaMalloc((void **)&h->x_perm, (size_t)n_beamlets * 4);
                if (e != cudaSuccess) { vmat_set_error("vmat_ddc_create: cudaMalloc(x_perm) failed"); rc = VMAT_ERR_OOM; }
                h->bytes_device += (int64_t)n_beamlets * 4;
            }
        }
    }
    if (rc == VMAT_OK) rc = vmat_build_layouts(h, coo_voxel, coo_beamlet, coo_val, index_bits, st);
    h->D.n_sec = n_beamlets;
    h->Dt.n_sec = n_voxels;
    if (rc == VMAT_OK) rc = build_sm_queues(h, st);
    if (rc == VMAT_OK) rc = vmat_ddc_set_schedule(h, -1);
    if (rc == VMAT_OK) rc = upload(&h->angle_col_offset, angle_col_offset, (int64_t)n_angles + 1, &h->bytes_device);
    if (rc == VMAT_OK) rc = upload(&h->angle_row_offset, angle_row_offset, (int64_t)n_angles + 1, &h->bytes_device);
    if (rc == VMAT_OK) rc = upload(&h->leafrow_col_offset, leafrow_col_offset, (int64_t)n_rows + 1, &h->bytes_device);
    if (rc == VMAT_OK) rc = upload(&h->leafrow_angle, row_angle.data(), (int64_t)n_rows, &h->bytes_device);
    if (rc == VMAT_OK) {
        const size_t b = ((size_t)n_beamlets + (size_t)n_rows + 1) * sizeof(double);
        cudaError_t e = cudaMalloc((void **)&h->S_scratch, b);
        if (e != cudaSuccess) { vmat_set_error("vmat_ddc_create: cudaMalloc(S_scratch) failed"); rc = VMAT_ERR_OOM; }
        h->bytes_device += (int64_t)b;
    }
    if (rc == VMAT_OK) {
        std::vector<int32_t> bl((size_t)(n_beamlets > 0 ? n_beamlets : 1), 0);
        for (int r = 0; r < n_rows; ++r)
            for (int j = leafrow_col_offset[r]; j < leafrow_col_offset[r + 1]; ++j) bl[j] = r;
        rc = upload(&h->beamlet_leafrow, bl.data(), (int64_t)n_beamlets, &h->bytes_device);
    }
    if (rc == VMAT_OK) {
        const size_t b = (size_t)(n_rows + 1) * sizeof(uint32_t);          // + 1: the aperture-price ticket
        cudaError_t e = cudaMalloc((void **)&h->leafrow_done, b);
        h->angle_ticket = h->leafrow_done + n_rows;
        if (e != cudaSuccess) { vmat_set_error("vmat_ddc_create: cudaMalloc(leafrow_done) failed"); rc = VMAT_ERR_OOM; }
        else cudaMemsetAsync(h->leafrow_done, 0, b, st);
        h->bytes_device += (int64_t)b;
    }
    unsigned absmax_bits = 0;
    if (rc == VMAT_OK) {                                      // scale of vmat_aperture_dose's fixed-point sums
        const size_t b = (size_t)(n_voxels > 0 ? n_voxels : 1) * 8;
        cudaError_t e = cudaMalloc((void **)&h->ad_acc, b);
        if (e != cudaSuccess) { vmat_set_error("vmat_ddc_create: cudaMalloc(ad_acc) failed"); rc = VMAT_ERR_OOM; }
        else {
            h->bytes_device += (int64_t)b;
            unsigned *d_max = (unsigned *)h->ad_acc;          // borrowed for the reduction
            cudaMemsetAsync(d_max, 0, 4, st);
            if (h->Dt.P > 0) k_absmax<<<1024, 256, 0, st>>>(h->Dt.val, h->Dt.P, d_max);
            cudaMemcpyAsync(&absmax_bits, d_max, 4, cudaMemcpyDeviceToHost, st);
        }
    }
    if (rc == VMAT_OK) {
        cudaError_t e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { vmat_set_error("vmat_ddc_create: %s", cudaGetErrorString(e)); rc = VMAT_ERR_CUDA; }
    }
    if (rc != VMAT_OK) { vmat_ddc_destroy(h); cudaGetLastError(); return rc; }
    {
        float mx;
        memcpy(&mx, &absmax_bits, 4);
        int E = 0, nb_max = 1;
        if (mx > 0.f) frexpf(mx, &E);                         // mx < 2^E
        for (int a = 0; a < n_angles; ++a)
            nb_max = angle_col_offset[a + 1] - angle_col_offset[a] > nb_max ? angle_col_offset[a + 1] - angle_col_offset[a] : nb_max;
        int bits = 1;
        while ((1 << bits) <= nb_max) ++bits;                 // a voxel sums < 2^bits beamlets of one control point
        h->ad_shift = 62 - bits - E;                          // |sum| * 2^shift < 2^62
    }
    *out = h;
    return VMAT_OK;
}

int vmat_ddc_info_get(const vmat_ddc *h, vmat_ddc_info *info)
{
    REQUIRE(h && info, "NULL argument");
    info->n_voxels = h->n_voxels; info->n_beamlets = h->n_beamlets; info->nnz = h->nnz;
    info->n_angles = h->n_angles; info->n_leaf_rows = h->n_leaf_rows;
    info->bytes_csr_d = 8 * h->nnz + 8 * ((int64_t)h->n_voxels + 1);
    info->bytes_csr_dt = 8 * h->nnz + 8 * ((int64_t)h->n_beamlets + 1);
    info->bytes_device_total = h->bytes_device;
    info->n_dose_blocks = h->n_seg;
    info->max_leaf_row_len = h->max_leaf_row_len;
    info->max_voxel_row_nnz = h->max_voxel_row_nnz;
    info->max_beamlet_row_nnz = h->max_beamlet_row_nnz;
    info->index_bits_d = h->D.index_bits; info->index_bits_dt = h->Dt.index_bits;
    info->padded_d = h->D.P; info->padded_dt = h->Dt.P;
    info->bytes_stream_d = h->D.bytes() + 4 * ((int64_t)h->n_seg + 1);      // + the segment table
    info->bytes_stream_dt = h->Dt.bytes();
    info->tiles_d = h->D.n_tiles; info->tiles_uniform_d = h->D.n_tiles_uniform;
    info->tiles_dt = h->Dt.n_tiles; info->tiles_uniform_dt = h->Dt.n_tiles_uniform;
    info->grid_dose = h->n_blocks > 0 ? vmat_dose_grid(h, true) : 0;
    info->grid_price = h->n_beamlets > 0 ? vmat_price_grid(h) : 0;
    info->sm_affine_dose = h->queues_dose().nq > 0; info->sm_affine_price = h->queues_price().nq > 0;
    return VMAT_OK;
}

int vmat_ddc_export_csr(const vmat_ddc *h, int which, int64_t *ptr, int32_t *idx, float *val)
{
    REQUIRE(h && ptr && ((idx == nullptr) == (val == nullptr)), "NULL argument");
    REQUIRE(which == 0 || which == 1, "which must be 0 (D) or 1 (D^T)");
    const PackedLayout &A = which == 0 ? h->D : h->Dt;
    VMAT_CUDA(cudaDeviceSynchronize());
    VMAT_CUDA(cudaMemcpy(ptr, A.ptr, ((size_t)A.n_rows + 1) * 8, cudaMemcpyDeviceToHost));
    if (idx == nullptr || h->nnz == 0) return VMAT_OK;       // row pointers only
    // Unpack the grouped layout (spmv.cuh) on the host: undo the tile interleave, add the group bases,
    // drop the pads.  Within a row the real entries ascend strictly and a pad repeats the index before it.
    const bool narrow = A.index_bits == 16;
    std::vector<int64_t> pp((size_t)A.n_rows + 1);
    std::vector<float> pv((size_t)A.P);
    std::vector<int32_t> pi32(narrow ? 0 : (size_t)A.P), pbase(narrow ? (size_t)(A.P / GROUP) : 0);
    std::vector<uint16_t> pi16(narrow ? (size_t)A.P : 0);
    VMAT_CUDA(cudaMemcpy(pp.data(), A.pptr, pp.size() * 8, cudaMemcpyDeviceToHost));
    VMAT_CUDA(cudaMemcpy(pv.data(), A.val, pv.size() * 4, cudaMemcpyDeviceToHost));
    if (narrow) {
        VMAT_CUDA(cudaMemcpy(pi16.data(), A.sec, pi16.size() * 2, cudaMemcpyDeviceToHost));
        VMAT_CUDA(cudaMemcpy(pbase.data(), A.base, pbase.size() * 4, cudaMemcpyDeviceToHost));
    } else {
        VMAT_CUDA(cudaMemcpy(pi32.data(), A.sec, pi32.size() * 4, cudaMemcpyDeviceToHost));
    }
    const int64_t n_seg = which == 0 ? (int64_t)h->n_seg : (int64_t)A.n_rows;
    for (int64_t w = 0; w < n_seg; ++w) {
        const int32_t r0 = which == 0 ? h->h_seg_row[w] : (int32_t)w;
        const int32_t r1 = which == 0 ? h->h_seg_row[w + 1] : (int32_t)w + 1;
        const int64_t S = pp[r0], G = (pp[r1] - S) / GROUP;
        for (int32_t r = r0; r < r1; ++r) {
            int64_t o = ptr[r];
            int32_t prev = -1;
            for (int64_t q = pp[r]; q < pp[r + 1]; ++q) {
                const int64_t sp = stored_pos(S, G, q);
                const int32_t c = narrow ? base_index(pbase[q >> 5]) + (int32_t)pi16[sp] : pi32[sp];
                if (c <= prev) continue;                              // a pad
                if (o >= ptr[r + 1]) { vmat_set_error("vmat_ddc_export_csr: layout inconsistent (row %d)", r); return VMAT_ERR_CUDA; }
                idx[o] = c; val[o] = pv[sp]; prev = c; ++o;
            }
            if (o != ptr[r + 1]) { vmat_set_error("vmat_ddc_export_csr: layout inconsistent (row %d)", r); return VMAT_ERR_CUDA; }
            if (which == 0 && !h->h_col_inv.empty()) {                // back to the caller's beamlet numbers, ascending
                const int64_t a = ptr[r], n = ptr[r + 1] - a;
                std::vector<std::pair<int32_t, float>> row((size_t)n);
                for (int64_t i = 0; i < n; ++i) row[(size_t)i] = {h->h_col_inv[idx[a + i]], val[a + i]};
                std::sort(row.begin(), row.end(), [](const std::pair<int32_t, float> &x, const std::pair<int32_t, float> &y) { return x.first < y.first; });
                for (int64_t i = 0; i < n; ++i) { idx[a + i] = row[(size_t)i].first; val[a + i] = row[(size_t)i].second; }
            }
        }
    }
    return VMAT_OK;
}

int vmat_dose(const vmat_ddc *h, const float *x, float *d, void *stream)
{
    REQUIRE(h && (x || h->n_beamlets == 0) && (d || h->n_voxels == 0), "NULL argument");
    g_vmat_launches = 0;
    return vmat_launch_dose(h, x, d, false, nullptr, 0, nullptr, nullptr, nullptr, nullptr, nullptr,
                            (cudaStream_t)stream);
}

int vmat_objective_grad(const vmat_ddc *h, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                        const float *T, const float *w_over, const float *w_under,
                        float *g, double *F, void *stream)
{
    REQUIRE(h && F && T && w_over && w_under, "NULL argument");
    REQUIRE(h->n_voxels == 0 || (d && voxel_struct && g), "NULL argument");
    REQUIRE(n_struct >= 1 && n_struct <= 256, "n_struct must be in 1..256");
    g_vmat_launches = 0;
    return vmat_launch_objective(h, d, voxel_struct, n_struct, T, w_over, w_under, g, F, (cudaStream_t)stream);
}

int vmat_price(const vmat_ddc *h, const float *g, float *p, void *stream)
{
    REQUIRE(h && (g || h->n_voxels == 0) && (p || h->n_beamlets == 0), "NULL argument");
    g_vmat_launches = 0;
    return vmat_launch_price(h, g, p, (cudaStream_t)stream);
}

int vmat_select_apertures(const vmat_ddc *h, const float *p, const uint8_t *angle_mask,
                          int32_t *L, int32_t *R, double *row_price, double *angle_price,
                          int32_t *best_angle, void *stream)
{
    REQUIRE(h && best_angle, "NULL argument");
    REQUIRE(h->n_beamlets == 0 || p, "p is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L && R && row_price), "NULL output");
    REQUIRE(h->n_angles == 0 || angle_price, "angle_price is NULL");
    g_vmat_launches = 0;
    TRY(vmat_launch_select(h, p, angle_mask, L, R, row_price, (cudaStream_t)stream));
    return vmat_launch_angle_price(h, row_price, angle_mask, angle_price, best_angle, (cudaStream_t)stream);
}

int vmat_price_eval(const vmat_ddc *h, const float *x,
                    const uint8_t *voxel_struct, int32_t n_struct,
                    const float *T, const float *w_over, const float *w_under,
                    const uint8_t *angle_mask,
                    float *d, float *g, double *F, float *p,
                    int32_t *L, int32_t *R, double *row_price, double *angle_price,
                    int32_t *best_angle, void *stream)
{
    REQUIRE(h && F && best_angle && T && w_over && w_under, "NULL argument");
    REQUIRE(h->n_voxels == 0 || (d && g && voxel_struct), "NULL voxel vector");
    REQUIRE(h->n_beamlets == 0 || (x && p), "NULL beamlet vector");
    REQUIRE(h->n_leaf_rows == 0 || (L && R && row_price), "NULL leaf-row output");
    REQUIRE(h->n_angles == 0 || angle_price, "angle_price is NULL");
    REQUIRE(n_struct >= 1 && n_struct <= 256, "n_struct must be in 1..256");
    cudaStream_t st = (cudaStream_t)stream;
    g_vmat_launches = 0;
    TRY(vmat_launch_dose(h, x, d, true, voxel_struct, n_struct, T, w_over, w_under, g, F, st));
    if (h->prof_ev[2]) VMAT_CUDA(cudaEventRecord(h->prof_ev[2], st));
    TRY(vmat_launch_price_select(h, g, angle_mask, p, L, R, row_price, st));
    if (h->prof_ev[3]) VMAT_CUDA(cudaEventRecord(h->prof_ev[3], st));
    return vmat_launch_angle_price(h, row_price, angle_mask, angle_price, best_angle, st);
}

int vmat_price_select(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p, int32_t *L, int32_t *R,
                      double *row_price, double *angle_price, int32_t *best_angle, void *stream)
{
    REQUIRE(h && best_angle, "NULL argument");
    REQUIRE(h->n_voxels == 0 || g, "g is NULL");
    REQUIRE(h->n_beamlets == 0 || p, "p is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L && R && row_price), "NULL leaf-row output");
    REQUIRE(h->n_angles == 0 || angle_price, "angle_price is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    g_vmat_launches = 0;
    TRY(vmat_launch_price_select(h, g, angle_mask, p, L, R, row_price, st));
    return vmat_launch_angle_price(h, row_price, angle_mask, angle_price, best_angle, st);
}

int vmat_best_pair(const vmat_ddc *h, const double *angle_price, const int32_t *best_angle, int32_t angle_lo,
                   double *pair, void *stream)
{
    REQUIRE(h && best_angle && pair, "NULL argument");
    REQUIRE(h->n_angles == 0 || angle_price, "angle_price is NULL");
    g_vmat_launches = 0;
    return vmat_launch_best_pair(h, angle_price, best_angle, angle_lo, pair, (cudaStream_t)stream);
}

int vmat_merge_best(const double *pairs, int32_t n, double *best, void *stream)
{
    REQUIRE(n >= 0 && (pairs || n == 0) && best, "NULL argument");
    g_vmat_launches = 0;
    return vmat_launch_merge_best(pairs, n, best, (cudaStream_t)stream);
}

int vmat_ddc_set_profile_events(vmat_ddc *h, void *const *ev)
{
    REQUIRE(h != nullptr, "handle is NULL");
    for (int i = 0; i < 4; ++i) h->prof_ev[i] = ev ? (cudaEvent_t)ev[i] : nullptr;
    return VMAT_OK;
}

int vmat_price_eval_host(vmat_ddc *h, const float *x_host,
                         const uint8_t *voxel_struct, int32_t n_struct,
                         const float *T, const float *w_over, const float *w_under,
                         const uint8_t *angle_mask,
                         double *F_host, int32_t *L_host, int32_t *R_host, double *row_price_host,
                         double *angle_price_host, int32_t *best_angle_host, void *stream)
{
    REQUIRE(h && F_host && best_angle_host, "NULL argument");
    REQUIRE(h->n_beamlets == 0 || x_host, "x_host is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L_host && R_host && row_price_host), "NULL leaf-row output");
    REQUIRE(h->n_angles == 0 || angle_price_host, "angle_price_host is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (!h->e2e_sync_ready) {                             // device scratch, allocated once: all of it or none of it
        const size_t nb = h->n_beamlets > 0 ? h->n_beamlets : 1;
        const size_t nr = h->n_leaf_rows > 0 ? h->n_leaf_rows : 1, na = h->n_angles > 0 ? h->n_angles : 1;
        TRY(e2e_alloc_vectors(h));
        void **const dst[] = {(void **)&h->e2e_x, (void **)&h->e2e_L, (void **)&h->e2e_R, (void **)&h->e2e_row_price,
                              (void **)&h->e2e_angle_price, (void **)&h->e2e_best, (void **)&h->e2e_F};
        const size_t sz[] = {nb * 4, nr * 4, nr * 4, nr * 8, na * 8, 4, 8};
        TRY(alloc_all_or_none(dst, sz, 7, &h->bytes_device));
        h->e2e_sync_ready = true;
    }
    if (h->n_beamlets > 0)
        VMAT_CUDA(cudaMemcpyAsync(h->e2e_x, x_host, (size_t)h->n_beamlets * 4, cudaMemcpyHostToDevice, st));
    TRY(vmat_price_eval(h, h->e2e_x, voxel_struct, n_struct, T, w_over, w_under, angle_mask, h->e2e_d, h->e2e_g,
                        h->e2e_F, h->e2e_p, h->e2e_L, h->e2e_R, h->e2e_row_price, h->e2e_angle_price, h->e2e_best, st));
    if (h->n_leaf_rows > 0) {
        VMAT_CUDA(cudaMemcpyAsync(L_host, h->e2e_L, (size_t)h->n_leaf_rows * 4, cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(cudaMemcpyAsync(R_host, h->e2e_R, (size_t)h->n_leaf_rows * 4, cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(cudaMemcpyAsync(row_price_host, h->e2e_row_price, (size_t)h->n_leaf_rows * 8, cudaMemcpyDeviceToHost, st));
    }
    if (h->n_angles > 0)
        VMAT_CUDA(cudaMemcpyAsync(angle_price_host, h->e2e_angle_price, (size_t)h->n_angles * 8, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaMemcpyAsync(best_angle_host, h->e2e_best, 4, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaMemcpyAsync(F_host, h->e2e_F, 8, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaStreamSynchronize(st));
    return VMAT_OK;
}

int vmat_price_eval_host_submit(vmat_ddc *h, int32_t slot, const float *x_host,
                                const uint8_t *voxel_struct, int32_t n_struct,
                                const float *T, const float *w_over, const float *w_under,
                                const uint8_t *angle_mask,
                                double *F_host, int32_t *L_host, int32_t *R_host, double *row_price_host,
                                double *angle_price_host, int32_t *best_angle_host, void *stream)
{
    REQUIRE(h && F_host && best_angle_host, "NULL argument");
    REQUIRE(slot == 0 || slot == 1, "slot must be 0 or 1");
    REQUIRE(h->n_beamlets == 0 || x_host, "x_host is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L_host && R_host && row_price_host), "NULL leaf-row output");
    REQUIRE(h->n_angles == 0 || angle_price_host, "angle_price_host is NULL");
    REQUIRE(!h->slot[slot].in_flight, "the slot is still in flight: call vmat_price_eval_host_wait first");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = h->n_beamlets > 0 ? h->n_beamlets : 1;
    const size_t nr = h->n_leaf_rows > 0 ? h->n_leaf_rows : 1, na = h->n_angles > 0 ? h->n_angles : 1;
    if (!h->e2e_slots_ready) {                            // streams, events and device scratch, allocated once.  A
        // failure part-way leaves the flag down: the next call creates what is still missing (every step below skips
        // what exists) and never launches with a NULL stream, event or buffer.
        if (!h->e2e_in) VMAT_CUDA(cudaStreamCreateWithFlags(&h->e2e_in, cudaStreamNonBlocking));
        if (!h->e2e_out) VMAT_CUDA(cudaStreamCreateWithFlags(&h->e2e_out, cudaStreamNonBlocking));
        TRY(e2e_alloc_vectors(h));
        for (auto &s : h->slot) {
            if (!s.F) {
                void **const dst[] = {(void **)&s.x, (void **)&s.L, (void **)&s.R, (void **)&s.row_price,
                                      (void **)&s.angle_price, (void **)&s.best, (void **)&s.F};
                const size_t sz[] = {nb * 4, nr * 4, nr * 4, nr * 8, na * 8, 4, 8};
                TRY(alloc_all_or_none(dst, sz, 7, &h->bytes_device));
            }
            if (!s.x_ready) VMAT_CUDA(cudaEventCreateWithFlags(&s.x_ready, cudaEventDisableTiming));
            if (!s.done) VMAT_CUDA(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
            if (!s.out_ready) VMAT_CUDA(cudaEventCreateWithFlags(&s.out_ready, cudaEventDisableTiming));
        }
        h->e2e_slots_ready = true;
    }
    vmat_ddc::E2ESlot &s = h->slot[slot];
    // x of this slot was last read by the evaluation submitted two calls ago: its `done` event has long fired
    // (that slot was waited for), so the copy-in stream may overwrite it now
    if (h->n_beamlets > 0)
        VMAT_CUDA(cudaMemcpyAsync(s.x, x_host, (size_t)h->n_beamlets * 4, cudaMemcpyHostToDevice, h->e2e_in));
    VMAT_CUDA(cudaEventRecord(s.x_ready, h->e2e_in));
    VMAT_CUDA(cudaStreamWaitEvent(st, s.x_ready, 0));
    TRY(vmat_price_eval(h, s.x, voxel_struct, n_struct, T, w_over, w_under, angle_mask, h->e2e_d, h->e2e_g, s.F, h->e2e_p,
                        s.L, s.R, s.row_price, s.angle_price, s.best, st));
    VMAT_CUDA(cudaEventRecord(s.done, st));
    VMAT_CUDA(cudaStreamWaitEvent(h->e2e_out, s.done, 0));
    if (h->n_leaf_rows > 0) {
        VMAT_CUDA(cudaMemcpyAsync(L_host, s.L, (size_t)h->n_leaf_rows * 4, cudaMemcpyDeviceToHost, h->e2e_out));
        VMAT_CUDA(cudaMemcpyAsync(R_host, s.R, (size_t)h->n_leaf_rows * 4, cudaMemcpyDeviceToHost, h->e2e_out));
        VMAT_CUDA(cudaMemcpyAsync(row_price_host, s.row_price, (size_t)h->n_leaf_rows * 8, cudaMemcpyDeviceToHost, h->e2e_out));
    }
    if (h->n_angles > 0)
        VMAT_CUDA(cudaMemcpyAsync(angle_price_host, s.angle_price, (size_t)h->n_angles * 8, cudaMemcpyDeviceToHost, h->e2e_out));
    VMAT_CUDA(cudaMemcpyAsync(best_angle_host, s.best, 4, cudaMemcpyDeviceToHost, h->e2e_out));
    VMAT_CUDA(cudaMemcpyAsync(F_host, s.F, 8, cudaMemcpyDeviceToHost, h->e2e_out));
    VMAT_CUDA(cudaEventRecord(s.out_ready, h->e2e_out));
    s.in_flight = true;
    return VMAT_OK;
}

int vmat_price_eval_host_wait(vmat_ddc *h, int32_t slot)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(slot == 0 || slot == 1, "slot must be 0 or 1");
    if (!h->slot[slot].in_flight) return VMAT_OK;
    VMAT_CUDA(cudaEventSynchronize(h->slot[slot].out_ready));
    h->slot[slot].in_flight = false;
    return VMAT_OK;
}

int vmat_aperture_dose(const vmat_ddc *h, int32_t angle, const int32_t *L, const int32_t *R,
                       float *x_scratch, float *DA, void *stream)
{
    REQUIRE(h && L && R && x_scratch && DA, "NULL argument");
    REQUIRE(angle >= 0 && angle < h->n_angles, "angle out of range");
    cudaStream_t st = (cudaStream_t)stream;
    g_vmat_launches = 0;
    const int32_t aro[2] = {h->h_angle_row_offset[angle], h->h_angle_row_offset[angle + 1]};
    k_aperture_indicator<<<(h->n_beamlets + 255) / 256, 256, 0, st>>>(h->n_beamlets, x_scratch, aro[0], aro[1],
                                                                      h->leafrow_col_offset, L, R);
    VMAT_LAUNCH_CHECK();
    if (h->n_voxels == 0) return VMAT_OK;
    VMAT_CUDA(cudaMemsetAsync(h->ad_acc, 0, (size_t)h->n_voxels * 8, st));
    const int j_lo = h->h_angle_col_offset[angle], j_hi = h->h_angle_col_offset[angle + 1];
    const double scale = ldexp(1.0, h->ad_shift);
    if (j_hi > j_lo) {
        const int grid = (j_hi - j_lo + 7) / 8;
        const MatView A = view_of(h->Dt);
        switch (fmt_of(h->Dt)) {
        case 0: k_aperture_scatter<FMT_WIDE><<<grid, 256, 0, st>>>(h->Dt.pptr, A, j_lo, j_hi, h->beamlet_leafrow, h->leafrow_col_offset, L, R, scale, h->ad_acc); break;
        case 1: k_aperture_scatter<FMT_NARROW><<<grid, 256, 0, st>>>(h->Dt.pptr, A, j_lo, j_hi, h->beamlet_leafrow, h->leafrow_col_offset, L, R, scale, h->ad_acc); break;
        default: k_aperture_scatter<FMT_NARROW_1BASE><<<grid, 256, 0, st>>>(h->Dt.pptr, A, j_lo, j_hi, h->beamlet_leafrow, h->leafrow_col_offset, L, R, scale, h->ad_acc); break;
        }
        VMAT_LAUNCH_CHECK();
    }
    k_aperture_finish<<<(h->n_voxels + 255) / 256, 256, 0, st>>>(h->n_voxels, h->ad_acc, 1.0 / scale, DA);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

}  // extern "C"
