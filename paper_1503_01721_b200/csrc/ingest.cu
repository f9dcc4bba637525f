// ingest.cu - A0: COO triplets -> CSR(D) (voxel rows) + CSR(D^T) (beamlet rows) on the device.
// D is produced as COO (values, voxel index, beamlet index) and converted to CSR
// "at the initialization stage"; the paper keeps only D^T rows on the GPU, the B200 build keeps both
// so neither product needs atomics.
//
//   count      one pass over the triplets: range / finiteness checks, per-row histograms of both layouts
//   scan       exclusive scans -> int64 row pointers
//   scatter    second pass: each triplet takes the next free slot of its voxel row and of its beamlet row
//              (integer cursor atomics, warp-aggregated; the order inside a row is arbitrary here)
//   sort       every row is sorted by its secondary index with a bitonic network (shared memory for rows
//              up to 24 k entries, in place in global memory beyond) -> canonical order, so every later
//              floating-point sum has a fixed order whatever the order of the input triplets (C14);
//              equal neighbours after the sort are duplicates -> VMAT_ERR_DUPLICATE
// Host-resident COO is streamed through a device staging buffer in chunks, twice.
#include "spmv.cuh"
#include <vector>
#include <algorithm>

enum { FLAG_RANGE = 0, FLAG_NONFINITE = 1, FLAG_DUP = 2, N_FLAGS = 4 };

constexpr int ING_THREADS = 256;

// next free slot of row `key` for every lane, with one atomic per distinct key in the warp
__device__ __forceinline__ uint32_t warp_agg_take(uint32_t *cursor, int key, bool valid)
{
    const unsigned lane = threadIdx.x & 31;
    const unsigned m = __match_any_sync(0xffffffffu, valid ? key : -1 - (int)lane);
    const int leader = __ffs(m) - 1;
    uint32_t base = 0;
    if (valid && (int)lane == leader) base = atomicAdd(cursor + key, (uint32_t)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    return base + __popc(m & ((1u << lane) - 1u));
}

__global__ void __launch_bounds__(ING_THREADS)
k_count(const int32_t *__restrict__ vox, const int32_t *__restrict__ beam, const float *__restrict__ val,
        int64_t n, int32_t n_voxels, int32_t n_beamlets, uint32_t *cntV, uint32_t *cntB, int *flags)
{
    const int64_t stride = (int64_t)gridDim.x * ING_THREADS;
    const int64_t n_round = (n + 31) / 32 * 32;               // whole warps stay converged for the match
    for (int64_t e = (int64_t)blockIdx.x * ING_THREADS + threadIdx.x; e < n_round; e += stride) {
        bool ok = e < n;
        int v = 0, b = 0;
        if (ok) {
            v = vox[e];
            b = beam[e];
            const float a = val[e];
            if (v < 0 || v >= n_voxels || b < 0 || b >= n_beamlets) { atomicOr(flags + FLAG_RANGE, 1); ok = false; }
            if (!isfinite(a)) atomicOr(flags + FLAG_NONFINITE, 1);
        }
        (void)warp_agg_take(cntV, v, ok);
        (void)warp_agg_take(cntB, b, ok);
    }
}

// Exclusive scan of n counts into int64 row pointers (ptr[n] = total); also the maximum count.
constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan(const uint32_t *__restrict__ cnt, int32_t n, int64_t *__restrict__ ptr, unsigned long long *max_out)
{
    __shared__ int64_t part[SCAN_THREADS];
    __shared__ unsigned int smax;
    const int t = threadIdx.x;
    if (t == 0) smax = 0;
    __syncthreads();
    const int64_t per = ((int64_t)n + SCAN_THREADS - 1) / SCAN_THREADS;
    const int64_t lo = min((int64_t)n, per * t), hi = min((int64_t)n, lo + per);
    int64_t s = 0;
    unsigned int mx = 0;
    for (int64_t i = lo; i < hi; ++i) { s += cnt[i]; mx = max(mx, cnt[i]); }
    part[t] = s;
    atomicMax(&smax, mx);
    __syncthreads();
    if (t == 0) {
        int64_t run = 0;
        for (int i = 0; i < SCAN_THREADS; ++i) { const int64_t c = part[i]; part[i] = run; run += c; }
        ptr[n] = run;
        *max_out = smax;
    }
    __syncthreads();
    int64_t run = part[t];
    for (int64_t i = lo; i < hi; ++i) { ptr[i] = run; run += cnt[i]; }
}

__global__ void __launch_bounds__(ING_THREADS)
k_scatter(const int32_t *__restrict__ vox, const int32_t *__restrict__ beam, const float *__restrict__ val,
          int64_t n, const int64_t *__restrict__ ptrD, const int64_t *__restrict__ ptrT,
          uint32_t *curV, uint32_t *curB, int32_t *__restrict__ idxD, float *__restrict__ valD,
          int32_t *__restrict__ idxT, float *__restrict__ valT)
{
    const int64_t stride = (int64_t)gridDim.x * ING_THREADS;
    const int64_t n_round = (n + 31) / 32 * 32;
    for (int64_t e = (int64_t)blockIdx.x * ING_THREADS + threadIdx.x; e < n_round; e += stride) {
        const bool ok = e < n;
        int v = 0, b = 0;
        float a = 0.f;
        if (ok) { v = vox[e]; b = beam[e]; a = val[e]; }
        const uint32_t sv = warp_agg_take(curV, v, ok);
        const uint32_t sb = warp_agg_take(curB, b, ok);
        if (ok) {
            const int64_t pd = ptrD[v] + sv, pt = ptrT[b] + sb;
            idxD[pd] = b; valD[pd] = a;
            idxT[pt] = v; valT[pt] = a;
        }
    }
}

// ---------------------------------------------------------------- per-row bitonic sort
// All compare-exchanges put the minimum at the lower position, so virtual +inf padding above `len`
// never moves and pairs that reach into it are simply skipped: any length, no power-of-two copy.
template <typename Cmpx>
__device__ __forceinline__ void bitonic_network(int len, int nt, Cmpx cmpx)
{
    int m = 1;
    while (m < len) m <<= 1;
    for (int k = 2; k <= m; k <<= 1) {
        const int hk = k >> 1;
        for (int t = threadIdx.x; t < (m >> 1); t += nt) {        // flip step: i <-> block end - offset
            const int blk = t / hk, off = t % hk;
            const int i = blk * k + off, l = blk * k + k - 1 - off;
            if (l < len) cmpx(i, l);
        }
        __syncthreads();
        for (int j = hk >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < (m >> 1); t += nt) {
                const int i = 2 * j * (t / j) + (t % j), l = i + j;
                if (l < len) cmpx(i, l);
            }
            __syncthreads();
        }
    }
}

// rows with lo < len <= hi, keys packed (idx << 32 | value bits) in shared memory
__global__ void k_sort_rows_smem(const int64_t *__restrict__ ptr, int32_t *idx, float *val, int lo, int hi,
                                 int *flags)
{
    extern __shared__ unsigned long long keys[];
    const int64_t s = ptr[blockIdx.x];
    const int64_t len64 = ptr[blockIdx.x + 1] - s;
    if (len64 <= lo || len64 > hi) return;
    const int len = (int)len64, nt = blockDim.x;
    for (int i = threadIdx.x; i < len; i += nt)
        keys[i] = ((unsigned long long)(uint32_t)idx[s + i] << 32) | __float_as_uint(val[s + i]);
    __syncthreads();
    bitonic_network(len, nt, [&](int i, int l) {
        const unsigned long long a = keys[i], b = keys[l];
        if (b < a) { keys[i] = b; keys[l] = a; }
    });
    for (int i = threadIdx.x; i < len; i += nt) {
        const unsigned long long k = keys[i];
        idx[s + i] = (int32_t)(k >> 32);
        val[s + i] = __uint_as_float((uint32_t)k);
        if (i > 0 && (uint32_t)(keys[i - 1] >> 32) == (uint32_t)(k >> 32)) atomicOr(flags + FLAG_DUP, 1);
    }
}

// rows longer than `lo`: in place in global memory (one CTA per row)
__global__ void k_sort_rows_gmem(const int64_t *__restrict__ ptr, int32_t *idx, float *val, int64_t lo, int *flags)
{
    const int64_t s = ptr[blockIdx.x];
    const int64_t len64 = ptr[blockIdx.x + 1] - s;
    if (len64 <= lo) return;
    const int len = (int)len64, nt = blockDim.x;      // a row holds < 2^31 entries (distinct int32 secondary indices)
    int32_t *ri = idx + s;
    float *rv = val + s;
    bitonic_network(len, nt, [&](int i, int l) {
        const int32_t a = ri[i], b = ri[l];
        if (b < a) {
            ri[i] = b; ri[l] = a;
            const float t = rv[i]; rv[i] = rv[l]; rv[l] = t;
        }
    });
    for (int i = threadIdx.x + 1; i < len; i += nt)
        if (ri[i] == ri[i - 1]) atomicOr(flags + FLAG_DUP, 1);
}

// ---------------------------------------------------------------- tile interleave (spmv.cuh)
// One warp per segment (a beamlet row of D^T when seg_row == NULL, else a dose segment of D): every full
// 256-entry tile is permuted in place so that stored word 8*l + t holds the tile's entry 32*t + l.
__global__ void __launch_bounds__(256)
k_interleave(const int64_t *__restrict__ ptr, const int32_t *__restrict__ seg_row, int n_seg,
             int32_t *idx, float *val)
{
    const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (w >= n_seg) return;
    const int r0 = seg_row ? seg_row[w] : w, r1 = seg_row ? seg_row[w + 1] : w + 1;
    const int64_t s = ptr[r0], e = ptr[r1];
    const Segment sg = segment_of(s, e);
    for (int64_t ti = 0; ti < sg.nt; ++ti) {
        const int64_t base = sg.a0 + ti * TILE;
        int32_t ci[8];
        float vi[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) { ci[t] = idx[base + t * 32 + lane]; vi[t] = val[base + t * 32 + lane]; }
        __syncwarp();
#pragma unroll
        for (int t = 0; t < 8; ++t) { idx[base + lane * 8 + t] = ci[t]; val[base + lane * 8 + t] = vi[t]; }
        __syncwarp();
    }
}

constexpr int SORT_SMALL = 2048;       // 16 KB of keys, 256 threads
constexpr int SORT_BIG = 24576;        // 192 KB of keys, 1024 threads

static int sort_layout(const CsrLayout &A, int64_t max_len, int *flags, cudaStream_t st)
{
    if (A.n_rows == 0 || max_len <= 1) return VMAT_OK;
    k_sort_rows_smem<<<A.n_rows, 256, SORT_SMALL * 8, st>>>(A.ptr, A.idx, A.val, 1, SORT_SMALL, flags);
    VMAT_LAUNCH_CHECK();
    if (max_len > SORT_SMALL) {
        VMAT_CUDA(cudaFuncSetAttribute(k_sort_rows_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_BIG * 8));
        k_sort_rows_smem<<<A.n_rows, 1024, SORT_BIG * 8, st>>>(A.ptr, A.idx, A.val, SORT_SMALL, SORT_BIG, flags);
        VMAT_LAUNCH_CHECK();
    }
    if (max_len > SORT_BIG) {
        k_sort_rows_gmem<<<A.n_rows, 1024, 0, st>>>(A.ptr, A.idx, A.val, SORT_BIG, flags);
        VMAT_LAUNCH_CHECK();
    }
    return VMAT_OK;
}

static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <typename T>
static int dev_alloc(T **p, int64_t n, int64_t *bytes)
{
    const size_t b = (size_t)std::max<int64_t>(n, 1) * sizeof(T);
    VMAT_CUDA(cudaMalloc((void **)p, b));
    *bytes += (int64_t)b;
    return VMAT_OK;
}

#define TRY(x) do { int rc_ = (x); if (rc_ != VMAT_OK) return rc_; } while (0)

int vmat_build_layouts(vmat_ddc *h, const int32_t *coo_voxel, const int32_t *coo_beamlet,
                       const float *coo_val, cudaStream_t st)
{
    const int64_t nnz = h->nnz;
    const int32_t nv = h->n_voxels, nb = h->n_beamlets;
    const int64_t PAD = 16;                                  // 256-bit loads may read up to 7 entries past a row
    h->D.n_rows = nv; h->D.nnz = nnz;
    h->Dt.n_rows = nb; h->Dt.nnz = nnz;
    TRY(dev_alloc(&h->D.ptr, (int64_t)nv + 1, &h->bytes_device));
    TRY(dev_alloc(&h->Dt.ptr, (int64_t)nb + 1, &h->bytes_device));
    TRY(dev_alloc(&h->D.idx, nnz + PAD, &h->bytes_device));
    TRY(dev_alloc(&h->D.val, nnz + PAD, &h->bytes_device));
    TRY(dev_alloc(&h->Dt.idx, nnz + PAD, &h->bytes_device));
    TRY(dev_alloc(&h->Dt.val, nnz + PAD, &h->bytes_device));
    VMAT_CUDA(cudaMemsetAsync(h->D.idx + nnz, 0, PAD * 4, st));
    VMAT_CUDA(cudaMemsetAsync(h->D.val + nnz, 0, PAD * 4, st));
    VMAT_CUDA(cudaMemsetAsync(h->Dt.idx + nnz, 0, PAD * 4, st));
    VMAT_CUDA(cudaMemsetAsync(h->Dt.val + nnz, 0, PAD * 4, st));

    // scratch (freed before returning)
    uint32_t *cntV = nullptr, *cntB = nullptr;
    int *flags = nullptr;
    unsigned long long *maxes = nullptr;
    int32_t *stg_v = nullptr, *stg_b = nullptr;
    float *stg_a = nullptr;
    int64_t scratch_bytes = 0;
    struct Guard {
        void **p[7]; int n = 0;
        ~Guard() { for (int i = 0; i < n; ++i) if (*p[i]) cudaFree(*p[i]); }
        void add(void **q) { p[n++] = q; }
    } guard;
    guard.add((void **)&cntV); guard.add((void **)&cntB); guard.add((void **)&flags); guard.add((void **)&maxes);
    guard.add((void **)&stg_v); guard.add((void **)&stg_b); guard.add((void **)&stg_a);
    TRY(dev_alloc(&cntV, nv, &scratch_bytes));
    TRY(dev_alloc(&cntB, nb, &scratch_bytes));
    TRY(dev_alloc(&flags, N_FLAGS, &scratch_bytes));
    TRY(dev_alloc(&maxes, 2, &scratch_bytes));
    VMAT_CUDA(cudaMemsetAsync(cntV, 0, (size_t)std::max(nv, 1) * 4, st));
    VMAT_CUDA(cudaMemsetAsync(cntB, 0, (size_t)std::max(nb, 1) * 4, st));
    VMAT_CUDA(cudaMemsetAsync(flags, 0, N_FLAGS * sizeof(int), st));

    const bool on_dev = nnz == 0 || (is_device_ptr(coo_voxel) && is_device_ptr(coo_beamlet) && is_device_ptr(coo_val));
    if (!on_dev && (is_device_ptr(coo_voxel) || is_device_ptr(coo_beamlet) || is_device_ptr(coo_val))) {
        vmat_set_error("vmat_ddc_create: the three COO arrays must be all host or all device memory");
        return VMAT_ERR_INVALID_ARG;
    }
    const int64_t CH = on_dev ? std::max<int64_t>(nnz, 1) : std::min<int64_t>(std::max<int64_t>(nnz, 1), int64_t(1) << 25);
    if (!on_dev) {
        TRY(dev_alloc(&stg_v, CH, &scratch_bytes));
        TRY(dev_alloc(&stg_b, CH, &scratch_bytes));
        TRY(dev_alloc(&stg_a, CH, &scratch_bytes));
    }
    auto grid_for = [](int64_t n) { return (int)std::min<int64_t>((n + ING_THREADS - 1) / ING_THREADS, 148 * 32); };

    for (int pass = 0; pass < 2; ++pass) {
        for (int64_t c0 = 0; c0 < nnz; c0 += CH) {
            const int64_t n = std::min(CH, nnz - c0);
            const int32_t *v = coo_voxel + c0, *b = coo_beamlet + c0;
            const float *a = coo_val + c0;
            if (!on_dev) {
                VMAT_CUDA(cudaMemcpyAsync(stg_v, v, n * 4, cudaMemcpyHostToDevice, st));
                VMAT_CUDA(cudaMemcpyAsync(stg_b, b, n * 4, cudaMemcpyHostToDevice, st));
                VMAT_CUDA(cudaMemcpyAsync(stg_a, a, n * 4, cudaMemcpyHostToDevice, st));
                v = stg_v; b = stg_b; a = stg_a;
            }
            if (pass == 0)
                k_count<<<grid_for(n), ING_THREADS, 0, st>>>(v, b, a, n, nv, nb, cntV, cntB, flags);
            else
                k_scatter<<<grid_for(n), ING_THREADS, 0, st>>>(v, b, a, n, h->D.ptr, h->Dt.ptr, cntV, cntB,
                                                               h->D.idx, h->D.val, h->Dt.idx, h->Dt.val);
            VMAT_LAUNCH_CHECK();
        }
        if (pass == 0) {
            int hf[N_FLAGS];
            VMAT_CUDA(cudaMemcpyAsync(hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
            VMAT_CUDA(cudaStreamSynchronize(st));
            if (hf[FLAG_RANGE]) { vmat_set_error("vmat_ddc_create: COO index out of range"); return VMAT_ERR_INDEX_RANGE; }
            if (hf[FLAG_NONFINITE]) { vmat_set_error("vmat_ddc_create: non-finite COO value"); return VMAT_ERR_NONFINITE; }
            k_scan<<<1, SCAN_THREADS, 0, st>>>(cntV, nv, h->D.ptr, maxes + 0);
            VMAT_LAUNCH_CHECK();
            k_scan<<<1, SCAN_THREADS, 0, st>>>(cntB, nb, h->Dt.ptr, maxes + 1);
            VMAT_LAUNCH_CHECK();
            VMAT_CUDA(cudaMemsetAsync(cntV, 0, (size_t)std::max(nv, 1) * 4, st));
            VMAT_CUDA(cudaMemsetAsync(cntB, 0, (size_t)std::max(nb, 1) * 4, st));
        }
    }
    unsigned long long hmax[2] = {0, 0};
    VMAT_CUDA(cudaMemcpyAsync(hmax, maxes, sizeof(hmax), cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaStreamSynchronize(st));
    h->max_voxel_row_nnz = (int64_t)hmax[0];
    h->max_beamlet_row_nnz = (int64_t)hmax[1];
    TRY(sort_layout(h->D, h->max_voxel_row_nnz, flags, st));
    TRY(sort_layout(h->Dt, h->max_beamlet_row_nnz, flags, st));
    int hf[N_FLAGS];
    VMAT_CUDA(cudaMemcpyAsync(hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaStreamSynchronize(st));
    if (hf[FLAG_DUP]) { vmat_set_error("vmat_ddc_create: duplicate (voxel, beamlet) pair"); return VMAT_ERR_DUPLICATE; }

    // ---- dose kernel segments (host, from the voxel row pointers): a long row alone, or consecutive
    //      short rows with at most DOSE_SEG_NNZ non-zeros together
    std::vector<int64_t> hptr((size_t)nv + 1);
    VMAT_CUDA(cudaMemcpy(hptr.data(), h->D.ptr, ((size_t)nv + 1) * 8, cudaMemcpyDeviceToHost));
    std::vector<int32_t> seg;
    seg.push_back(0);
    int32_t r = 0;
    while (r < nv) {
        int32_t r1 = r + 1;                                   // a segment always takes at least one row
        while (r1 < nv && r1 - r < DOSE_MAX_ROWS && hptr[r1 + 1] - hptr[r] <= DOSE_SEG_NNZ) ++r1;
        seg.push_back(r1);
        r = r1;
    }
    h->n_seg = (int32_t)seg.size() - 1;
    h->n_blocks = (h->n_seg + DOSE_THREADS / 32 - 1) / (DOSE_THREADS / 32);
    TRY(dev_alloc(&h->seg_row, (int64_t)seg.size(), &h->bytes_device));
    VMAT_CUDA(cudaMemcpy(h->seg_row, seg.data(), seg.size() * 4, cudaMemcpyHostToDevice));
    h->h_seg_row = seg;
    // ---- tile-interleave both layouts: segments = dose segments of D, beamlet rows of D^T
    if (nnz > 0) {
        k_interleave<<<(h->n_seg + 7) / 8, 256, 0, st>>>(h->D.ptr, h->seg_row, h->n_seg, h->D.idx, h->D.val);
        VMAT_LAUNCH_CHECK();
        k_interleave<<<(nb + 7) / 8, 256, 0, st>>>(h->Dt.ptr, nullptr, nb, h->Dt.idx, h->Dt.val);
        VMAT_LAUNCH_CHECK();
        VMAT_CUDA(cudaStreamSynchronize(st));
    }
    TRY(dev_alloc(&h->F_partial, h->n_blocks, &h->bytes_device));
    h->n_obj_blocks = (nv + 255) / 256;
    TRY(dev_alloc(&h->F_partial_obj, h->n_obj_blocks, &h->bytes_device));
    return VMAT_OK;
}
