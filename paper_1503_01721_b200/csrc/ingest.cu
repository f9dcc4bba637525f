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
//   pack       the canonical CSR arrays are cut into segments and 32-entry groups and copied into the
//              final padded, tile-interleaved arrays (spmv.cuh), with u16 offsets + a base per group where
//              that is smaller than int32 indices; the canonical arrays are freed
// Host-resident COO is streamed through a device staging buffer in chunks, twice.
#include "spmv.cuh"
#include <vector>
#include <algorithm>
#include <climits>

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
          int32_t *__restrict__ idxT, float *__restrict__ valT, const int32_t *__restrict__ col_perm)
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
            idxD[pd] = col_perm ? col_perm[b] : b; valD[pd] = a;       // CSR(D) in the tiled column order (common.cuh)
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

// ---------------------------------------------------------------- pack: canonical CSR -> grouped, padded layout
// One warp per segment (rows [seg_row[w], seg_row[w+1]); seg_row == NULL: segment w = row w).  The warp
// walks the segment's canonical entries and forms groups greedily: a group takes the next entries while it
// holds fewer than 32 and the span max - min of its secondary indices stays <= span_limit (65535 for u16
// offsets; INT32_MAX for the wide format, where only the segment's last group is short).  Greedy prefixes
// give the fewest groups any such partition can have, in particular never more than packing each row alone.
//   WRITE = false: n_groups[w] = number of groups of the segment.
//   WRITE = true : gstart[w] = first group of the segment (exclusive scan of n_groups); writes the values,
//                  offsets + bases (narrow) or indices (wide) at their tile-interleaved position, pads
//                  (value 0, index of the entry before) and the padded row starts pptr.
template <bool WRITE>
__global__ void __launch_bounds__(256)
k_pack(const int64_t *__restrict__ ptr, const int32_t *__restrict__ cidx, const float *__restrict__ cval,
       const int32_t *__restrict__ seg_row, int n_seg, int64_t span_limit, bool narrow,
       uint32_t *__restrict__ n_groups, const int64_t *__restrict__ gstart,
       float *__restrict__ val, void *__restrict__ sec, int32_t *__restrict__ base, int64_t *__restrict__ pptr)
{
    const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (w >= n_seg) return;
    const int r0 = seg_row ? seg_row[w] : w, r1 = seg_row ? seg_row[w + 1] : w + 1;
    const int64_t s = ptr[r0], e = ptr[r1];
    int64_t S = 0, G = 0;
    if (WRITE) { S = gstart[w] * GROUP; G = gstart[w + 1] - gstart[w]; }
    int64_t k = s, gl = 0;
    while (k < e) {
        const bool valid = k + lane < e;
        const int c = valid ? cidx[k + lane] : 0;
        int mn = valid ? c : INT32_MAX, mx = valid ? c : INT32_MIN;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {                       // inclusive prefix min / max
            const int a = __shfl_up_sync(0xffffffffu, mn, o), b = __shfl_up_sync(0xffffffffu, mx, o);
            if (lane >= o) { mn = min(mn, a); mx = max(mx, b); }
        }
        const bool ok = valid && (int64_t)mx - (int64_t)mn <= span_limit;
        const int n_take = __popc(__ballot_sync(0xffffffffu, ok));       // a prefix of the lanes, >= 1
        if (WRITE) {
            const int b = __shfl_sync(0xffffffffu, mn, n_take - 1);       // the group's minimum index
            const int c_last = __shfl_sync(0xffffffffu, c, n_take - 1);
            const bool real = lane < n_take;
            const int ci = real ? c : c_last;                             // pad: index of the entry before it
            const float vi = real ? cval[k + lane] : 0.f;
            const int64_t pos = stored_pos(S, G, S + gl * GROUP + lane);
            val[pos] = vi;
            if (narrow) {
                ((uint16_t *)sec)[pos] = (uint16_t)(ci - b);
                if (lane == 0) base[gstart[w] + gl] = b;
            } else {
                ((int32_t *)sec)[pos] = ci;
            }
            for (int r = r0 + lane; r < r1; r += 32) {                    // rows whose first entry is in this group
                const int64_t pr = ptr[r];
                if (pr >= k && pr < k + n_take) pptr[r] = S + gl * GROUP + (pr - k);
            }
        }
        k += n_take;
        ++gl;
    }
    if (WRITE) {
        for (int r = r0 + lane; r < r1; r += 32)                          // empty rows at the segment's end
            if (ptr[r] == e) pptr[r] = S + G * GROUP;
    } else if (lane == 0) {
        n_groups[w] = (uint32_t)gl;
    }
}

// Narrow layouts, after the pack: every full tile whose 256 indices span <= 65535 gets ONE base (its minimum)
// for all 8 groups, flagged in bit 31 of the tile's first base word (spmv.cuh: the kernels then read one
// broadcast word per tile instead of shuffling 8 bases around).  One warp per segment.
__global__ void __launch_bounds__(256)
k_tile_base(const int64_t *__restrict__ pptr, const int32_t *__restrict__ seg_row, int n_seg,
            uint16_t *__restrict__ off, int32_t *__restrict__ base, unsigned long long *__restrict__ n_tiles /* [2]: all, uniform */)
{
    const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (w >= n_seg) return;
    const int r0 = seg_row ? seg_row[w] : w, r1 = seg_row ? seg_row[w + 1] : w + 1;
    const int64_t s = pptr[r0], e = pptr[r1];
    const int nt = (int)((e - s) >> 8);
    int n_uniform = 0;
    for (int ti = 0; ti < nt; ++ti) {
        const int64_t k = s + (int64_t)ti * TILE;
        int c[8], mn = INT32_MAX, mx = INT32_MIN;
#pragma unroll
        for (int t = 0; t < 8; ++t) {                              // stored word 8*lane + t = entry `lane` of group t
            c[t] = base[(k >> 5) + t] + (int)off[k + 8 * lane + t];
            mn = min(mn, c[t]); mx = max(mx, c[t]);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
            mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        }
        if ((int64_t)mx - (int64_t)mn > 65535) continue;           // warp-uniform
#pragma unroll
        for (int t = 0; t < 8; ++t) off[k + 8 * lane + t] = (uint16_t)(c[t] - mn);
        __syncwarp();
        if (lane < 8) base[(k >> 5) + lane] = lane == 0 ? (mn | TILE_UNIFORM_BIT) : mn;
        ++n_uniform;
    }
    if (lane == 0 && nt > 0) {
        atomicAdd(n_tiles + 0, (unsigned long long)nt);
        atomicAdd(n_tiles + 1, (unsigned long long)n_uniform);
    }
}

constexpr int SORT_SMALL = 2048;       // 16 KB of keys, 256 threads
constexpr int SORT_BIG = 24576;        // 192 KB of keys, 1024 threads

struct CanonCsr { int32_t n_rows; int64_t *ptr; int32_t *idx; float *val; };

static int sort_layout(const CanonCsr &A, int64_t max_len, int *flags, cudaStream_t st)
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

// frees device scratch on every exit path
struct DevGuard {
    std::vector<void **> p;
    ~DevGuard() { for (void **q : p) if (*q) { cudaFree(*q); *q = nullptr; } }
    void add(void **q) { p.push_back(q); }
};

// ---------------------------------------------------------------- segments + groups of one layout
struct PackPlan {
    bool narrow = false;
    std::vector<int32_t> seg;          // segment -> first row, [n_seg+1] (empty when every row is a segment)
    int32_t n_seg = 0;
    int32_t *d_seg = nullptr;          // device copy of seg (NULL when every row is a segment)
    int64_t *d_gstart = nullptr;       // [n_seg+1] first group of each segment
    int64_t P = 0;                     // padded entries
    void release() { if (d_seg) cudaFree(d_seg); if (d_gstart) cudaFree(d_gstart); d_seg = nullptr; d_gstart = nullptr; }
};

// Plans the layout of the canonical CSR C in the given format.  group_short: voxel rows (D) - consecutive
// short rows share a warp; otherwise every row is its own segment (beamlet rows of D^T).
static int plan_layout(const CanonCsr &C, bool narrow, bool group_short, PackPlan *pl, cudaStream_t st)
{
    const int32_t n_rows = C.n_rows;
    const int64_t span = narrow ? 65535 : (int64_t)INT32_MAX;
    uint32_t *d_cnt = nullptr;
    unsigned long long *d_max = nullptr;
    DevGuard guard;
    guard.add((void **)&d_cnt); guard.add((void **)&d_max);
    int64_t dummy = 0;
    TRY(dev_alloc(&d_cnt, n_rows, &dummy));
    TRY(dev_alloc(&d_max, 1, &dummy));
    pl->narrow = narrow;
    const int grid_rows = (n_rows + 7) / 8;
    if (n_rows > 0) {                                            // groups of every row packed alone
        k_pack<false><<<grid_rows, 256, 0, st>>>(C.ptr, C.idx, C.val, nullptr, n_rows, span, narrow, d_cnt, nullptr,
                                                 nullptr, nullptr, nullptr, nullptr);
        VMAT_LAUNCH_CHECK();
    }
    pl->n_seg = n_rows;
    if (group_short) {
        // dose-kernel segments: a row of more than DOSE_SEG_NNZ padded entries alone, else consecutive rows
        // with at most DOSE_SEG_NNZ padded entries together (packed together they never need more groups)
        std::vector<uint32_t> c((size_t)std::max(n_rows, 1));
        VMAT_CUDA(cudaMemcpyAsync(c.data(), d_cnt, (size_t)n_rows * 4, cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(cudaStreamSynchronize(st));
        const uint32_t SEG_GROUPS = DOSE_SEG_NNZ / GROUP;
        pl->seg.clear();
        pl->seg.push_back(0);
        int32_t r = 0;
        while (r < n_rows) {
            int32_t q = r + 1;                                   // a segment always takes at least one row
            uint64_t tot = c[r];
            while (q < n_rows && q - r < DOSE_MAX_ROWS && tot + c[q] <= SEG_GROUPS) tot += c[q++];
            pl->seg.push_back(q);
            r = q;
        }
        pl->n_seg = (int32_t)pl->seg.size() - 1;
        TRY(dev_alloc(&pl->d_seg, (int64_t)pl->seg.size(), &dummy));
        VMAT_CUDA(cudaMemcpyAsync(pl->d_seg, pl->seg.data(), pl->seg.size() * 4, cudaMemcpyHostToDevice, st));
        if (pl->n_seg > 0) {
            k_pack<false><<<(pl->n_seg + 7) / 8, 256, 0, st>>>(C.ptr, C.idx, C.val, pl->d_seg, pl->n_seg, span, narrow,
                                                               d_cnt, nullptr, nullptr, nullptr, nullptr, nullptr);
            VMAT_LAUNCH_CHECK();
        }
    }
    TRY(dev_alloc(&pl->d_gstart, (int64_t)pl->n_seg + 1, &dummy));
    k_scan<<<1, SCAN_THREADS, 0, st>>>(d_cnt, pl->n_seg, pl->d_gstart, d_max);
    VMAT_LAUNCH_CHECK();
    int64_t total = 0;
    VMAT_CUDA(cudaMemcpyAsync(&total, pl->d_gstart + pl->n_seg, 8, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaStreamSynchronize(st));
    pl->P = total * GROUP;
    if (pl->P >= (int64_t)1 << 35) {                     // spmv.cuh: the kernels' cursor counts units of 8 entries in 32 bits
        vmat_set_error("vmat_ddc_create: %lld padded entries exceed the layout limit of 2^35", (long long)pl->P);
        return VMAT_ERR_INVALID_ARG;
    }
    return VMAT_OK;
}

// Chooses the format (index_bits: 16, 32, or 0 = the smaller one), allocates the final arrays of layout A
// and fills them from the canonical CSR C.  A.ptr is C.ptr (kept); A.pptr must be allocated.
static int pack_layout(vmat_ddc *h, PackedLayout &A, const CanonCsr &C, int32_t n_cols, bool group_short,
                       int index_bits, PackPlan *chosen, cudaStream_t st)
{
    PackPlan narrow_pl, wide_pl;
    struct Rel { PackPlan &a, &b; ~Rel() { a.release(); b.release(); } } rel{narrow_pl, wide_pl};
    bool use_narrow;
    if (index_bits == 16 || (index_bits == 0 && n_cols <= 65536)) {          // every span fits: no early closes
        TRY(plan_layout(C, true, group_short, &narrow_pl, st));
        use_narrow = true;
    } else if (index_bits == 32) {
        TRY(plan_layout(C, false, group_short, &wide_pl, st));
        use_narrow = false;
    } else {
        TRY(plan_layout(C, true, group_short, &narrow_pl, st));
        TRY(plan_layout(C, false, group_short, &wide_pl, st));
        // bytes per padded entry: 6.125 narrow, 8 wide; narrow must save at least 5 %
        use_narrow = 6.125 * (double)narrow_pl.P <= 0.95 * 8.0 * (double)wide_pl.P;
    }
    PackPlan &pl = use_narrow ? narrow_pl : wide_pl;
    A.P = pl.P;
    A.index_bits = use_narrow ? 16 : 32;
    const int64_t SLACK = 64;
    TRY(dev_alloc(&A.val, A.P + SLACK, &h->bytes_device));
    if (use_narrow) {
        uint16_t *off = nullptr;
        TRY(dev_alloc(&off, A.P + SLACK, &h->bytes_device));
        A.sec = off;
        TRY(dev_alloc(&A.base, A.P / GROUP + SLACK, &h->bytes_device));
    } else {
        int32_t *idx = nullptr;
        TRY(dev_alloc(&idx, A.P + SLACK, &h->bytes_device));
        A.sec = idx;
    }
    if (pl.n_seg > 0) {
        k_pack<true><<<(pl.n_seg + 7) / 8, 256, 0, st>>>(C.ptr, C.idx, C.val, pl.d_seg, pl.n_seg,
                                                         use_narrow ? 65535 : (int64_t)INT32_MAX, use_narrow, nullptr,
                                                         pl.d_gstart, A.val, A.sec, A.base, A.pptr);
        VMAT_LAUNCH_CHECK();
    }
    VMAT_CUDA(cudaMemcpyAsync(A.pptr + A.n_rows, &A.P, 8, cudaMemcpyHostToDevice, st));
    if (use_narrow && pl.n_seg > 0) {
        unsigned long long *d_nt = nullptr, h_nt[2] = {0, 0};
        DevGuard g2;
        g2.add((void **)&d_nt);
        int64_t dummy = 0;
        TRY(dev_alloc(&d_nt, 2, &dummy));
        VMAT_CUDA(cudaMemsetAsync(d_nt, 0, 16, st));
        k_tile_base<<<(pl.n_seg + 7) / 8, 256, 0, st>>>(A.pptr, pl.d_seg, pl.n_seg, (uint16_t *)A.sec, A.base, d_nt);
        VMAT_LAUNCH_CHECK();
        VMAT_CUDA(cudaMemcpyAsync(h_nt, d_nt, 16, cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(cudaStreamSynchronize(st));
        A.n_tiles = (int64_t)h_nt[0];
        A.n_tiles_uniform = (int64_t)h_nt[1];
    }
    VMAT_CUDA(cudaStreamSynchronize(st));
    if (chosen) {                                               // hand the segment table to the caller
        chosen->seg = pl.seg; chosen->n_seg = pl.n_seg; chosen->d_seg = pl.d_seg; pl.d_seg = nullptr;
    }
    return VMAT_OK;
}

int vmat_build_layouts(vmat_ddc *h, const int32_t *coo_voxel, const int32_t *coo_beamlet,
                       const float *coo_val, int index_bits, cudaStream_t st)
{
    const int64_t nnz = h->nnz;
    const int32_t nv = h->n_voxels, nb = h->n_beamlets;
    h->D.n_rows = nv; h->D.nnz = nnz;
    h->Dt.n_rows = nb; h->Dt.nnz = nnz;
    TRY(dev_alloc(&h->D.ptr, (int64_t)nv + 1, &h->bytes_device));
    TRY(dev_alloc(&h->Dt.ptr, (int64_t)nb + 1, &h->bytes_device));
    TRY(dev_alloc(&h->D.pptr, (int64_t)nv + 1, &h->bytes_device));
    TRY(dev_alloc(&h->Dt.pptr, (int64_t)nb + 1, &h->bytes_device));

    // scratch (freed before returning): the canonical CSR arrays of both layouts, counters, staging
    CanonCsr cD{nv, h->D.ptr, nullptr, nullptr}, cT{nb, h->Dt.ptr, nullptr, nullptr};
    uint32_t *cntV = nullptr, *cntB = nullptr;
    int *flags = nullptr;
    unsigned long long *maxes = nullptr;
    int32_t *stg_v = nullptr, *stg_b = nullptr;
    float *stg_a = nullptr;
    int64_t scratch_bytes = 0;
    DevGuard guard;
    guard.add((void **)&cD.idx); guard.add((void **)&cD.val); guard.add((void **)&cT.idx); guard.add((void **)&cT.val);
    guard.add((void **)&cntV); guard.add((void **)&cntB); guard.add((void **)&flags); guard.add((void **)&maxes);
    guard.add((void **)&stg_v); guard.add((void **)&stg_b); guard.add((void **)&stg_a);
    TRY(dev_alloc(&cD.idx, nnz, &scratch_bytes));
    TRY(dev_alloc(&cD.val, nnz, &scratch_bytes));
    TRY(dev_alloc(&cT.idx, nnz, &scratch_bytes));
    TRY(dev_alloc(&cT.val, nnz, &scratch_bytes));
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
                k_scatter<<<grid_for(n), ING_THREADS, 0, st>>>(v, b, a, n, cD.ptr, cT.ptr, cntV, cntB,
                                                               cD.idx, cD.val, cT.idx, cT.val, h->col_perm);
            VMAT_LAUNCH_CHECK();
        }
        if (pass == 0) {
            int hf[N_FLAGS];
            VMAT_CUDA(cudaMemcpyAsync(hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
            VMAT_CUDA(cudaStreamSynchronize(st));
            if (hf[FLAG_RANGE]) { vmat_set_error("vmat_ddc_create: COO index out of range"); return VMAT_ERR_INDEX_RANGE; }
            if (hf[FLAG_NONFINITE]) { vmat_set_error("vmat_ddc_create: non-finite COO value"); return VMAT_ERR_NONFINITE; }
            k_scan<<<1, SCAN_THREADS, 0, st>>>(cntV, nv, cD.ptr, maxes + 0);
            VMAT_LAUNCH_CHECK();
            k_scan<<<1, SCAN_THREADS, 0, st>>>(cntB, nb, cT.ptr, maxes + 1);
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
    TRY(sort_layout(cD, h->max_voxel_row_nnz, flags, st));
    TRY(sort_layout(cT, h->max_beamlet_row_nnz, flags, st));
    int hf[N_FLAGS];
    VMAT_CUDA(cudaMemcpyAsync(hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(cudaStreamSynchronize(st));
    if (hf[FLAG_DUP]) { vmat_set_error("vmat_ddc_create: duplicate (voxel, beamlet) pair"); return VMAT_ERR_DUPLICATE; }

    // ---- pack D (voxel rows; dose-kernel segments), free its canonical arrays, then D^T (one segment per row)
    PackPlan segD;
    TRY(pack_layout(h, h->D, cD, nb, true, index_bits, &segD, st));
    cudaFree(cD.idx); cD.idx = nullptr;
    cudaFree(cD.val); cD.val = nullptr;
    h->seg_row = segD.d_seg;                                    // owned by the handle from here on
    h->bytes_device += (int64_t)segD.seg.size() * 4;
    h->n_seg = segD.n_seg;
    h->n_blocks = (h->n_seg + DOSE_THREADS / 32 - 1) / (DOSE_THREADS / 32);
    h->h_seg_row = segD.seg;
    TRY(pack_layout(h, h->Dt, cT, nv, false, index_bits, nullptr, st));
    TRY(dev_alloc(&h->F_partial, h->n_blocks, &h->bytes_device));
    h->n_obj_blocks = (nv + 255) / 256;
    TRY(dev_alloc(&h->F_partial_obj, h->n_obj_blocks, &h->bytes_device));
    return VMAT_OK;
}
