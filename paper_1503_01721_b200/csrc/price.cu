// price.cu - A3 beamlet prices p = D^T g (Eq. (3), "Pi = D^T g" L121) through the
// beamlet-row CSR, A4 per-leaf-row best opening and A5 aperture price / best control point (L133).
//
// Beamlet rows are long and even (a radius-`cutoff` cylinder through the body: 10^3-10^4 non-zeros),
// so the paper's mapping holds on sm_100a: one warp per beamlet row (L127), here over lane-interleaved
// 256-entry tiles read with 256-bit loads, with u16 index offsets where the layout allows (spmv.cuh).  Measured on B200 the warp-per-row kernel beats
// a CTA-per-leaf-row kernel by 12 % (perfect balance, more independent streams), so the row selection
// is fused differently: for every ITEM (8 consecutive beamlet rows, the unit a CTA takes at a time) the CTA
// hands in tickets for the leaf rows it priced, and the CTA whose ticket completes a leaf row selects that
// row's opening on the spot - the selection costs no launch and no second pass over p, and the price kernel
// keeps its balance.  Items reach the CTAs one CTA per item or through the per-SM queues of smqueue.cuh.
//
// Selection arithmetic (readings C4-C6, C8): S_0 = 0, S_{c+1} = S_c + (double)p_c left to
// right in FP64; candidates all 0 <= L <= R <= n with V = S_R - S_L; result = smallest (V, L, R).
// All pairs are enumerated - the definition itself, n <= ~10^2 - so the leaf positions are
// bit-identical to the exhaustive CPU definition for the same FP32 p.
#include "spmv.cuh"
#include "smqueue.cuh"

struct Opening {
    double V;
    int L, R;
};
__device__ __forceinline__ bool opening_less(const Opening &a, const Opening &b)
{
    if (a.V != b.V) return a.V < b.V;
    if (a.L != b.L) return a.L < b.L;
    return a.R < b.R;
}

// Best opening of one leaf row whose n FP32 prices are sp[0..n).  S: n+1 doubles of scratch.
// Executed by all NT threads of the CTA; the result is returned in thread 0.
template <int NT>
__device__ __forceinline__ Opening select_row(const float *sp, int n, double *S, Opening *red /* [NT/32] */)
{
    if (threadIdx.x == 0) {
        double s = 0.0;
        S[0] = 0.0;
        for (int c = 0; c < n; ++c) {
            s = s + (double)sp[c];                 // strictly left to right
            S[c + 1] = s;
        }
    }
    __syncthreads();
    Opening best = {0.0, 0, 0};                    // the closed opening (C4)
    for (int L = threadIdx.x; L <= n; L += NT) {
        const double SL = S[L];
        for (int R = L; R <= n; ++R) {
            const double V = S[R] - SL;
            if (V < best.V) { best.V = V; best.L = L; best.R = R; }   // visited in (L,R) order: strict < keeps the first
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Opening other;
        other.V = __shfl_xor_sync(0xffffffffu, best.V, o);
        other.L = __shfl_xor_sync(0xffffffffu, best.L, o);
        other.R = __shfl_xor_sync(0xffffffffu, best.R, o);
        if (opening_less(other, best)) best = other;
    }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0)
        for (int i = 1; i < NT / 32; ++i)
            if (opening_less(red[i], best)) best = red[i];
    return best;
}

// Best opening of one leaf row by ONE WARP (the fused path).  p_row: the row's n prices in global memory,
// written by other warps (read through L2).  S: n+1 doubles of global scratch private to this row.
__device__ __noinline__ Opening warp_select_row(const float *p_row, int n, double *S, int lane)
{
    if (lane == 0) {
        double s = 0.0;
        S[0] = 0.0;
        for (int c = 0; c < n; ++c) {
            s = s + (double)__ldcg(p_row + c);     // strictly left to right
            S[c + 1] = s;
        }
    }
    __syncwarp();
    Opening best = {0.0, 0, 0};                    // the closed opening (C4)
    for (int L = lane; L <= n; L += 32) {
        const double SL = S[L];
        for (int R = L; R <= n; ++R) {
            const double V = S[R] - SL;
            if (V < best.V) { best.V = V; best.L = L; best.R = R; }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Opening other;
        other.V = __shfl_xor_sync(0xffffffffu, best.V, o);
        other.L = __shfl_xor_sync(0xffffffffu, best.L, o);
        other.R = __shfl_xor_sync(0xffffffffu, best.R, o);
        if (opening_less(other, best)) best = other;
    }
    return best;
}

struct SelectArgs {
    const int32_t *beamlet_leafrow;      // [n_beamlets]
    const int32_t *leafrow_col_offset;   // [n_leaf_rows+1]
    const int32_t *leafrow_angle;        // [n_leaf_rows]
    const uint8_t *angle_mask;           // [n_angles] or NULL
    uint32_t *leafrow_done;              // [n_leaf_rows] tickets, zero between launches
    double *S;                           // [n_beamlets + n_leaf_rows + 1]
    int32_t *L, *R;
    double *row_price;
    int n_leaf_rows;
};

// ---------------------------------------------------------------- A3 (+ A4 fused): one warp per beamlet row
#ifndef VMAT_PRICE_MINB
#define VMAT_PRICE_MINB 6        // 40 registers, 1536 threads per SM: fastest of 4..8 on B200 (cfg 3)
#endif
// SKIP (the column-generation loop: prices are computed "at the unoccupied control points (k not in
// C)"): beamlet rows of occupied control points (sa.angle_mask) are not streamed, their price is written as 0.
template <bool SELECT, int FMT, bool SKIP = false>
__global__ void __launch_bounds__(PRICE_THREADS, VMAT_PRICE_MINB)
k_price(const int64_t *__restrict__ pptr, const MatView A, int n_rows, const float *__restrict__ g,
        float *__restrict__ p, SelectArgs sa, const SmQueues Q)
{
    __shared__ int s_item[3];
    __shared__ int done_rows[PRICE_WARPS];
    __shared__ int n_done;
    const int lane = threadIdx.x & 31;
    if (SELECT) {                                   // leaf rows without beamlets draw no ticket: close them here
        for (int r = blockIdx.x * PRICE_THREADS + threadIdx.x; r < sa.n_leaf_rows; r += gridDim.x * PRICE_THREADS)
            if (sa.leafrow_col_offset[r + 1] == sa.leafrow_col_offset[r]) {
                sa.L[r] = 0; sa.R[r] = 0; sa.row_price[r] = 0.0;
            }
    }
    const int warp = threadIdx.x >> 5;
    const int n_items = (n_rows + PRICE_WARPS - 1) / PRICE_WARPS;      // item = 8 consecutive beamlet rows
    sq_init(Q, s_item);
#pragma unroll 1
    for (;;) {
        const int item = sq_next_item(Q, s_item);
        if (item < 0 || item >= n_items) break;
        {
            const int row = item * PRICE_WARPS + warp;
            float acc = 0.f;
            if (row < n_rows && !(SKIP && sa.angle_mask[sa.leafrow_angle[sa.beamlet_leafrow[row]]] != 0))
                acc = warp_sum(segment_dot<FMT, VMAT_PRICE_DEPTH>(A, pptr[row], pptr[row + 1], g, lane));
            // the item is re-read from shared memory (nobody writes it before the next fetch): no register holds it
            // across the streaming loop, which has none to spare at 40 registers
            const int row_w = ((volatile int *)s_item)[0] * PRICE_WARPS + warp;
            if (lane == 0 && row_w < n_rows) p[row_w] = acc;                // 0 for a skipped row
        }
        if (SELECT) {
            // One ticket per item and leaf row: the item's 8 consecutive beamlet rows lie in a few leaf rows.
            // Thread 0 adds, for each of them, the number of its rows priced here; the CTA whose add
            // completes a leaf row selects that row's opening (warp w takes the w-th completed row).
            __syncthreads();                                                // the item's prices are written
            if (threadIdx.x == 0) {
                __threadfence();                                            // ... and visible before the tickets
                int nd = 0;
                const int row0 = ((volatile int *)s_item)[0] * PRICE_WARPS;
                const int row1 = min(row0 + PRICE_WARPS, n_rows);
                int c = row0;
                while (c < row1) {
                    const int r = sa.beamlet_leafrow[c];
                    const int j1 = sa.leafrow_col_offset[r + 1];
                    const int cnt = min(row1, j1) - c;                      // rows of leaf row r priced here
                    const int n = j1 - sa.leafrow_col_offset[r];
                    if (atomicAdd(sa.leafrow_done + r, (uint32_t)cnt) + cnt == (uint32_t)n) {
                        sa.leafrow_done[r] = 0;                             // ready for the next launch
                        done_rows[nd++] = r;
                    }
                    c += cnt;
                }
                if (nd > 0) __threadfence();
                n_done = nd;
            }
            __syncthreads();
            if (warp < n_done) {                                            // every price of leaf row r is written
                const int r = done_rows[warp];
                const int j0 = sa.leafrow_col_offset[r];
                const int n = sa.leafrow_col_offset[r + 1] - j0;
                const bool occupied = sa.angle_mask != nullptr && sa.angle_mask[sa.leafrow_angle[r]] != 0;   // C7
                const Opening best = warp_select_row(p + j0, occupied ? 0 : n, sa.S + j0 + r, lane);
                if (lane == 0) {
                    sa.L[r] = best.L;
                    sa.R[r] = best.R;
                    sa.row_price[r] = best.V;
                }
            }
        }
    }
}

// ---------------------------------------------------------------- A4 alone (vmat_select_apertures)
// S_glob: global scratch of n_beamlets + n_leaf_rows doubles, used only by rows longer than
// SELECT_MAX_ROW (NULL when no such row exists).
__global__ void __launch_bounds__(PRICE_THREADS)
k_select(const float *__restrict__ p, const int32_t *__restrict__ leafrow_col_offset,
         const int32_t *__restrict__ leafrow_angle, const uint8_t *__restrict__ angle_mask,
         double *__restrict__ S_glob, int32_t *__restrict__ Lout, int32_t *__restrict__ Rout,
         double *__restrict__ row_price)
{
    __shared__ double S[SELECT_MAX_ROW + 1];
    __shared__ float sp[SELECT_MAX_ROW];
    __shared__ Opening red[PRICE_WARPS];
    const int r = blockIdx.x;
    const int j0 = leafrow_col_offset[r];
    int n = leafrow_col_offset[r + 1] - j0;
    if (angle_mask != nullptr && angle_mask[leafrow_angle[r]] != 0) n = 0;               // C7
    Opening best;
    if (n <= SELECT_MAX_ROW) {
        for (int c = threadIdx.x; c < n; c += PRICE_THREADS) sp[c] = p[j0 + c];
        __syncthreads();
        best = select_row<PRICE_THREADS>(sp, n, S, red);
    } else {
        best = select_row<PRICE_THREADS>(p + j0, n, S_glob + j0 + r, red);
    }
    if (threadIdx.x == 0) {
        Lout[r] = best.L;
        Rout[r] = best.R;
        row_price[r] = best.V;
    }
}

// ---------------------------------------------------------------- A5: aperture price per control point, best one
// One warp per control point: the FP64 sum of its rows' prices IN ROW ORDER (lanes load 32 prices at a
// time, every lane then adds them one by one - the same additions in the same order as the definition).
// The CTA that draws the last ticket picks the best control point.
constexpr int ANGLE_THREADS = 256;
__global__ void __launch_bounds__(ANGLE_THREADS)
k_angle_price(int n_angles, const int32_t *__restrict__ angle_row_offset, const double *__restrict__ row_price,
              const uint8_t *__restrict__ angle_mask, double *__restrict__ angle_price,
              int32_t *__restrict__ best_angle, uint32_t *__restrict__ ticket)
{
    __shared__ double bv[ANGLE_THREADS / 32];
    __shared__ int bi[ANGLE_THREADS / 32];
    __shared__ int is_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.x * (ANGLE_THREADS / 32) + warp;
    if (a < n_angles) {
        double s;
        if (angle_mask != nullptr && angle_mask[a] != 0) {
            s = __longlong_as_double(0x7ff0000000000000LL);          // +inf: occupied (C7)
        } else {
            s = 0.0;
            const int r1 = angle_row_offset[a + 1];
            for (int base = angle_row_offset[a]; base < r1; base += 32) {
                const double v = base + lane < r1 ? row_price[base + lane] : 0.0;
                const int m = min(32, r1 - base);
                for (int i = 0; i < m; ++i) s += __shfl_sync(0xffffffffu, v, i);   // row order
            }
        }
        if (lane == 0) angle_price[a] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
        if (is_last) { *ticket = 0; __threadfence(); }
    }
    __syncthreads();
    if (!is_last) return;
    // arg-min over the unoccupied control points: smaller price wins, ties -> smaller index; -1 = none < 0 (L56)
    double best = 0.0;
    int besta = -1;
    for (int k = threadIdx.x; k < n_angles; k += ANGLE_THREADS) {
        const double v = __ldcg(angle_price + k);
        if (v < best) { best = v; besta = k; }                       // ascending k: strict < keeps the smallest k
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, best, o);
        const int oa = __shfl_xor_sync(0xffffffffu, besta, o);
        if (oa >= 0 && (besta < 0 || ov < best || (ov == best && oa < besta))) { best = ov; besta = oa; }
    }
    if (lane == 0) { bv[warp] = best; bi[warp] = besta; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < ANGLE_THREADS / 32; ++i)
            if (bi[i] >= 0 && (besta < 0 || bv[i] < best || (bv[i] == best && bi[i] < besta))) { best = bv[i]; besta = bi[i]; }
        best_angle[0] = besta;
    }
}

// ---------------------------------------------------------------- A5 across column blocks (NEXT-4)
__global__ void k_best_pair(int n_angles, const double *__restrict__ angle_price, const int32_t *__restrict__ best_angle,
                            int angle_lo, double *__restrict__ pair)
{
    const int b = best_angle[0];
    const bool ok = b >= 0 && b < n_angles;
    pair[0] = ok ? angle_price[b] : 0.0;
    pair[1] = ok ? (double)(b + angle_lo) : -1.0;
}
// smaller price wins, ties -> smaller control point; a pair without a control point (-1) never wins (L56)
__global__ void k_merge_best(const double *__restrict__ pairs, int n, double *__restrict__ best)
{
    double bp = 0.0, bk = -1.0;
    for (int i = 0; i < n; ++i) {
        const double p = pairs[2 * i], k = pairs[2 * i + 1];
        if (k >= 0.0 && (p < bp || (p == bp && bk >= 0.0 && k < bk))) { bp = p; bk = k; }
    }
    best[0] = bp;
    best[1] = bk;
}

int vmat_launch_best_pair(const vmat_ddc *h, const double *angle_price, const int32_t *best_angle, int32_t angle_lo,
                          double *pair, cudaStream_t st)
{
    k_best_pair<<<1, 1, 0, st>>>(h->n_angles, angle_price, best_angle, angle_lo, pair);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}
int vmat_launch_merge_best(const double *pairs, int32_t n, double *best, cudaStream_t st)
{
    k_merge_best<<<1, 1, 0, st>>>(pairs, n, best);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

// ---------------------------------------------------------------- launchers
// Launch geometry: SM-affine queues -> a persistent grid of SM count x resident CTAs per SM; static -> one CTA per item.
template <bool SELECT, int FMT, bool SKIP>
static int price_grid(const vmat_ddc *h)
{
    const int n_items = (h->n_beamlets + PRICE_WARPS - 1) / PRICE_WARPS;
    if (h->queues_price().nq == 0) return n_items;
    static std::atomic<int> occ[VMAT_MAX_DEVICES];                   // per kernel instance and device
    return min(n_items, h->n_sm * vmat_resident_ctas(k_price<SELECT, FMT, SKIP>, PRICE_THREADS, h->device, occ));
}
int vmat_price_grid(const vmat_ddc *h)                                // of the fused price + selection launch
{
    switch (fmt_of(h->Dt)) {
    case 0: return price_grid<true, FMT_WIDE, false>(h);
    case 1: return price_grid<true, FMT_NARROW, false>(h);
    default: return price_grid<true, FMT_NARROW_1BASE, false>(h);
    }
}
template <bool SELECT, int FMT, bool SKIP>
static void launch_k_price_fmt(const vmat_ddc *h, const float *g, float *p, const SelectArgs &sa, cudaStream_t st)
{
    k_price<SELECT, FMT, SKIP><<<price_grid<SELECT, FMT, SKIP>(h), PRICE_THREADS, 0, st>>>(
        h->Dt.pptr, view_of(h->Dt), h->n_beamlets, g, p, sa, h->queues_price());
}
template <bool SELECT, bool SKIP = false>
static void launch_k_price(const vmat_ddc *h, const float *g, float *p, const SelectArgs &sa, cudaStream_t st)
{
    switch (fmt_of(h->Dt)) {
    case 0: launch_k_price_fmt<SELECT, FMT_WIDE, SKIP>(h, g, p, sa, st); break;
    case 1: launch_k_price_fmt<SELECT, FMT_NARROW, SKIP>(h, g, p, sa, st); break;
    default: launch_k_price_fmt<SELECT, FMT_NARROW_1BASE, SKIP>(h, g, p, sa, st); break;
    }
}

int vmat_launch_price(const vmat_ddc *h, const float *g, float *p, cudaStream_t st)
{
    if (h->n_beamlets == 0) return VMAT_OK;
    launch_k_price<false>(h, g, p, SelectArgs{}, st);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

int vmat_launch_select(const vmat_ddc *h, const float *p, const uint8_t *angle_mask, int32_t *L, int32_t *R,
                       double *row_price, cudaStream_t st)
{
    if (h->n_leaf_rows == 0) return VMAT_OK;
    k_select<<<h->n_leaf_rows, PRICE_THREADS, 0, st>>>(p, h->leafrow_col_offset, h->leafrow_angle, angle_mask,
                                                       h->S_scratch, L, R, row_price);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

// Prices of the unoccupied control points only (angle_mask != NULL): the others' rows are not read, their p is 0.
int vmat_launch_price_unoccupied(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p, cudaStream_t st)
{
    if (h->n_beamlets == 0) return VMAT_OK;
    SelectArgs sa{};
    sa.beamlet_leafrow = h->beamlet_leafrow; sa.leafrow_angle = h->leafrow_angle; sa.angle_mask = angle_mask;
    launch_k_price<false, true>(h, g, p, sa, st);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

int vmat_launch_price_select(const vmat_ddc *h, const float *g, const uint8_t *angle_mask, float *p,
                             int32_t *L, int32_t *R, double *row_price, cudaStream_t st, bool skip_occupied)
{
    if (h->n_leaf_rows == 0) return VMAT_OK;
    if (h->n_beamlets == 0) {                       // nothing to price: the selection kernel closes every row
        int rc = vmat_launch_price(h, g, p, st);
        return rc != VMAT_OK ? rc : vmat_launch_select(h, p, angle_mask, L, R, row_price, st);
    }
    SelectArgs sa{h->beamlet_leafrow, h->leafrow_col_offset, h->leafrow_angle, angle_mask, h->leafrow_done,
                  h->S_scratch, L, R, row_price, h->n_leaf_rows};
    if (skip_occupied && angle_mask != nullptr) launch_k_price<true, true>(h, g, p, sa, st);
    else launch_k_price<true>(h, g, p, sa, st);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

int vmat_launch_angle_price(const vmat_ddc *h, const double *row_price, const uint8_t *angle_mask,
                            double *angle_price, int32_t *best_angle, cudaStream_t st)
{
    const int grid = h->n_angles > 0 ? (h->n_angles + ANGLE_THREADS / 32 - 1) / (ANGLE_THREADS / 32) : 1;
    k_angle_price<<<grid, ANGLE_THREADS, 0, st>>>(h->n_angles, h->angle_row_offset, row_price, angle_mask,
                                                  angle_price, best_angle, h->angle_ticket);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}
