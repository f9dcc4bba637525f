// constrained.cu - NEXT-3: aperture selection under MLC hardware constraints.
//
//   "When there is an interdigitation constraint of MLC leaves in adjacent rows, that is, L_{k,irow} <=
//    min{R_{k,irow-1}, R_{k,irow+1}}, the MLC rows are not independent any longer ... each thread would be
//    responsible for one control point and for calculating the prices of all the combinations of openings at
//    different MLC rows that can satisfy the interdigitation constraint."  (L135)
//
// The paper enumerates the combinations with one thread per control point.  Here one CTA owns a control point
// and walks its leaf rows once: f_r(a,b) = V_r(a,b) + min{ f_{r-1}(a',b') : a' <= b, a <= b' } is the exact
// minimum over all compatible combinations of rows 0..r ending in state (a,b) (readings C22-C24).
// The inner minimum is a 2-D dominance query, answered for every (a,b) at once by a prefix-minimum table
//   M_r[x][y] = min{ f_r(a',b') : a' <= x, b' >= y }      (so the query above is M_{r-1}[b][a]),
// built in shared memory by two sweeps (down the columns, then right-to-left along the rows).  The table holds
// Wd x Wd doubles, Wd = positions of the control point's field range; minima carry their arg (a',b') packed in
// 16 bits, smaller packed value = smaller (a',b') in lexicographic order = the oracle's tie rule.  The arg tables
// go to global memory row by row and are walked backwards by one thread at the end.
// Every value is produced by the oracle's operations in the oracle's order (S_R - S_L, then V + minimum; minima
// are exact), so leaf positions, row prices and aperture prices are bit-identical to oracle_select_constrained
// applied to the same FP32 price vector.
#include "common.cuh"

constexpr int CS_THREADS = 256;
constexpr int CS_MAX_POS = 255;                       // positions are packed in 8 bits each

__device__ __forceinline__ double cs_inf() { return __longlong_as_double(0x7ff0000000000000LL); }

// FP64 prefix sums of every leaf row, left to right (C6): S[j0 + r + c], c = 0 .. n.  One thread per leaf row.
__global__ void k_cs_prefix(int n_rows, const int32_t *__restrict__ leafrow_col_offset, const float *__restrict__ p,
                            double *__restrict__ S)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const int j0 = leafrow_col_offset[r], n = leafrow_col_offset[r + 1] - j0;
    double *s = S + j0 + r;
    double acc = 0.0;
    s[0] = 0.0;
    for (int c = 0; c < n; ++c) { acc += (double)p[j0 + c]; s[c + 1] = acc; }
}

struct CsArgs {
    const int32_t *angle_row_offset, *leafrow_col_offset, *pos0, *angle_pmin, *angle_wd;
    const int64_t *angle_bp_offset;
    const uint8_t *angle_mask;
    const int32_t *L_lo, *L_hi, *R_lo, *R_hi;         // each may be NULL
    const double *S;
    uint16_t *bp;
    int32_t *L, *R;
    double *row_price, *angle_price;
    int interdigitation;
};

__device__ __forceinline__ int cs_stride_d(int wd) { return wd | 1; }                 // doubles per table row: odd
__device__ __forceinline__ int cs_stride_a(int wd)                                  // u16 per arg row: 2 * odd
{
    int s = (wd + 1) & ~1;
    return ((s >> 1) & 1) ? s : s + 2;
}

__global__ void __launch_bounds__(CS_THREADS)
k_cs_dp(CsArgs A)
{
    extern __shared__ __align__(16) unsigned char cs_smem[];
    const int k = blockIdx.x;
    const int r0 = A.angle_row_offset[k], r1 = A.angle_row_offset[k + 1], nr = r1 - r0;
    const bool masked = A.angle_mask != nullptr && A.angle_mask[k] != 0;
    if (masked || nr == 0) {                                                          // C7: occupied control point
        for (int r = r0 + threadIdx.x; r < r1; r += CS_THREADS) { A.L[r] = 0; A.R[r] = 0; A.row_price[r] = 0.0; }
        if (threadIdx.x == 0) A.angle_price[k] = masked ? cs_inf() : 0.0;
        return;
    }
    const int pmin = A.angle_pmin[k], wd = A.angle_wd[k];
    const int SD = cs_stride_d(wd), SA = cs_stride_a(wd);
    double *T = (double *)cs_smem;                                                    // [wd][SD]
    uint16_t *G = (uint16_t *)(T + (size_t)wd * SD);                                  // [wd][SA]
    __shared__ double s_gmin;
    uint16_t *bp_k = A.bp + A.angle_bp_offset[k];
    const size_t bp_row = A.interdigitation ? (size_t)wd * wd : 1;                    // u16 stored per leaf row
    const int cells = wd * wd;
    for (int q = 0; q < nr; ++q) {
        const int r = r0 + q;
        const int j0 = A.leafrow_col_offset[r], n = A.leafrow_col_offset[r + 1] - j0;
        const int off = n > 0 ? A.pos0[r] - pmin : 0;                                 // table position of row-local 0
        const int llo = A.L_lo ? A.L_lo[r] : INT_MIN, lhi = A.L_hi ? A.L_hi[r] : INT_MAX;
        const int rlo = A.R_lo ? A.R_lo[r] : INT_MIN, rhi = A.R_hi ? A.R_hi[r] : INT_MAX;
        const double *S = A.S + j0 + r;
        if (q > 0 && threadIdx.x == 0) s_gmin = T[(size_t)(wd - 1) * SD];             // M[wd-1][0]: the row's minimum
        __syncthreads();
        // ---- f_q(a,b) for a <= b: reads M_{q-1}[b][a] (on or below the diagonal), writes on or above it
        for (int e = threadIdx.x; e < cells; e += CS_THREADS) {
            const int a = e / wd, b = e - a * wd;
            if (a > b) continue;
            const int L = a - off, R = b - off;
            bool ok = L >= llo && L <= lhi && R >= rlo && R <= rhi;
            if (a < b) ok = ok && n > 0 && L >= 0 && R <= n;                          // an open state exposes existing beamlets
            double f = cs_inf();
            if (ok) {
                const double V = a < b ? S[R] - S[L] : 0.0;
                if (q == 0) f = V;
                else {
                    const double m = A.interdigitation ? T[(size_t)b * SD + a] : s_gmin;
                    f = V + m;                                                        // +inf when no compatible predecessor
                }
            }
            T[(size_t)a * SD + b] = f;
            G[(size_t)a * SA + b] = (uint16_t)((a << 8) | b);
        }
        __syncthreads();
        for (int e = threadIdx.x; e < cells; e += CS_THREADS) {                       // no states below the diagonal
            const int a = e / wd, b = e - a * wd;
            if (a > b) { T[(size_t)a * SD + b] = cs_inf(); G[(size_t)a * SA + b] = 0xffffu; }
        }
        __syncthreads();
        // ---- sweep 1: down every column b: min over a' <= a (ascending a: strict < keeps the smaller arg)
        if (threadIdx.x < wd) {
            const int b = threadIdx.x;
            double v = cs_inf();
            uint16_t g = 0xffffu;
            for (int a = 0; a < wd; ++a) {
                const double c = T[(size_t)a * SD + b];
                if (c < v) { v = c; g = G[(size_t)a * SA + b]; }
                T[(size_t)a * SD + b] = v;
                G[(size_t)a * SA + b] = g;
            }
        }
        __syncthreads();
        // ---- sweep 2: along every row a from the right: min over b' >= b; ties -> smaller packed arg
        if (threadIdx.x < wd) {
            const int a = threadIdx.x;
            double v = cs_inf();
            uint16_t g = 0xffffu;
            for (int b = wd - 1; b >= 0; --b) {
                const double c = T[(size_t)a * SD + b];
                const uint16_t cg = G[(size_t)a * SA + b];
                if (c < v || (c == v && cg < g)) { v = c; g = cg; }
                T[(size_t)a * SD + b] = v;
                G[(size_t)a * SA + b] = g;
            }
        }
        __syncthreads();
        // ---- the arg table of this row goes to global memory for the walk back
        uint16_t *dst = bp_k + (size_t)q * bp_row;
        if (A.interdigitation) {
            for (int e = threadIdx.x; e < cells; e += CS_THREADS) {
                const int x = e / wd, y = e - x * wd;
                dst[e] = G[(size_t)x * SA + y];
            }
        } else if (threadIdx.x == 0) dst[0] = G[(size_t)(wd - 1) * SA];
    }
    __syncthreads();                                                                  // the stores above are visible to thread 0
    if (threadIdx.x != 0) return;
    const double total = T[(size_t)(wd - 1) * SD];
    if (!(total < cs_inf())) {                                                        // no feasible combination
        for (int r = r0; r < r1; ++r) { A.L[r] = 0; A.R[r] = 0; A.row_price[r] = 0.0; }
        A.angle_price[k] = cs_inf();
        return;
    }
    A.angle_price[k] = total;
    int g = G[(size_t)(wd - 1) * SA];
    for (int q = nr - 1; q >= 0; --q) {
        const int r = r0 + q, a = g >> 8, b = g & 255;
        const int j0 = A.leafrow_col_offset[r], n = A.leafrow_col_offset[r + 1] - j0;
        const int off = n > 0 ? A.pos0[r] - pmin : 0;
        const double *S = A.S + j0 + r;
        A.L[r] = a - off;
        A.R[r] = b - off;
        A.row_price[r] = a < b ? S[b - off] - S[a - off] : 0.0;
        if (q > 0) {
            const uint16_t *src = bp_k + (size_t)(q - 1) * bp_row;
            g = A.interdigitation ? src[(size_t)b * wd + a] : src[0];
        }
    }
}

// best control point: smallest price, ties -> smallest index, none below 0 -> -1 (L56).  One CTA.
__global__ void __launch_bounds__(CS_THREADS)
k_cs_best(int n_angles, const double *__restrict__ angle_price, int32_t *__restrict__ best_angle)
{
    __shared__ double bv[CS_THREADS];
    __shared__ int bi[CS_THREADS];
    double best = 0.0;
    int besta = -1;
    for (int k = threadIdx.x; k < n_angles; k += CS_THREADS) {
        const double v = angle_price[k];
        if (v < best) { best = v; besta = k; }
    }
    bv[threadIdx.x] = best; bi[threadIdx.x] = besta;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < CS_THREADS; ++i)
            if (bi[i] >= 0 && (besta < 0 || bv[i] < best || (bv[i] == best && bi[i] < besta))) { best = bv[i]; besta = bi[i]; }
        best_angle[0] = besta;
    }
}

static size_t cs_smem_bytes(int wd)
{
    const int SD = wd | 1;
    int SA = (wd + 1) & ~1;
    if (!((SA >> 1) & 1)) SA += 2;
    return (size_t)wd * SD * 8 + (size_t)wd * SA * 2;
}

#define REQUIRE(cond, msg)                                            \
    do {                                                              \
        if (!(cond)) { vmat_set_error("%s: %s", __func__, msg); return VMAT_ERR_INVALID_ARG; } \
    } while (0)

int vmat_launch_select_constrained(vmat_ddc *h, const float *p, const uint8_t *angle_mask, int interdigitation,
                                   const int32_t *L_lo, const int32_t *L_hi, const int32_t *R_lo, const int32_t *R_hi,
                                   int32_t *L, int32_t *R, double *row_price, double *angle_price, int32_t *best_angle,
                                   cudaStream_t st)
{
    REQUIRE(h->leafrow_pos0 != nullptr, "call vmat_ddc_set_leaf_geometry first");
    // back-pointer tables: wd^2 u16 per leaf row with interdigitation, one u16 without
    const int64_t need = interdigitation ? h->cs_bp_elems : (int64_t)h->n_leaf_rows + 1;
    if (need > h->cs_bp_alloc) {
        if (h->cs_bp) { VMAT_CUDA(cudaStreamSynchronize(st)); cudaFree(h->cs_bp); h->cs_bp = nullptr; h->cs_bp_alloc = 0; }
        VMAT_CUDA(cudaMalloc((void **)&h->cs_bp, (size_t)need * 2));
        h->cs_bp_alloc = need;
    }
    if (h->n_leaf_rows > 0) {
        k_cs_prefix<<<(h->n_leaf_rows + 127) / 128, 128, 0, st>>>(h->n_leaf_rows, h->leafrow_col_offset, p, h->S_scratch);
        VMAT_LAUNCH_CHECK();
    }
    if (h->n_angles > 0) {
        CsArgs A{h->angle_row_offset, h->leafrow_col_offset, h->leafrow_pos0, h->angle_pmin, h->angle_wd,
                 h->angle_bp_offset, angle_mask, L_lo, L_hi, R_lo, R_hi, h->S_scratch, h->cs_bp, L, R, row_price,
                 angle_price, interdigitation ? 1 : 0};
        k_cs_dp<<<h->n_angles, CS_THREADS, cs_smem_bytes(h->cs_max_wd), st>>>(A);
        VMAT_LAUNCH_CHECK();
    }
    k_cs_best<<<1, CS_THREADS, 0, st>>>(h->n_angles, angle_price, best_angle);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

extern "C" {

int vmat_ddc_set_leaf_geometry(vmat_ddc *h, const int32_t *leafrow_pos0)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(leafrow_pos0 != nullptr || h->n_leaf_rows == 0, "leafrow_pos0 is NULL");
    const int n_rows = h->n_leaf_rows, n_a = h->n_angles;
    std::vector<int32_t> lco((size_t)n_rows + 1, 0);
    VMAT_CUDA(cudaMemcpy(lco.data(), h->leafrow_col_offset, ((size_t)n_rows + 1) * 4, cudaMemcpyDeviceToHost));
    std::vector<int32_t> pmin((size_t)(n_a > 0 ? n_a : 1), 0), wd((size_t)(n_a > 0 ? n_a : 1), 1);
    std::vector<int64_t> bpo((size_t)n_a + 1, 0);
    int max_wd = 1;
    for (int k = 0; k < n_a; ++k) {
        bool any = false;
        int lo = 0, hi = 0;
        for (int r = h->h_angle_row_offset[k]; r < h->h_angle_row_offset[k + 1]; ++r) {
            const int n = lco[r + 1] - lco[r];
            if (n <= 0) continue;
            const int64_t e = (int64_t)leafrow_pos0[r] + n;
            REQUIRE(e <= INT32_MAX, "leaf row position overflows int32");
            if (!any || leafrow_pos0[r] < lo) lo = leafrow_pos0[r];
            if (!any || (int)e > hi) hi = (int)e;
            any = true;
        }
        REQUIRE((int64_t)hi - lo + 1 <= CS_MAX_POS + 1,
                "a control point's field range exceeds 255 beamlet widths (positions are packed in 8 bits)");
        pmin[k] = lo;
        wd[k] = hi - lo + 1;
        max_wd = wd[k] > max_wd ? wd[k] : max_wd;
        bpo[k + 1] = bpo[k] + (int64_t)wd[k] * wd[k] * (h->h_angle_row_offset[k + 1] - h->h_angle_row_offset[k]);
    }
    int smem_optin = 0;
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    if (smem_optin > 0 && cs_smem_bytes(max_wd) > (size_t)smem_optin) {
        vmat_set_error("vmat_ddc_set_leaf_geometry: a field range of %d positions needs %zu bytes of shared memory (%d available)",
                       max_wd, cs_smem_bytes(max_wd), smem_optin);
        return VMAT_ERR_INVALID_ARG;
    }
    VMAT_CUDA(cudaFuncSetAttribute(k_cs_dp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cs_smem_bytes(max_wd)));
    for (void **q : {(void **)&h->leafrow_pos0, (void **)&h->angle_pmin, (void **)&h->angle_wd, (void **)&h->angle_bp_offset})
        if (*q) { cudaFree(*q); *q = nullptr; }
    auto up = [&](void **dst, const void *src, size_t bytes) -> int {
        VMAT_CUDA(cudaMalloc(dst, bytes > 0 ? bytes : 1));
        if (bytes > 0) VMAT_CUDA(cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
        return VMAT_OK;
    };
    int rc = up((void **)&h->leafrow_pos0, leafrow_pos0, (size_t)n_rows * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_pmin, pmin.data(), (size_t)n_a * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_wd, wd.data(), (size_t)n_a * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_bp_offset, bpo.data(), ((size_t)n_a + 1) * 8);
    if (rc != VMAT_OK) return rc;
    h->cs_bp_elems = bpo[n_a] > 0 ? bpo[n_a] : 1;
    h->cs_max_wd = max_wd;
    h->h_leafrow_pos0.assign(leafrow_pos0, leafrow_pos0 + n_rows);
    return VMAT_OK;
}

int vmat_select_apertures_constrained(vmat_ddc *h, const float *p, const uint8_t *angle_mask, int32_t interdigitation,
                                      const int32_t *L_lo, const int32_t *L_hi, const int32_t *R_lo,
                                      const int32_t *R_hi, int32_t *L, int32_t *R, double *row_price,
                                      double *angle_price, int32_t *best_angle, void *stream)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(p != nullptr || h->n_beamlets == 0, "p is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L && R && row_price), "NULL leaf-row output");
    REQUIRE((angle_price || h->n_angles == 0) && best_angle, "NULL control-point output");
    g_vmat_launches = 0;
    return vmat_launch_select_constrained(h, p, angle_mask, interdigitation, L_lo, L_hi, R_lo, R_hi, L, R, row_price,
                                          angle_price, best_angle, (cudaStream_t)stream);
}

}  // extern "C"
