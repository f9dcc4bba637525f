/*
 * vmat_oracle.c - plain, slow, obviously-correct CPU oracle (FP64) for the beamlet-price
 * step of the column-generation VMAT optimiser of arXiv 1503.01721.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with the CUDA library (paper_1503_01721_b200/csrc) and never sees a value
 * the CUDA path produced, except where a test deliberately feeds it the GPU's own FP32 price
 * vector to check the selection protocol (reading C6).
 *
 * The method reaches exactly (up to rounding order) results that have plain definitions, so
 * the oracle is those definitions written out over the COO triplets in input order: no CSR,
 * no blocking, no reordering.
 *
 *   O1  dose        d_i = sum_j D_ij x_j                          PAPER.md L43  (z = sum DA y)
 *   O2  objective   F = sum_i w+_i max(0,d_i-T_i)^2 + w-_i max(0,T_i-d_i)^2   Eq.(1)
 *       gradient    g_i = dF/dd_i = 2 w+_i max(0,d_i-T_i) - 2 w-_i max(0,T_i-d_i)
 *                   (the paper's g is -grad F, Eq.(4); sign reading C1: we keep +grad and
 *                    MINIMISE, pi = -p, identical selections)
 *   O3  price       p_j = sum_i D_ij g_i                          Eq.(3), "Pi = D^T g" L121
 *   O4  row opening per MLC leaf row, the contiguous opening [L,R) with the best (minimum)
 *                   summed price, by exhaustive enumeration       L133
 *   O5  aperture    price of the best aperture of each control point = sum of its rows'
 *                   best prices; the control point with the best price is chosen   L133
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): column reproduction, adjoint identity,
 * finite differences, closed forms for 1x1, the paper's first iteration (z=0, L56), scipy.sparse
 * products, O(n^3) direct enumeration, hand-worked rows in tests/golden/.  O4/O5 have no example
 * printed in the paper: pinned by brute force and invariants only.
 */
#include <stdint.h>
#include <stddef.h>
#include <math.h>

/* O1: d = D x.  COO in any order; d is overwritten. */
void oracle_dose(int64_t nnz, const int32_t *coo_voxel, const int32_t *coo_beamlet,
                 const float *coo_val, int32_t n_voxels, const float *x, double *d)
{
    for (int32_t i = 0; i < n_voxels; ++i) d[i] = 0.0;
    for (int64_t e = 0; e < nnz; ++e)
        d[coo_voxel[e]] += (double)coo_val[e] * (double)x[coo_beamlet[e]];
}

/* O2 (Eq. (1), Eq. (4) L63 with sign reading C1; factor 2 kept, C2).
 * Per-voxel structure id -> per-structure {T, w_over (omega+), w_under (omega-)} (C9, C10).
 * Returns F; g is overwritten. */
double oracle_objective_grad(int32_t n_voxels, const double *d, const uint8_t *voxel_struct,
                             const float *T, const float *w_over, const float *w_under, double *g)
{
    double F = 0.0;
    for (int32_t i = 0; i < n_voxels; ++i) {
        int s = voxel_struct[i];
        double over = d[i] - (double)T[s];
        double under = (double)T[s] - d[i];
        if (over < 0.0) over = 0.0;
        if (under < 0.0) under = 0.0;
        F += (double)w_over[s] * over * over + (double)w_under[s] * under * under;
        g[i] = 2.0 * (double)w_over[s] * over - 2.0 * (double)w_under[s] * under;
    }
    return F;
}

/* O3 (Eq. (3)): p = D^T g.  Second pass over the same COO triplets. */
void oracle_price(int64_t nnz, const int32_t *coo_voxel, const int32_t *coo_beamlet,
                  const float *coo_val, int32_t n_beamlets, const double *g, double *p)
{
    for (int32_t j = 0; j < n_beamlets; ++j) p[j] = 0.0;
    for (int64_t e = 0; e < nnz; ++e)
        p[coo_beamlet[e]] += (double)coo_val[e] * g[coo_voxel[e]];
}

/* O4 (L133, readings C4-C6, C8).  The selection is a function of an FP32 price vector.
 * For the leaf row holding beamlets j0 .. j0+n-1 (left -> right):
 *   S_0 = 0, S_{c+1} = S_c + (double)p[j0+c]   strictly left to right;
 *   every pair 0 <= L <= R <= n is a candidate with value V(L,R) = S_R - S_L
 *   (all closed openings L == R have V = 0);
 *   the result is the candidate that is smallest in the order (V, L, R): minimum value,
 *   ties -> smallest L, then smallest R.  At V = 0 that is the closed opening (0,0).
 * S is caller scratch of max_n+1 doubles. */
void oracle_select_rows(int32_t n_rows, const int32_t *leafrow_col_offset, const float *p,
                        int32_t *Lout, int32_t *Rout, double *row_price, double *S)
{
    for (int32_t r = 0; r < n_rows; ++r) {
        int32_t j0 = leafrow_col_offset[r];
        int32_t n = leafrow_col_offset[r + 1] - j0;
        S[0] = 0.0;
        for (int32_t c = 0; c < n; ++c) S[c + 1] = S[c] + (double)p[j0 + c];
        double bestV = 0.0;
        int32_t bestL = 0, bestR = 0;
        for (int32_t L = 0; L <= n; ++L)
            for (int32_t R = L; R <= n; ++R) {
                double V = S[R] - S[L];
                if (V < bestV) { bestV = V; bestL = L; bestR = R; }   /* strict: first in (L,R) order wins ties */
            }
        Lout[r] = bestL; Rout[r] = bestR; row_price[r] = bestV;
    }
}

/* O5 (L133; readings C7).  angle_price[a] = sum of the row prices of control point a, in row
 * order; occupied control points (angle_mask[a] != 0) are skipped: price +inf, and the caller
 * is expected to have closed their rows.  best = smallest a with the minimum price among the
 * unoccupied ones; if that minimum is >= 0 no aperture improves F (L56) and best = -1. */
int32_t oracle_angle_price(int32_t n_angles, const int32_t *angle_row_offset,
                           const double *row_price, const uint8_t *angle_mask, double *angle_price)
{
    int32_t best = -1;
    double bestV = 0.0;
    for (int32_t a = 0; a < n_angles; ++a) {
        if (angle_mask && angle_mask[a]) { angle_price[a] = INFINITY; continue; }
        double s = 0.0;
        for (int32_t r = angle_row_offset[a]; r < angle_row_offset[a + 1]; ++r) s += row_price[r];
        angle_price[a] = s;
        if (s < bestV) { bestV = s; best = a; }
    }
    return best;
}
