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
 *
 *   O6  constrained aperture selection (interdigitation L135, leaf windows L66), at the end of this file;
 *       pins in tests/test_constrained_selection_oracle.py: hand-worked control points, exhaustive enumeration of
 *       all combinations, reduction to O4/O5.  No example is printed in the paper either ("parity unpinned" by
 *       publication).
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

/* ------------------------------------------------------------------------------------------------
 * O6 (NEXT-3) aperture selection under MLC hardware constraints, PAPER.md L133-L135 and L66:
 *   "When there is an interdigitation constraint of MLC leaves in adjacent rows, that is,
 *    L_{k,irow} <= min{R_{k,irow-1}, R_{k,irow+1}}, the MLC rows are not independent any longer ...
 *    each thread would be responsible for one control point and for calculating the prices of all the
 *    combinations of openings at different MLC rows that can satisfy the interdigitation constraint.
 *    It would then choose the best aperture for that control point."                       (L135)
 *   "the candidate apertures need to be compatible with those chosen apertures" (neighbouring
 *    control points, L66): here per-row windows on the two leaf positions.
 * Readings C22-C24 of DESIGN.md:
 *   - A leaf row r of a control point has a state (a, b), a <= b: the physical positions of its left
 *     and right leaf ends in beamlet widths on the control point's grid; row-local L = a - pos0[r],
 *     R = b - pos0[r] (pos0 = physical column of the row's first beamlet).  Open states a < b need
 *     pos0 <= a and b <= pos0 + n (they expose beamlets L .. R-1 of the row); a closed pair a == b
 *     may be parked at any position of the control point's field range [Pmin, Pmax] = [min pos0,
 *     max pos0 + n] over its non-empty rows (0, 0 when it has none).  The formula of L135 applies to
 *     every row, closed ones included.
 *   - Windows (each array may be NULL): L_lo[r] <= L <= L_hi[r], R_lo[r] <= R <= R_hi[r], row-local.
 *   - Value of a state: V = S_R - S_L for an open one (S as in O4: FP64 prefix sums of the FP32
 *     prices, left to right), 0 for a closed one.
 *   - Interdigitation between adjacent rows r, r+1 of one control point: a_r <= b_{r+1} and
 *     a_{r+1} <= b_r (L135 written for both rows of the pair).
 *   - The aperture price is f_last with f_0 = V_0, f_r = V_r + min over compatible states s of row
 *     r-1 of f_{r-1}(s): the exhaustive minimum over all combinations, organised row by row.
 *   - Ties: the last row takes its smallest optimal state in the order (a, b); every earlier row
 *     the smallest state, in the same order, among those attaining the minimum it feeds.
 *   - A control point with no feasible combination: price +inf, rows L = R = 0, row prices 0.
 * Returns the best control point as O5 does.  O(states^2) per row pair: the plain recursion, no
 * prefix-minimum tables. */
#include <stdlib.h>

int32_t oracle_select_constrained(int32_t n_angles, const int32_t *angle_row_offset,
                                  const int32_t *leafrow_col_offset, const int32_t *pos0, const float *p,
                                  const uint8_t *angle_mask, int32_t interdigitation,
                                  const int32_t *L_lo, const int32_t *L_hi, const int32_t *R_lo,
                                  const int32_t *R_hi, int32_t *Lout, int32_t *Rout, double *row_price,
                                  double *angle_price)
{
    int32_t best_angle = -1;
    double best_price = 0.0;
    for (int32_t k = 0; k < n_angles; ++k) {
        const int32_t r0 = angle_row_offset[k], r1 = angle_row_offset[k + 1], nr = r1 - r0;
        for (int32_t r = r0; r < r1; ++r) { Lout[r] = 0; Rout[r] = 0; row_price[r] = 0.0; }
        if (angle_mask && angle_mask[k]) { angle_price[k] = INFINITY; continue; }
        if (nr == 0) { angle_price[k] = 0.0; continue; }
        /* field range of the control point */
        int32_t Pmin = 0, Pmax = 0, any = 0, nmax = 0;
        for (int32_t r = r0; r < r1; ++r) {
            const int32_t n = leafrow_col_offset[r + 1] - leafrow_col_offset[r];
            if (n <= 0) continue;
            if (!any || pos0[r] < Pmin) Pmin = pos0[r];
            if (!any || pos0[r] + n > Pmax) Pmax = pos0[r] + n;
            if (n > nmax) nmax = n;
            any = 1;
        }
        const int32_t Wd = Pmax - Pmin + 1;
        const size_t cap = (size_t)Wd * (Wd + 1) / 2;                    /* states per row at most */
        int32_t *sa = (int32_t *)malloc(sizeof(int32_t) * cap * nr), *sb = (int32_t *)malloc(sizeof(int32_t) * cap * nr);
        int32_t *arg = (int32_t *)malloc(sizeof(int32_t) * cap * nr), *cnt = (int32_t *)malloc(sizeof(int32_t) * nr);
        double *V = (double *)malloc(sizeof(double) * cap * nr), *f = (double *)malloc(sizeof(double) * cap * nr);
        double *S = (double *)malloc(sizeof(double) * (nmax + 1));
        int feasible = 1;
        for (int32_t q = 0; q < nr && feasible; ++q) {
            const int32_t r = r0 + q, j0 = leafrow_col_offset[r], n = leafrow_col_offset[r + 1] - j0;
            const int32_t u0 = n > 0 ? pos0[r] : Pmin;                    /* empty rows: row-local = offset from Pmin */
            S[0] = 0.0;
            for (int32_t c = 0; c < n; ++c) S[c + 1] = S[c] + (double)p[j0 + c];
            int32_t m = 0;
            for (int32_t a = Pmin; a <= Pmax; ++a)
                for (int32_t b = a; b <= Pmax; ++b) {
                    const int32_t L = a - u0, R = b - u0;
                    if (a < b && !(n > 0 && L >= 0 && R <= n)) continue;  /* an open state exposes existing beamlets */
                    if (L_lo && L < L_lo[r]) continue;
                    if (L_hi && L > L_hi[r]) continue;
                    if (R_lo && R < R_lo[r]) continue;
                    if (R_hi && R > R_hi[r]) continue;
                    sa[q * cap + m] = a; sb[q * cap + m] = b;
                    V[q * cap + m] = a < b ? S[R] - S[L] : 0.0;
                    ++m;
                }
            cnt[q] = m;
            /* the recursion */
            for (int32_t t = 0; t < m; ++t) {
                if (q == 0) { f[t] = V[t]; arg[t] = -1; continue; }
                double bestf = INFINITY;
                int32_t bests = -1;
                for (int32_t s = 0; s < cnt[q - 1]; ++s) {
                    const double fs = f[(q - 1) * cap + s];
                    if (interdigitation) {
                        if (sa[(q - 1) * cap + s] > sb[q * cap + t]) continue;       /* a_{r-1} <= b_r  */
                        if (sa[q * cap + t] > sb[(q - 1) * cap + s]) continue;       /* a_r <= b_{r-1}  */
                    }
                    if (fs < bestf) { bestf = fs; bests = s; }                       /* strict: first in (a,b) order */
                }
                f[q * cap + t] = bests >= 0 ? V[q * cap + t] + bestf : INFINITY;
                arg[q * cap + t] = bests;
            }
            int ok = 0;
            for (int32_t t = 0; t < m; ++t) ok |= f[q * cap + t] < INFINITY;
            if (!ok) feasible = 0;
        }
        if (!feasible) angle_price[k] = INFINITY;
        else {
            int32_t t = -1;
            double bf = INFINITY;
            for (int32_t s = 0; s < cnt[nr - 1]; ++s)
                if (f[(nr - 1) * cap + s] < bf) { bf = f[(nr - 1) * cap + s]; t = s; }
            angle_price[k] = bf;
            for (int32_t q = nr - 1; q >= 0; --q) {
                const int32_t r = r0 + q, n = leafrow_col_offset[r + 1] - leafrow_col_offset[r];
                const int32_t u0 = n > 0 ? pos0[r] : Pmin;
                Lout[r] = sa[q * cap + t] - u0; Rout[r] = sb[q * cap + t] - u0; row_price[r] = V[q * cap + t];
                t = arg[q * cap + t];
            }
            if (bf < best_price) { best_price = bf; best_angle = k; }
        }
        free(sa); free(sb); free(arg); free(cnt); free(V); free(f); free(S);
    }
    return best_angle;
}
