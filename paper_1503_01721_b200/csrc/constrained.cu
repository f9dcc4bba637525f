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
// The inner minimum is a 2-D dominance query.  The states of a row are its closed pairs (c,c), c anywhere in
// the control point's field range (wd positions), and its open states inside its own n beamlets, so the query
// splits into
//   - a range minimum of the previous row's closed values over c in [a, b], carried along as b grows, and
//   - a look-up in the prefix-minimum table PB[I][J] = min{ f(i,j) : i <= I, j >= J, i < j } of the previous
//     row's open states (row-local i, j), built in shared memory by two sweeps of n+1 steps.
// Work per row is O(n^2 + wd) instead of the O(wd^2) of a table over the whole field range (the first version of
// this kernel: 10.4 ms per call on config 3, where rows hold 14 beamlets on average in fields 100-130 wide).
// Minima carry their arg (a',b') packed in 16 bits; a smaller packed value is a smaller (a',b') in lexicographic
// order = the oracle's tie rule.  Every state's predecessor goes to global memory and one thread walks them back.
// Every value is produced by the oracle's operations in the oracle's order (S_R - S_L, then V + minimum; minima
// are exact), so leaf positions, row prices and aperture prices are bit-identical to oracle_select_constrained
// applied to the same FP32 price vector.
#include "common.cuh"
#include <algorithm>

constexpr int CS_THREADS = 256;
constexpr int CS_SMALL_ROW = 64;                      // control points without a longer leaf row use the small table
constexpr int CS_MAX_POS = 255;                       // positions are packed in 8 bits each
constexpr unsigned CS_NONE = 0xffffu;

__device__ __forceinline__ double cs_inf() { return __longlong_as_double(0x7ff0000000000000LL); }

// (v, g) <- the smaller of (v, g) and (c, cg): by value, ties by packed arg
__device__ __forceinline__ void cs_take(double &v, unsigned &g, double c, unsigned cg)
{
    if (c < v || (c == v && cg < g)) { v = c; g = cg; }
}

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
    const int32_t *angle_row_offset, *leafrow_col_offset, *pos0, *angle_pmin, *angle_wd, *angle_order;
    const int64_t *row_bp_offset;
    const uint8_t *angle_mask;
    const int32_t *L_lo, *L_hi, *R_lo, *R_hi;         // each may be NULL
    const double *S;
    uint16_t *bp;
    int32_t *L, *R;
    double *row_price, *angle_price;
    int interdigitation;
    int tab_n, max_wd, max_rows;                      // shared-memory table: tab_n x tab_n entries; fc arrays: max_wd; chain: max_rows
};

static __host__ __device__ __forceinline__ int cs_stride_d(int t) { return t | 1; }   // doubles per table row: odd
static __host__ __device__ __forceinline__ int cs_stride_a(int t)                     // u16 per arg row: 2 * odd
{
    const int s = (t + 1) & ~1;
    return ((s >> 1) & 1) ? s : s + 2;
}

// threads sharing one line (an i of the open-state walk, a column or a row of the sweeps) of a row with n1 = n + 1
// positions: the largest power of two that keeps n1 lines inside the CTA, at most 16
__device__ __forceinline__ int cs_segments(int n1)
{
    int s = 1;
    while (s < 16 && 2 * s * n1 <= CS_THREADS) s <<= 1;
    return s;
}

__global__ void __launch_bounds__(CS_THREADS)
k_cs_dp(CsArgs A)
{
    extern __shared__ __align__(16) unsigned char cs_smem[];
    const int k = A.angle_order[blockIdx.x];                                          // heaviest control points first
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r0 = A.angle_row_offset[k], r1 = A.angle_row_offset[k + 1], nr = r1 - r0;
    const bool masked = A.angle_mask != nullptr && A.angle_mask[k] != 0;
    if (masked || nr == 0) {                                                          // C7: occupied control point
        for (int r = r0 + tid; r < r1; r += CS_THREADS) { A.L[r] = 0; A.R[r] = 0; A.row_price[r] = 0.0; }
        if (tid == 0) A.angle_price[k] = masked ? cs_inf() : 0.0;
        return;
    }
    const int pmin = A.angle_pmin[k], wd = A.angle_wd[k];
    const int SD = cs_stride_d(A.tab_n), SA = cs_stride_a(A.tab_n);
    // PB [tab_n][SD]: on and below the diagonal the prefix minima of the PREVIOUS row's open states (the queries
    // read PB[I][J] with I >= J only); strictly above it the open states of THIS row are written while those
    // queries run - the two regions never meet, so one table serves both rows.
    double *PB = (double *)cs_smem;
    double *fcp = PB + (size_t)A.tab_n * SD;                                          // [max_wd] closed states, previous row
    double *fcn = fcp + A.max_wd;                                                     // [max_wd] closed states, this row
    double *Sa = fcn + A.max_wd;                                                      // [tab_n] prefix sums of this row ...
    double *Sb = Sa + A.tab_n;                                                        // [tab_n] ... and of the next one
    uint16_t *PG = (uint16_t *)(Sb + A.tab_n);                                        // [tab_n][SA] args of PB
    __shared__ double tot_v[CS_THREADS];                                              // chunk totals of the segmented sweeps
    __shared__ unsigned tot_g[CS_THREADS];
    __shared__ double s_gv;                                                           // minimum of the previous row ...
    __shared__ unsigned s_ga;                                                         // ... and its smallest state
    const bool inter = A.interdigitation != 0;
    int np = 0, offp = 0;                                                             // previous row: beamlets, table position of its 0
    {
        const int j0 = A.leafrow_col_offset[r0], n = A.leafrow_col_offset[r0 + 1] - j0;
        for (int t = tid; t <= n; t += CS_THREADS) Sa[t] = A.S[j0 + r0 + t];
    }
    __syncthreads();
    // the tables of a row are fetched two rows ahead and its prefix sums one row ahead, so their latency hides behind
    // the work on the rows before
    struct RowMeta { int j0, n, pos0, llo, lhi, rlo, rhi; int64_t bpo; };
    auto fetch = [&](int r) {
        RowMeta m;
        m.j0 = A.leafrow_col_offset[r];
        m.n = A.leafrow_col_offset[r + 1] - m.j0;
        m.pos0 = A.pos0[r];
        m.llo = A.L_lo ? A.L_lo[r] : INT_MIN; m.lhi = A.L_hi ? A.L_hi[r] : INT_MAX;
        m.rlo = A.R_lo ? A.R_lo[r] : INT_MIN; m.rhi = A.R_hi ? A.R_hi[r] : INT_MAX;
        m.bpo = A.row_bp_offset[r];
        return m;
    };
    RowMeta nxt = fetch(r0), nn = nr > 1 ? fetch(r0 + 1) : nxt;                        // rows q + 1 and q + 2 of the loop below
    for (int q = 0; q < nr; ++q) {
        const int r = r0 + q;
        const RowMeta cur = nxt;
        nxt = nn;
        if (q + 2 < nr) nn = fetch(r + 2);
        double s_ahead = 0.0;                                                         // this thread's prefix sum of the next row: in
        if (q + 1 < nr && tid <= nxt.n) s_ahead = A.S[nxt.j0 + r + 1 + tid];          // flight during this row's work
        const int n = cur.n, n1 = n + 1;
        const int off = n > 0 ? cur.pos0 - pmin : 0;
        const int llo = cur.llo, lhi = cur.lhi, rlo = cur.rlo, rhi = cur.rhi;
        uint16_t *bp_row = A.bp + cur.bpo;
        const bool first = q == 0, last = q == nr - 1;
        const bool query = !first && inter;                                           // predecessors depend on the state
        double gv = 0.0;
        unsigned ga = CS_NONE;
        if (!first && !inter) { gv = s_gv; ga = s_ga; }
        // ---- closed states (c,c), c anywhere in the field range
        for (int c = tid; c < wd; c += CS_THREADS) {
            const int Lc = c - off;
            double f = cs_inf();
            unsigned pg = CS_NONE;
            if (Lc >= llo && Lc <= lhi && Lc >= rlo && Lc <= rhi) {
                if (first) f = 0.0;
                else {
                    double pv = gv;
                    unsigned pa = ga;
                    if (inter) {                                                      // a' <= c <= b'
                        pv = fcp[c]; pa = (unsigned)((c << 8) | c);
                        const int I = c - offp;
                        if (np > 0 && I >= 0 && I <= np) cs_take(pv, pa, PB[(size_t)I * SD + I], PG[(size_t)I * SA + I]);
                    }
                    f = 0.0 + pv;
                    pg = pa;
                }
            }
            fcn[c] = f;
            bp_row[c] = (uint16_t)pg;
        }
        // ---- open states (off+i, off+j), 0 <= i < j <= n.  SEG threads share the j range of one i; each first scans
        //      the previous row's closed states from a up to its first b (the range minimum it would have carried),
        //      then walks its own j's four at a time (loads first)
        const int SEG = cs_segments(n1);
        {
            const int i = tid / SEG, seg = tid - i * SEG;
            const int chunk = i < n ? (n - i + SEG - 1) / SEG : 0;
            const int js = i + 1 + seg * chunk, je = min(n, js + chunk - 1);
            if (i < n && js <= je) {
                const int a = off + i;
                double rv = cs_inf();
                unsigned ra = CS_NONE;
                if (query) {
                    rv = fcp[a]; ra = (unsigned)((a << 8) | a);
                    for (int b = a + 1; b < off + js; ++b) {                          // ascending b: strict < keeps the leftmost
                        const double c = fcp[b];
                        if (c < rv) { rv = c; ra = (unsigned)((b << 8) | b); }
                    }
                }
                const double Si = Sa[i];
                const int J = a - offp, Jc = max(J, 0);
                const bool okL = i >= llo && i <= lhi;
                for (int jb = js; jb <= je; jb += 4) {
                    double cf[4], cS[4], cp[4];
                    unsigned cg[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = min(jb + u, je), b = off + j, I = b - offp;
                        cS[u] = Sa[j];
                        cf[u] = cs_inf(); cp[u] = cs_inf(); cg[u] = CS_NONE;
                        if (query) {
                            cf[u] = fcp[b];
                            if (np > 0 && I >= 0 && J <= np) {                        // a' <= b and b' >= a
                                const int Ic = min(I, np);
                                cp[u] = PB[(size_t)Ic * SD + Jc];
                                cg[u] = PG[(size_t)Ic * SA + Jc];
                            }
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = jb + u, b = off + j;
                        if (j > je) break;
                        if (query && cf[u] < rv) { rv = cf[u]; ra = (unsigned)((b << 8) | b); }
                        double f = cs_inf();
                        unsigned pg = CS_NONE;
                        if (okL && j >= rlo && j <= rhi) {
                            const double V = cS[u] - Si;
                            if (first) f = V;
                            else {
                                double pv = gv;
                                unsigned pa = ga;
                                if (inter) { pv = rv; pa = ra; cs_take(pv, pa, cp[u], cg[u]); }
                                f = V + pv;                                           // +inf when no compatible predecessor
                                pg = pa;
                            }
                        }
                        PB[(size_t)i * SD + j] = f;
                        PG[(size_t)i * SA + j] = (uint16_t)((a << 8) | b);
                        bp_row[wd + j * n1 + i] = (uint16_t)pg;
                    }
                }
            }
        }
        if (!last) {                                                                  // prefix sums of the next row
            if (tid <= nxt.n) Sb[tid] = s_ahead;                                      // n + 1 <= CS_THREADS
        }
        __syncthreads();
        // ---- PB of this row: sweep down the columns, then along the rows from the right.  SEG threads share a line:
        //      each scans its chunk, leaves the chunk's total in shared memory, and after a barrier folds the totals
        //      of the chunks before it into its own entries
        if (n > 0) {
            const int line = tid / SEG, seg = tid - line * SEG;
            const int chunk = (n1 + SEG - 1) / SEG, cs0 = seg * chunk, cs1 = min(n, cs0 + chunk - 1);
            const bool act = line <= n && cs0 <= cs1;
            if (act) {                                                                // column j: min over i' <= i (ascending: strict <)
                const int j = line;
                double v = cs_inf();
                unsigned g = CS_NONE;
                for (int i0 = cs0; i0 <= cs1; i0 += 4) {
                    double c[4];
                    unsigned cg[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int i = min(i0 + u, cs1);
                        const bool st = i < j;                                        // states live strictly above the diagonal
                        c[u] = st ? PB[(size_t)i * SD + j] : cs_inf();
                        cg[u] = st ? PG[(size_t)i * SA + j] : CS_NONE;
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int i = i0 + u;
                        if (i <= cs1) {
                            if (c[u] < v) { v = c[u]; g = cg[u]; }
                            PB[(size_t)i * SD + j] = v;
                            PG[(size_t)i * SA + j] = (uint16_t)g;
                        }
                    }
                }
                if (SEG > 1) { tot_v[tid] = v; tot_g[tid] = g; }
            }
            __syncthreads();
            if (SEG > 1) {
                if (act && seg > 0) {
                    const int j = line;
                    double cv = cs_inf();
                    unsigned cgc = CS_NONE;
                    for (int t = 0; t < seg; ++t)                                     // earlier chunks hold smaller i: they win ties
                        if (tot_v[tid - seg + t] < cv) { cv = tot_v[tid - seg + t]; cgc = tot_g[tid - seg + t]; }
                    for (int i = cs0; i <= cs1; ++i)
                        if (!(PB[(size_t)i * SD + j] < cv)) { PB[(size_t)i * SD + j] = cv; PG[(size_t)i * SA + j] = (uint16_t)cgc; }
                }
                __syncthreads();
            }
            if (act) {                                                                // row i: min over j' >= j; ties -> smaller arg
                const int i = line;
                double v = cs_inf();
                unsigned g = CS_NONE;
                for (int jt = cs1; jt >= cs0; jt -= 4) {
                    double c[4];
                    unsigned cg[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = max(jt - u, cs0);
                        c[u] = PB[(size_t)i * SD + j];
                        cg[u] = PG[(size_t)i * SA + j];
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = jt - u;
                        if (j >= cs0) {
                            cs_take(v, g, c[u], cg[u]);
                            PB[(size_t)i * SD + j] = v;
                            PG[(size_t)i * SA + j] = (uint16_t)g;
                        }
                    }
                }
                if (SEG > 1) { tot_v[tid] = v; tot_g[tid] = g; }
            }
            __syncthreads();
            if (SEG > 1) {
                if (act && seg < SEG - 1) {
                    const int i = line;
                    double cv = cs_inf();
                    unsigned cgc = CS_NONE;
                    for (int t = seg + 1; t < SEG; ++t)                               // the chunks to the right
                        if ((line * SEG + t) < CS_THREADS && t * chunk <= n) cs_take(cv, cgc, tot_v[tid - seg + t], tot_g[tid - seg + t]);
                    for (int j = cs0; j <= cs1; ++j) {
                        double v = PB[(size_t)i * SD + j];
                        unsigned g = PG[(size_t)i * SA + j];
                        cs_take(v, g, cv, cgc);
                        PB[(size_t)i * SD + j] = v;
                        PG[(size_t)i * SA + j] = (uint16_t)g;
                    }
                }
                __syncthreads();
            }
        }
        // ---- the row's minimum and its smallest state: the predecessor of every state of the next row when the
        //      rows are independent, and the whole answer after the last row
        if (!inter || last) {
            if (warp == 0) {
                double v = cs_inf();
                unsigned g = CS_NONE;
                for (int c = lane; c < wd; c += 32) {
                    const double x = fcn[c];
                    if (x < v) { v = x; g = (unsigned)((c << 8) | c); }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ov = __shfl_xor_sync(0xffffffffu, v, o);
                    const unsigned og = __shfl_xor_sync(0xffffffffu, g, o);
                    cs_take(v, g, ov, og);
                }
                if (lane == 0) {
                    if (n > 0) cs_take(v, g, PB[(size_t)n * SD], PG[(size_t)n * SA]);
                    s_gv = v;
                    s_ga = g;
                }
            }
            __syncthreads();
        }
        double *t = fcp; fcp = fcn; fcn = t;
        t = Sa; Sa = Sb; Sb = t;
        np = n; offp = off;
    }
    // ---- walk back: one thread follows the predecessors (one dependent load per row) into shared memory, then all
    //      threads write the rows out
    const double total = s_gv;
    if (!(total < cs_inf())) {                                                        // no feasible combination
        for (int r = r0 + tid; r < r1; r += CS_THREADS) { A.L[r] = 0; A.R[r] = 0; A.row_price[r] = 0.0; }
        if (tid == 0) A.angle_price[k] = cs_inf();
        return;
    }
    uint16_t *chain = (uint16_t *)(PG + (size_t)A.tab_n * SA);                        // [max_rows] state of every row
    if (tid == 0) {
        A.angle_price[k] = total;
        unsigned g = s_ga;
        for (int q = nr - 1; q >= 0; --q) {
            chain[q] = (uint16_t)g;
            if (q > 0) {
                const int r = r0 + q, a = (int)(g >> 8), b = (int)(g & 255u);
                const int n = A.leafrow_col_offset[r + 1] - A.leafrow_col_offset[r];
                const int off = n > 0 ? A.pos0[r] - pmin : 0;
                const uint16_t *bp_row = A.bp + A.row_bp_offset[r];
                g = a == b ? bp_row[a] : bp_row[wd + (b - off) * (n + 1) + (a - off)];
            }
        }
    }
    __syncthreads();
    for (int q = tid; q < nr; q += CS_THREADS) {
        const int r = r0 + q, a = chain[q] >> 8, b = chain[q] & 255;
        const int j0 = A.leafrow_col_offset[r], n = A.leafrow_col_offset[r + 1] - j0;
        const int off = n > 0 ? A.pos0[r] - pmin : 0;
        const double *S = A.S + j0 + r;
        A.L[r] = a - off;
        A.R[r] = b - off;
        A.row_price[r] = a < b ? S[b - off] - S[a - off] : 0.0;
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

// Leaf-travel windows (reading C25): one thread per leaf row of every unoccupied control point k.  The nearest
// occupied control point on either side of k inside k's arc bounds both leaf ends of the same leaf row:
// |a_k - a_k'| <= travel * |k - k'|.  Positions are physical; the windows are written row-local, -/+ CS_BIG where
// nothing binds.
constexpr int CS_MAX_ARCS = 16;
constexpr int CS_BIG = 1 << 30;
struct CsArcs { int n; int off[CS_MAX_ARCS + 1]; };

__global__ void k_leaf_windows(int n_rows, CsArcs arcs, int travel, const uint8_t *__restrict__ angle_mask,
                               const int32_t *__restrict__ leafrow_angle, const int32_t *__restrict__ angle_row_offset,
                               const int32_t *__restrict__ leafrow_col_offset, const int32_t *__restrict__ pos0,
                               const int32_t *__restrict__ angle_pmin, const int32_t *__restrict__ L,
                               const int32_t *__restrict__ R, int32_t *__restrict__ L_lo, int32_t *__restrict__ L_hi,
                               int32_t *__restrict__ R_lo, int32_t *__restrict__ R_hi)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const int k = leafrow_angle[r];
    int llo = -CS_BIG, lhi = CS_BIG, rlo = -CS_BIG, rhi = CS_BIG;
    if (angle_mask[k] == 0) {
        int s = 0;
        while (s + 1 < arcs.n && k >= arcs.off[s + 1]) ++s;
        const int rho = r - angle_row_offset[k];
        const int u0 = leafrow_col_offset[r + 1] > leafrow_col_offset[r] ? pos0[r] : angle_pmin[k];
        for (int step = -1; step <= 1; step += 2) {
            int kk = k + step;
            while (kk >= arcs.off[s] && kk < arcs.off[s + 1] && angle_mask[kk] == 0) kk += step;
            if (kk < arcs.off[s] || kk >= arcs.off[s + 1]) continue;
            const int rr = angle_row_offset[kk] + rho;
            const int v0 = leafrow_col_offset[rr + 1] > leafrow_col_offset[rr] ? pos0[rr] : angle_pmin[kk];
            const int a = L[rr] + v0, b = R[rr] + v0, reach = travel * abs(kk - k);
            llo = max(llo, a - reach - u0); lhi = min(lhi, a + reach - u0);
            rlo = max(rlo, b - reach - u0); rhi = min(rhi, b + reach - u0);
        }
    }
    L_lo[r] = llo; L_hi[r] = lhi; R_lo[r] = rlo; R_hi[r] = rhi;
}

static size_t cs_smem_bytes(int tab_n, int max_wd, int max_rows)
{
    return (size_t)tab_n * cs_stride_d(tab_n) * 8 + (size_t)max_wd * 16 + (size_t)tab_n * 16 +
           (size_t)tab_n * cs_stride_a(tab_n) * 2 + (size_t)max_rows * 2;
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
    if (h->n_leaf_rows > 0) {
        k_cs_prefix<<<(h->n_leaf_rows + 127) / 128, 128, 0, st>>>(h->n_leaf_rows, h->leafrow_col_offset, p, h->S_scratch);
        VMAT_LAUNCH_CHECK();
    }
    // bin 0 (long rows, full-size table, one CTA per SM) on the caller's stream, bin 1 (short rows, small table, several
    // CTAs per SM) on the auxiliary stream at the same time; fork / join by events
    const int cnt0 = h->cs_bin_off[1] - h->cs_bin_off[0], cnt1 = h->cs_bin_off[2] - h->cs_bin_off[1];
    const bool both = cnt0 > 0 && cnt1 > 0;
    if (both) {
        VMAT_CUDA(cudaEventRecord(h->cs_fork, st));
        VMAT_CUDA(cudaStreamWaitEvent(h->cs_aux, h->cs_fork, 0));
    }
    for (int b = 0; b < 2; ++b) {
        const int cnt = b == 0 ? cnt0 : cnt1;
        if (cnt <= 0) continue;
        const int tab_n = h->cs_bin_tab[b];
        cudaStream_t sb = (b == 1 && both) ? h->cs_aux : st;
        CsArgs A{h->angle_row_offset, h->leafrow_col_offset, h->leafrow_pos0, h->angle_pmin, h->angle_wd,
                 h->angle_order + h->cs_bin_off[b], h->row_bp_offset, angle_mask, L_lo, L_hi, R_lo, R_hi, h->S_scratch,
                 h->cs_bp, L, R, row_price, angle_price, interdigitation ? 1 : 0, tab_n, h->cs_max_wd, h->cs_max_rows};
        k_cs_dp<<<cnt, CS_THREADS, cs_smem_bytes(tab_n, h->cs_max_wd, h->cs_max_rows), sb>>>(A);
        VMAT_LAUNCH_CHECK();
    }
    if (both) {
        VMAT_CUDA(cudaEventRecord(h->cs_join, h->cs_aux));
        VMAT_CUDA(cudaStreamWaitEvent(st, h->cs_join, 0));
    }
    k_cs_best<<<1, CS_THREADS, 0, st>>>(h->n_angles, angle_price, best_angle);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

int vmat_launch_leaf_windows(const vmat_ddc *h, const uint8_t *angle_mask, const int32_t *L, const int32_t *R,
                              int32_t n_arcs, const int32_t *arc_angle_offset, int32_t max_leaf_travel, int32_t *L_lo,
                              int32_t *L_hi, int32_t *R_lo, int32_t *R_hi, cudaStream_t st)
{
    REQUIRE(h->leafrow_pos0 != nullptr, "call vmat_ddc_set_leaf_geometry first");
    REQUIRE(n_arcs >= 1 && n_arcs <= CS_MAX_ARCS && arc_angle_offset != nullptr, "n_arcs must be in 1..16");
    REQUIRE(max_leaf_travel >= 0 && max_leaf_travel <= (1 << 16), "max_leaf_travel out of range");
    REQUIRE(arc_angle_offset[0] == 0 && arc_angle_offset[n_arcs] == h->n_angles, "arc_angle_offset must span the control points");
    CsArcs arcs;
    arcs.n = n_arcs;
    for (int s = 0; s <= n_arcs; ++s) arcs.off[s] = arc_angle_offset[s];
    for (int s = 0; s < n_arcs; ++s) {
        REQUIRE(arcs.off[s + 1] >= arcs.off[s], "arc_angle_offset not monotone");
        for (int k = arcs.off[s]; k + 1 < arcs.off[s + 1]; ++k)                          // one MLC per arc
            REQUIRE(h->h_angle_row_offset[k + 1] - h->h_angle_row_offset[k] ==
                        h->h_angle_row_offset[k + 2] - h->h_angle_row_offset[k + 1],
                    "the control points of an arc must have the same number of leaf rows");
    }
    if (h->n_leaf_rows == 0) return VMAT_OK;
    k_leaf_windows<<<(h->n_leaf_rows + 127) / 128, 128, 0, st>>>(h->n_leaf_rows, arcs, max_leaf_travel, angle_mask,
                                                                 h->leafrow_angle, h->angle_row_offset,
                                                                 h->leafrow_col_offset, h->leafrow_pos0, h->angle_pmin, L,
                                                                 R, L_lo, L_hi, R_lo, R_hi);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

extern "C" {

int vmat_leaf_windows(const vmat_ddc *h, const uint8_t *angle_mask, const int32_t *L, const int32_t *R, int32_t n_arcs,
                      const int32_t *arc_angle_offset, int32_t max_leaf_travel, int32_t *L_lo, int32_t *L_hi,
                      int32_t *R_lo, int32_t *R_hi, void *stream)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(h->n_angles == 0 || angle_mask != nullptr, "angle_mask is NULL");
    REQUIRE(h->n_leaf_rows == 0 || (L && R && L_lo && L_hi && R_lo && R_hi), "NULL leaf-row array");
    g_vmat_launches = 0;
    return vmat_launch_leaf_windows(h, angle_mask, L, R, n_arcs, arc_angle_offset, max_leaf_travel, L_lo, L_hi, R_lo, R_hi,
                                    (cudaStream_t)stream);
}

int vmat_ddc_set_leaf_geometry(vmat_ddc *h, const int32_t *leafrow_pos0)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(leafrow_pos0 != nullptr || h->n_leaf_rows == 0, "leafrow_pos0 is NULL");
    const int n_rows = h->n_leaf_rows, n_a = h->n_angles;
    std::vector<int32_t> lco((size_t)n_rows + 1, 0);
    VMAT_CUDA(cudaMemcpy(lco.data(), h->leafrow_col_offset, ((size_t)n_rows + 1) * 4, cudaMemcpyDeviceToHost));
    std::vector<int32_t> pmin((size_t)(n_a > 0 ? n_a : 1), 0), wd((size_t)(n_a > 0 ? n_a : 1), 1);
    std::vector<int64_t> bpo((size_t)n_rows + 1, 0);
    std::vector<int64_t> work((size_t)(n_a > 0 ? n_a : 1), 0);                            // ~ sequential steps of k_cs_dp
    std::vector<int32_t> amax((size_t)(n_a > 0 ? n_a : 1), 0);                            // longest leaf row of a control point
    int max_wd = 1, max_n = 0, max_rows = 1;
    for (int k = 0; k < n_a; ++k) {
        bool any = false;
        int lo = 0, hi = 0;
        const int ra = h->h_angle_row_offset[k], rb = h->h_angle_row_offset[k + 1];
        max_rows = rb - ra > max_rows ? rb - ra : max_rows;
        for (int r = ra; r < rb; ++r) {
            const int n = lco[r + 1] - lco[r];
            if (n <= 0) continue;
            const int64_t e = (int64_t)leafrow_pos0[r] + n;
            REQUIRE(e <= INT32_MAX, "leaf row position overflows int32");
            if (!any || leafrow_pos0[r] < lo) lo = leafrow_pos0[r];
            if (!any || (int)e > hi) hi = (int)e;
            max_n = n > max_n ? n : max_n;
            amax[k] = n > amax[k] ? n : amax[k];
            any = true;
        }
        REQUIRE((int64_t)hi - lo + 1 <= CS_MAX_POS,
                "a control point's field range exceeds 254 beamlet widths (positions 0..254 are packed in 8 bits each; "
                "the pair (255, 255) is the 'no predecessor' mark)");
        pmin[k] = lo;
        wd[k] = hi - lo + 1;
        max_wd = wd[k] > max_wd ? wd[k] : max_wd;
        for (int r = ra; r < rb; ++r) {                          // back pointers of a row: wd closed + (n+1)^2 open states
            const int64_t n1 = (int64_t)(lco[r + 1] - lco[r]) + 1;
            bpo[r + 1] = bpo[r] + wd[k] + n1 * n1;
            work[k] += 3 * n1 + 40;
        }
    }
    const int tab_n = max_n + 1;
    int smem_optin = 0;
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    if (smem_optin > 0 && cs_smem_bytes(tab_n, max_wd, max_rows) + 8192 > (size_t)smem_optin) {
        vmat_set_error("vmat_ddc_set_leaf_geometry: leaf rows of %d beamlets need %zu bytes of shared memory (%d available)",
                       max_n, cs_smem_bytes(tab_n, max_wd, max_rows), smem_optin);
        return VMAT_ERR_INVALID_ARG;
    }
    // The attribute belongs to the kernel on a device, not to this handle: always the device's maximum, so that a
    // second handle with shorter leaf rows can never lower it under what this one launches with.
    {
        int cur = 0;
        VMAT_CUDA(cudaGetDevice(&cur));
        if (cur != h->device) VMAT_CUDA(cudaSetDevice(h->device));
        cudaFuncAttributes fa;
        cudaError_t e = cudaFuncGetAttributes(&fa, k_cs_dp);      // the opt-in maximum covers static + dynamic
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_cs_dp, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - (int)fa.sharedSizeBytes);
        if (cur != h->device) cudaSetDevice(cur);
        VMAT_CUDA(e);
    }
    // launch order: the control points with the most sequential work first, so that the last wave is made of light ones
    std::vector<int32_t> order((size_t)(n_a > 0 ? n_a : 1), 0);
    for (int k = 0; k < n_a; ++k) order[k] = k;
    // ... within two bins: control points with a leaf row beyond CS_SMALL_ROW beamlets first, then the others
    auto bin_of = [&](int k) { return amax[k] > CS_SMALL_ROW ? 0 : 1; };
    std::stable_sort(order.begin(), order.begin() + n_a, [&](int a, int b) {
        return bin_of(a) != bin_of(b) ? bin_of(a) < bin_of(b) : work[a] > work[b];
    });
    h->cs_bin_off[0] = h->cs_bin_off[1] = h->cs_bin_off[2] = 0;
    h->cs_bin_tab[0] = h->cs_bin_tab[1] = 1;
    for (int k = 0; k < n_a; ++k) {
        const int b = bin_of(k);
        h->cs_bin_off[b + 1]++;
        h->cs_bin_tab[b] = amax[k] + 1 > h->cs_bin_tab[b] ? amax[k] + 1 : h->cs_bin_tab[b];
    }
    h->cs_bin_off[2] += h->cs_bin_off[1];
    if (!h->cs_aux) {
        VMAT_CUDA(cudaStreamCreateWithFlags(&h->cs_aux, cudaStreamNonBlocking));
        VMAT_CUDA(cudaEventCreateWithFlags(&h->cs_fork, cudaEventDisableTiming));
        VMAT_CUDA(cudaEventCreateWithFlags(&h->cs_join, cudaEventDisableTiming));
    }
    for (void **q : {(void **)&h->leafrow_pos0, (void **)&h->angle_pmin, (void **)&h->angle_wd, (void **)&h->row_bp_offset,
                     (void **)&h->cs_bp, (void **)&h->angle_order})
        if (*q) { cudaFree(*q); *q = nullptr; }
    auto up = [&](void **dst, const void *src, size_t bytes) -> int {
        VMAT_CUDA(cudaMalloc(dst, bytes > 0 ? bytes : 1));
        if (bytes > 0 && src) VMAT_CUDA(cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
        return VMAT_OK;
    };
    int rc = up((void **)&h->leafrow_pos0, leafrow_pos0, (size_t)n_rows * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_pmin, pmin.data(), (size_t)n_a * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_wd, wd.data(), (size_t)n_a * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->angle_order, order.data(), (size_t)n_a * 4);
    if (rc == VMAT_OK) rc = up((void **)&h->row_bp_offset, bpo.data(), ((size_t)n_rows + 1) * 8);
    if (rc == VMAT_OK) rc = up((void **)&h->cs_bp, nullptr, (size_t)bpo[n_rows] * 2);
    if (rc != VMAT_OK) return rc;
    h->cs_max_wd = max_wd;
    h->cs_max_n = max_n;
    h->cs_max_rows = max_rows;
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
