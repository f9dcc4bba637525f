// master.cu - NEXT-2: the master problem (MP) of the column-generation loop, Eq. (6)-(10) L70-L101
// and the four BB steps of L139: fluence rates y_k in [lo_k, hi_k] of the apertures chosen so far that minimise
// F(z), z = sum_k DA(A_k) y_k, by the Barzilai-Borwein iteration with the subspace step rule.
// Readings C15-C20: DESIGN.md section 2.
//
// Storage: DA is dense, VOXEL-MAJOR, float [n_voxels][m_cap] (the paper's aperture dose vectors are "dense-ish",
// <= 0.15 % of the DDC matrix, L264).  One BB iteration then needs ONE pass over DA: a group of G lanes owns a
// voxel row, its lanes hold the row's entries in registers, the row dot gives z_i (step 4 of L139), the
// voxel's gradient follows (Eq. (1)), and every lane adds DA_ik * dF/dz_i to its own entries of the aperture
// gradient g_A (step 1) - no second read, no atomics.  HBM-bound: 4 m n_voxels bytes per iteration.
// All sums are FP64 in a fixed order (FP32 storage of DA, T, weights): deterministic, and a trajectory differs
// from the FP64 oracle's by summation order only.
#include "common.cuh"
#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>
#include <new>
#include <stdlib.h>
#include <vector>

constexpr int MP_THREADS = 256;
constexpr int MP_WARPS = MP_THREADS / 32;
constexpr int MP_STEP_THREADS = 1024;         // the one-CTA step kernel
constexpr int MP_STEP_WARPS = MP_STEP_THREADS / 32;
constexpr int MP_MAX_NC = 12;                 // up to 12 x 32 = 384 apertures
#ifndef VMAT_MP_CTAS_PER_SM
#define VMAT_MP_CTAS_PER_SM 3
#endif
constexpr int MP_HIST = 6;                    // objective values the "last five changes" rule looks at

struct MpState {                              // device-resident scalars of one solve
    int it;                                   // iteration counter
    int reason;                               // 0 running, 1 stationary, 2 objective, 3 step, 4 max_iter (C19)
    int max_iter;
    double eps_F, eps_y;
    double delta;                             // last step size
    double F;                                 // objective at the current iterate
    double Fh[MP_HIST];                       // F(it), F(it-1), ...
};

struct vmat_mp {
    int32_t n_voxels = 0, m_cap = 0, m = 0;
    int n_cta = 0, n_sm = 0, device = 0;         // n_cta: CTAs of the pass = n_sm x (3 up to 128 apertures, else 2)
    float *DA = nullptr;                      // [n_voxels][m_cap]
    double *y = nullptr, *y_prev = nullptr, *g = nullptr, *g_prev = nullptr, *lo = nullptr, *hi = nullptr;   // [m_cap]
    double *gpart = nullptr;                  // [m_cap][n_cta] per-CTA partials of g_A
    double *spart = nullptr;                  // [n_cta][2]: F partial, curvature partial
    MpState *st = nullptr;
    double *F_hist = nullptr, *delta_hist = nullptr;   // [hist_cap + 1]
    int32_t hist_cap = 0;
    int32_t last_n_iter = 0;
    // the voxels some aperture reaches (rows of DA with a non-zero): only they are visited by the passes
    uint8_t *row_flag = nullptr;              // [n_voxels] set by vmat_mp_add_aperture
    int32_t *active = nullptr;                // [n_voxels] their indices, ascending; valid while active_valid
    int32_t *n_active_dev = nullptr;          // [1]
    void *select_tmp = nullptr;               // scratch of the compaction
    size_t select_tmp_bytes = 0;
    int32_t n_active = 0;
    bool active_valid = false;
    double *F_unreached = nullptr;            // [1] F of the other voxels (z = 0), per solve
};

__device__ __forceinline__ double shfl_xor_d(double v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }

// deterministic block sum of doubles (NW warps); result valid in every thread
template <int NW = MP_WARPS>
__device__ __forceinline__ double mp_block_sum(double v, double *red /* [NW + 1] */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += shfl_xor_d(v, o);
    __syncthreads();                                         // red may still be read from the previous call
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < NW; ++i) s += red[i];
        red[NW] = s;
    }
    __syncthreads();
    return red[NW];
}

// column k of DA; a voxel that any aperture reaches is flagged: only those rows are ever read again
__global__ void k_mp_set_column(int n_voxels, int m_cap, int k, const float *__restrict__ col, float *__restrict__ DA,
                                uint8_t *__restrict__ row_flag)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_voxels) {
        const float v = col[i];
        DA[(size_t)i * m_cap + k] = v;
        if (v != 0.f) row_flag[i] = 1;
    }
}

// F of the voxels no aperture reaches (z_i = 0 whatever y): their terms of Eq. (1) at z = 0.  One CTA, fixed order.
__global__ void __launch_bounds__(1024)
k_mp_unreached_F(int n_voxels, const uint8_t *__restrict__ row_flag, const uint8_t *__restrict__ vstruct,
                 const float *__restrict__ T, const float *__restrict__ w_over, const float *__restrict__ w_under,
                 double *__restrict__ out)
{
    __shared__ double red[33];
    double s = 0.0;
    for (int i = threadIdx.x; i < n_voxels; i += 1024)
        if (!row_flag[i]) {
            const int sid = vstruct[i];
            const double Ti = (double)T[sid], over = fmax(0.0 - Ti, 0.0), under = fmax(Ti - 0.0, 0.0);
            s += (double)w_over[sid] * over * over + (double)w_under[sid] * under * under;
        }
    const double tot = mp_block_sum<32>(s, red);
    if (threadIdx.x == 0) out[0] = tot;
}

__global__ void k_mp_clip(int m, double *__restrict__ y, const double *__restrict__ lo, const double *__restrict__ hi)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < m) y[k] = fmin(fmax(y[k], lo[k]), hi[k]);
}

// ---------------------------------------------------------------- the pass over DA
// CURV = false: z = DA y, F, dF/dz, partials of g_A = DA^T dF/dz            (steps 4 and 1 of L139)
// CURV = true : z = DA y, q = DA g, partials of sum_i w_i q_i^2              (first step size, C17)
//
// A group of LPR = 2^LOG lanes owns a voxel row, lane gl of the group holds
// columns (c LPR + gl) 4 .. + 3 of it for c < NC (one 16-byte load each; the group reads the row contiguously), and a
// warp works on 8 x (32 / LPR) rows at a time (4 when a row is wider than 128 entries).  Every lane forms its part
// of the 8 row dot products in FP64; a halving butterfly (8 -> 4 -> 2 -> 1 values per lane, 7 + LOG - 3 double
// shuffles for 8 rows instead of 8 LOG) leaves the sum of row (gl >> (LOG - 3)) in the lane.  The objective and
// dF/dz_i follow per row, dF/dz_i is broadcast back, and every lane adds DA_ik dF/dz_i into the FP64 accumulators of
// its own columns, which it keeps over all its rows - the row's entries are still in the lane's own shared-memory
// FIFO slot (filled by cp.async one step ahead, read conflict-free), so DA is read from HBM once.
// Fixed assignment of rows to warps and fixed reduction trees: deterministic.
// (History: lanes-per-row with a full FP64 shuffle tree per row ran at 0.7-1.3 TB/s; shared-memory tiles filled by
// cp.async with thread-per-row dot products at 3.6 TB/s under ncu, L1TEX-bound at 79 % by the tile being written
// once and read twice plus 32 bytes of y per 16 bytes of tile.)
// 2^RBL (8 or 4) values per lane, summed over the LPR lanes of a group by a halving butterfly: lane gl ends with the
// total of value gl >> (LOG - RBL)
template <int LOG, int RBL>
__device__ __forceinline__ double mp_reduce(const double (&v)[1 << RBL], int gl)
{
    constexpr int LPR = 1 << LOG;
    double w4[4], w2[2];
    if (RBL == 3) {
        const bool up = (gl & (LPR / 2)) != 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double keep = up ? v[(i + 4) & ((1 << RBL) - 1)] : v[i], send = up ? v[i] : v[(i + 4) & ((1 << RBL) - 1)];
            w4[i] = keep + shfl_xor_d(send, LPR / 2);
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) w4[i] = v[i & ((1 << RBL) - 1)];
    }
    constexpr int O2 = RBL == 3 ? LPR / 4 : LPR / 2;          // offsets of the 4 -> 2 and 2 -> 1 steps
    {
        const bool up = (gl & O2) != 0;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double keep = up ? w4[i + 2] : w4[i], send = up ? w4[i] : w4[i + 2];
            w2[i] = keep + shfl_xor_d(send, O2);
        }
    }
    const bool up = (gl & (O2 / 2)) != 0;
    double w1 = (up ? w2[1] : w2[0]) + shfl_xor_d(up ? w2[0] : w2[1], O2 / 2);
#pragma unroll
    for (int o = O2 / 4; o > 0; o >>= 1) w1 += shfl_xor_d(w1, o);
    return w1;
}

// 16-byte asynchronous copy global -> shared, bypassing L1
__device__ __forceinline__ void mp_cp_async16(void *smem, const void *gmem)
{
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void mp_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// a shared-memory read the compiler may not merge with an earlier one of the same address
__device__ __forceinline__ float4 mp_lds_again(const float4 *p)
{
    float4 r;
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(p);
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "r"(sa));
    return r;
}
template <int N>
__device__ __forceinline__ void mp_cp_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

// rows per lane group and step: 8, or 4 for wide rows, so that a stage stays at 4-6 KB per warp and two CTAs fit an SM
__host__ __device__ constexpr int mp_rbl(int NC) { return NC >= 2 ? 2 : 3; }
__host__ __device__ constexpr int mp_stages(int NC) { return 2; }
__host__ __device__ constexpr size_t mp_ring_bytes(int NC)
{
    return (size_t)MP_WARPS * mp_stages(NC) * (1 << mp_rbl(NC)) * NC * 32 * 16;
}

template <bool CURV, int LOG, int NC>
__global__ void __launch_bounds__(MP_THREADS, NC <= 2 ? 3 : 2)
k_mp_pass(int n_voxels /* rows to visit: the reached voxels */, const int32_t *__restrict__ active /* their indices */,
          int m, int m_cap, const float *__restrict__ DA, const double *__restrict__ y, const double *__restrict__ gvec,
          const uint8_t *__restrict__ vstruct, int n_struct, const float *__restrict__ T,
          const float *__restrict__ w_over, const float *__restrict__ w_under, float *__restrict__ z_out,
          double *__restrict__ gpart, double *__restrict__ spart, const MpState *__restrict__ st)
{
    if (st->reason != 0) return;                              // the solve has stopped: nothing to do
    constexpr int RBL = mp_rbl(NC), RB = 1 << RBL;
    constexpr int LPR = 1 << LOG, GPW = 32 / LPR, LOWB = LOG - RBL, COLS = LPR * NC * 4;
    constexpr int STAGES = mp_stages(NC), ITEMS = RB * NC;    // 16-byte chunks per lane and stage
    extern __shared__ float4 mp_ring[];                       // [warp][STAGES][ITEMS][32]: every lane's own prefetch FIFO
    __shared__ double red_s[MP_WARPS + 1];
    __shared__ float sT[256], sWo[256], sWu[256];             // the objective's tables
    for (int t = threadIdx.x; t < n_struct; t += MP_THREADS) { sT[t] = T[t]; sWo[t] = w_over[t]; sWu[t] = w_under[t]; }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gl = lane & (LPR - 1), grp = lane >> LOG;
    double yk[NC][4], vk[NC][4], acc[NC][4];
    bool colok[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const int col = (c * LPR + gl) * 4;
        colok[c] = col < m;                                   // m_cap is a multiple of 8: the 16-byte chunk stays inside the row
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            yk[c][j] = col + j < m ? y[col + j] : 0.0;
            vk[c][j] = (CURV && col + j < m) ? gvec[col + j] : 0.0;
            acc[c][j] = 0.0;
        }
    }
    double ssum = 0.0;
    const int my_slot = gl >> LOWB;                           // the row slot whose total this lane ends up with
    const bool leader = (gl & ((1 << LOWB) - 1)) == 0;        // one lane per row adds to F and writes z
    const int64_t step = (int64_t)gridDim.x * MP_WARPS * (RB * GPW);
    const int64_t base0 = (int64_t)(blockIdx.x * MP_WARPS + warp) * (RB * GPW);
    float4 *my = mp_ring + (size_t)warp * STAGES * ITEMS * 32 + lane;
    // a stage = the 8 row slots of one step; every lane copies the chunks it will read itself, so no barrier is needed
    auto issue = [&](int64_t base, int st) {
        if (base < n_voxels) {
#pragma unroll
            for (int s = 0; s < RB; ++s) {                    // slot s of group grp is row base + s GPW + grp
                const int64_t pos = base + s * GPW + grp;
                const int64_t row = pos < n_voxels ? (int64_t)active[pos] : 0;
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    float4 *dst = my + (size_t)(st * ITEMS + s * NC + c) * 32;
                    if (pos < n_voxels && colok[c]) mp_cp_async16(dst, DA + row * m_cap + (c * LPR + gl) * 4);
                    else *dst = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
        }
        mp_cp_commit();
    };
#pragma unroll
    for (int st = 0; st < STAGES - 1; ++st) issue(base0 + st * step, st);
    int cur = 0;
    for (int64_t base = base0; base < n_voxels; base += step) {
        {
            int nxt = cur + STAGES - 1;
            if (nxt >= STAGES) nxt -= STAGES;
            issue(base + (STAGES - 1) * step, nxt);
        }
        mp_cp_wait<STAGES - 1>();
        const float4 *stg = my + (size_t)cur * ITEMS * 32;
        if (++cur == STAGES) cur = 0;
        double pz[RB], pq[RB];
#pragma unroll
        for (int s = 0; s < RB; ++s) {
            double zi = 0.0, qi = 0.0;
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const float4 e = stg[(size_t)(s * NC + c) * 32];
                const double a0 = (double)e.x, a1 = (double)e.y, a2 = (double)e.z, a3 = (double)e.w;
                zi = fma(a0, yk[c][0], zi); zi = fma(a1, yk[c][1], zi); zi = fma(a2, yk[c][2], zi); zi = fma(a3, yk[c][3], zi);
                if (CURV) {
                    qi = fma(a0, vk[c][0], qi); qi = fma(a1, vk[c][1], qi); qi = fma(a2, vk[c][2], qi); qi = fma(a3, vk[c][3], qi);
                }
            }
            pz[s] = zi; pq[s] = qi;
        }
        const double zi = mp_reduce<LOG, RBL>(pz, gl);
        const double qi = CURV ? mp_reduce<LOG, RBL>(pq, gl) : 0.0;
        const int64_t pos = base + my_slot * GPW + grp;
        double gz = 0.0;
        if (pos < n_voxels) {
            const int i = active[pos];
            const int sid = vstruct[i];
            const double Ti = (double)sT[sid], wo = (double)sWo[sid], wu = (double)sWu[sid];
            if (!CURV) {
                const double over = fmax(zi - Ti, 0.0), under = fmax(Ti - zi, 0.0);
                gz = 2.0 * wo * over - 2.0 * wu * under;                                 // Eq. (1), sign C1
                if (leader) {
                    ssum += wo * over * over + wu * under * under;
                    if (z_out) z_out[i] = (float)zi;
                }
            } else if (leader) {
                const double w = zi > Ti ? wo : (zi < Ti ? wu : 0.0);                    // C17
                ssum += w * qi * qi;
            }
        }
        if (!CURV) {
#pragma unroll NC >= 2 ? 1 : 2
            for (int s = 0; s < RB; ++s) {                    // g_A += DA_i: * dF/dz_i; wide rows: rolled, to bound the registers
                const double gs = __shfl_sync(0xffffffffu, gz, (grp << LOG) + (s << LOWB));
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const float4 e = mp_lds_again(stg + (size_t)(s * NC + c) * 32);   // not kept in registers
                    acc[c][0] = fma((double)e.x, gs, acc[c][0]); acc[c][1] = fma((double)e.y, gs, acc[c][1]);
                    acc[c][2] = fma((double)e.z, gs, acc[c][2]); acc[c][3] = fma((double)e.w, gs, acc[c][3]);
                }
            }
        }
    }
    // ---- CTA partials in a fixed order: the groups of a warp, then the warps (in the ring's memory, free by now)
    if (!CURV) {
        double *accs = (double *)mp_ring;                     // [MP_WARPS][COLS] <= 24 KB
        mp_cp_wait<0>();
        __syncthreads();
#pragma unroll
        for (int c = 0; c < NC; ++c)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                double v = acc[c][j];
#pragma unroll
                for (int o = LPR; o < 32; o <<= 1) v += shfl_xor_d(v, o);
                if (grp == 0) accs[warp * COLS + (c * LPR + gl) * 4 + j] = v;
            }
        __syncthreads();
        for (int k = threadIdx.x; k < m; k += MP_THREADS) {
            double sacc = 0.0;
            for (int w = 0; w < MP_WARPS; ++w) sacc += accs[w * COLS + k];
            gpart[(size_t)k * gridDim.x + blockIdx.x] = sacc;                             // [m_cap][n_cta]
        }
    }
    const double tot = mp_block_sum(ssum, red_s);
    if (threadIdx.x == 0) spart[2 * blockIdx.x + (CURV ? 1 : 0)] = tot;
}

// ---------------------------------------------------------------- the step: one CTA
// PHASE 0: after the first gradient pass (it = 0): finish g_A, subspace rule, stopping rules; no update.
// PHASE 1: after the curvature pass: delta_0 (C17), update.
// PHASE 2: after a gradient pass, it >= 1: finish g_A, subspace rule, stopping rules, Eq. (7)/(8), update.
template <int PHASE>
__global__ void __launch_bounds__(MP_STEP_THREADS)
k_mp_step(int m, int m_cap, int n_cta, double *__restrict__ y, double *__restrict__ y_prev, double *__restrict__ g,
          double *__restrict__ g_prev, const double *__restrict__ lo, const double *__restrict__ hi,
          const double *__restrict__ gpart, const double *__restrict__ spart, MpState *__restrict__ st,
          double *__restrict__ F_hist, double *__restrict__ delta_hist, const double *__restrict__ F_unreached)
{
    if (st->reason != 0) return;
    __shared__ double red_s[MP_STEP_WARPS + 1];
    __shared__ int s_flag;
    const int it = st->it;
    if (PHASE != 1) {
        // ---- g_A = sum of the CTA partials (fixed order), subspace rule Eq. (9)/(10) with the sign of C15
        int nonzero = 0;
        double dy_max = 0.0;
        // one warp per aperture: lane l adds partials l, l+32, ... in that order, then a fixed shuffle tree
        for (int k = threadIdx.x >> 5; k < m; k += MP_STEP_WARPS) {
            const double *col = gpart + (size_t)k * n_cta;
            double s = 0.0;
            for (int c0 = threadIdx.x & 31; c0 < n_cta; c0 += 32 * 16) {        // 16 loads in flight, added in the same order
                double v[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) v[u] = c0 + 32 * u < n_cta ? col[c0 + 32 * u] : 0.0;
#pragma unroll
                for (int u = 0; u < 16; ++u)
                    if (c0 + 32 * u < n_cta) s += v[u];
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += shfl_xor_d(s, o);
            const double yk = y[k];
            if ((yk <= lo[k] && s > 0.0) || (yk >= hi[k] && s < 0.0)) s = 0.0;
            if ((threadIdx.x & 31) == 0) g[k] = s;
            nonzero |= s != 0.0;
            if (it >= 1) dy_max = fmax(dy_max, fabs(yk - y_prev[k]));
        }
        double fs = 0.0;
        for (int c = threadIdx.x; c < n_cta; c += MP_STEP_THREADS) fs += spart[2 * c];
        const double F = mp_block_sum<MP_STEP_WARPS>(fs, red_s) + F_unreached[0];
        if (threadIdx.x == 0) s_flag = 0;
        __syncthreads();
        if (nonzero) atomicOr(&s_flag, 1);
        // max over the block of dy_max (exact, order-free)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dy_max = fmax(dy_max, shfl_xor_d(dy_max, o));
        __shared__ double red_m[MP_STEP_WARPS];
        if ((threadIdx.x & 31) == 0) red_m[threadIdx.x >> 5] = dy_max;
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int i = 0; i < MP_STEP_WARPS; ++i) dy_max = fmax(dy_max, red_m[i]);
            for (int j = MP_HIST - 1; j > 0; --j) st->Fh[j] = st->Fh[j - 1];
            st->Fh[0] = F;
            st->F = F;
            F_hist[it] = F;
            // ---- stopping rules, in the order of C19
            int reason = 0;
            if (!s_flag) reason = 1;
            else {
                bool flat = it >= 5;
                for (int j = 0; flat && j < 5; ++j)
                    flat = fabs(st->Fh[j] - st->Fh[j + 1]) <= st->eps_F * fabs(st->Fh[j + 1]);
                if (flat) reason = 2;
                else if (it >= 1 && dy_max <= st->eps_y) reason = 3;
                else if (it >= st->max_iter) reason = 4;
            }
            st->reason = reason;
            s_flag = reason;
        }
        __syncthreads();
        if (s_flag != 0 || PHASE == 0) return;           // (the barrier above also publishes g to the whole CTA)
    }
    // ---- step size
    double delta;
    if (PHASE == 1) {
        double cs = 0.0, gg = 0.0;
        for (int c = threadIdx.x; c < n_cta; c += MP_STEP_THREADS) cs += spart[2 * c + 1];
        for (int k = threadIdx.x; k < m; k += MP_STEP_THREADS) gg += g[k] * g[k];
        const double den = 2.0 * mp_block_sum<MP_STEP_WARPS>(cs, red_s);
        const double num = mp_block_sum<MP_STEP_WARPS>(gg, red_s);
        delta = den > 0.0 ? num / den : 1.0;                                             // C17
    } else {
        double ss = 0.0, sv = 0.0, tt = 0.0;
        for (int k = threadIdx.x; k < m; k += MP_STEP_THREADS) {
            const double s = y[k] - y_prev[k], t = g[k] - g_prev[k];
            ss += s * s; sv += s * t; tt += t * t;
        }
        ss = mp_block_sum<MP_STEP_WARPS>(ss, red_s);
        sv = mp_block_sum<MP_STEP_WARPS>(sv, red_s);
        tt = mp_block_sum<MP_STEP_WARPS>(tt, red_s);
        delta = st->delta;                                                               // kept when <s,t> <= 0 (C18)
        if (sv > 0.0 && tt > 0.0) delta = (it & 1) ? ss / sv : sv / tt;                  // Eq. (7) odd, Eq. (8) even
    }
    // ---- update within the box (step 3; C16)
    for (int k = threadIdx.x; k < m; k += MP_STEP_THREADS) {
        const double yk = y[k], gk = g[k];
        y_prev[k] = yk;
        g_prev[k] = gk;
        y[k] = fmin(fmax(yk - delta * gk, lo[k]), hi[k]);
    }
    if (threadIdx.x == 0) {
        st->delta = delta;
        delta_hist[it] = delta;
        st->it = it + 1;
    }
}

// ---------------------------------------------------------------- host side
static void mp_set_smem_attributes()
{
#define MP_ATTR(CURV, LOG, NC) \
    cudaFuncSetAttribute(k_mp_pass<CURV, LOG, NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mp_ring_bytes(NC))
    MP_ATTR(false, 3, 1); MP_ATTR(false, 4, 1); MP_ATTR(false, 5, 1); MP_ATTR(false, 5, 2); MP_ATTR(false, 5, 3);
    MP_ATTR(true, 3, 1); MP_ATTR(true, 4, 1); MP_ATTR(true, 5, 1); MP_ATTR(true, 5, 2); MP_ATTR(true, 5, 3);
#undef MP_ATTR
}

template <bool CURV>
static void mp_launch_pass(const vmat_mp *h, const uint8_t *vs, int n_struct, const float *T, const float *wo,
                           const float *wu, float *z, cudaStream_t s)
{
#define MP_PASS(LOG, NC)                                                                                            \
    k_mp_pass<CURV, LOG, NC><<<h->n_cta, MP_THREADS, mp_ring_bytes(NC), s>>>(h->n_active, h->active, h->m, h->m_cap, h->DA, h->y, h->g, vs,   \
                                                             n_struct, T, wo, wu, z, h->gpart, h->spart, h->st)
    const int m = h->m;                                      // lanes per row x 16-byte chunks per lane covering m columns
    if (m <= 32) MP_PASS(3, 1);                              // (8 columns per lane up to m = 128 measured 6-13 % slower)
    else if (m <= 64) MP_PASS(4, 1);
    else if (m <= 128) MP_PASS(5, 1);
    else if (m <= 256) MP_PASS(5, 2);
    else MP_PASS(5, 3);
#undef MP_PASS
}

template <int PHASE>
static void mp_launch_step(const vmat_mp *h, cudaStream_t s)
{
    k_mp_step<PHASE><<<1, MP_STEP_THREADS, 0, s>>>(h->m, h->m_cap, h->n_cta, h->y, h->y_prev, h->g, h->g_prev, h->lo, h->hi,
                                              h->gpart, h->spart, h->st, h->F_hist, h->delta_hist, h->F_unreached);
}

#define REQUIRE(cond, msg)                                            \
    do {                                                              \
        if (!(cond)) { vmat_set_error("%s: %s", __func__, msg); return VMAT_ERR_INVALID_ARG; } \
    } while (0)

extern "C" {

int vmat_mp_destroy(vmat_mp *h)
{
    if (!h) return VMAT_OK;
    void *ptrs[] = {h->DA, h->y, h->y_prev, h->g, h->g_prev, h->lo, h->hi, h->gpart, h->spart, h->st, h->F_hist,
                    h->delta_hist, h->row_flag, h->active, h->n_active_dev, h->select_tmp, h->F_unreached};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    delete h;
    return VMAT_OK;
}

int vmat_mp_create(vmat_mp **out, int32_t n_voxels, int32_t max_apertures, void *stream)
{
    REQUIRE(out != nullptr, "out is NULL");
    REQUIRE(n_voxels >= 0, "negative n_voxels");
    REQUIRE(max_apertures >= 1 && max_apertures <= MP_MAX_NC * 32, "max_apertures must be in 1..384");
    vmat_mp *h = new (std::nothrow) vmat_mp();
    if (!h) { vmat_set_error("vmat_mp_create: host allocation failed"); return VMAT_ERR_OOM; }
    h->n_voxels = n_voxels;
    h->m_cap = (max_apertures + 7) / 8 * 8;                  // rows start on 32-byte boundaries
    cudaGetDevice(&h->device);
    int n_sm = 1;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, h->device);
    mp_set_smem_attributes();
    h->n_sm = n_sm;
    h->n_cta = n_sm * VMAT_MP_CTAS_PER_SM;                                     // the most a pass uses (allocation)
    cudaStream_t s = (cudaStream_t)stream;
    auto alloc = [&](void **p, size_t bytes) { return cudaMalloc(p, bytes > 0 ? bytes : 1) == cudaSuccess; };
    const size_t mc = (size_t)h->m_cap;
    bool ok = alloc((void **)&h->DA, (size_t)n_voxels * mc * 4) && alloc((void **)&h->y, mc * 8) &&
              alloc((void **)&h->y_prev, mc * 8) && alloc((void **)&h->g, mc * 8) && alloc((void **)&h->g_prev, mc * 8) &&
              alloc((void **)&h->lo, mc * 8) && alloc((void **)&h->hi, mc * 8) &&
              alloc((void **)&h->gpart, (size_t)h->n_cta * mc * 8) && alloc((void **)&h->spart, (size_t)h->n_cta * 16) &&
              alloc((void **)&h->st, sizeof(MpState)) && alloc((void **)&h->row_flag, (size_t)n_voxels) &&
              alloc((void **)&h->active, (size_t)n_voxels * 4) && alloc((void **)&h->n_active_dev, 4) &&
              alloc((void **)&h->F_unreached, 8);
    if (ok) {
        cub::DeviceSelect::Flagged(nullptr, h->select_tmp_bytes, thrust::counting_iterator<int32_t>(0), h->row_flag, h->active,
                                   h->n_active_dev, n_voxels, s);
        ok = alloc(&h->select_tmp, h->select_tmp_bytes);
    }
    if (!ok) {
        cudaGetLastError();
        vmat_mp_destroy(h);
        vmat_set_error("vmat_mp_create: device allocation failed (%lld voxels x %d apertures)", (long long)n_voxels, h->m_cap);
        return VMAT_ERR_OOM;
    }
    cudaMemsetAsync(h->DA, 0, (size_t)n_voxels * mc * 4, s);
    cudaMemsetAsync(h->row_flag, 0, (size_t)(n_voxels > 0 ? n_voxels : 1), s);
    cudaMemsetAsync(h->y, 0, mc * 8, s);
    cudaMemsetAsync(h->spart, 0, (size_t)h->n_cta * 16, s);
    h->n_cta = 0;                                                              // set per solve
    VMAT_CUDA(cudaStreamSynchronize(s));
    *out = h;
    return VMAT_OK;
}

// forgets the apertures and the reached-voxel flags (on stream s)
static int mp_forget(vmat_mp *h, cudaStream_t s)
{
    h->m = 0;
    h->active_valid = false;
    if (h->n_voxels > 0) VMAT_CUDA(cudaMemsetAsync(h->row_flag, 0, (size_t)h->n_voxels, s));
    return VMAT_OK;
}

int vmat_mp_reset(vmat_mp *h)
{
    REQUIRE(h != nullptr, "handle is NULL");
    VMAT_CUDA(cudaDeviceSynchronize());                      // no stream argument: order against everything
    int rc = mp_forget(h, nullptr);
    if (rc == VMAT_OK) VMAT_CUDA(cudaDeviceSynchronize());
    return rc;
}

int vmat_mp_add_aperture(vmat_mp *h, const float *DA, double y0, double y_lo, double y_hi, void *stream)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(DA != nullptr || h->n_voxels == 0, "DA is NULL");
    REQUIRE(h->m < h->m_cap, "the handle is full (max_apertures)");
    REQUIRE(y_lo <= y_hi, "y_lo > y_hi");
    cudaStream_t s = (cudaStream_t)stream;
    g_vmat_launches = 0;
    const int k = h->m;
    if (h->n_voxels > 0) {
        k_mp_set_column<<<(h->n_voxels + 255) / 256, 256, 0, s>>>(h->n_voxels, h->m_cap, k, DA, h->DA, h->row_flag);
        h->active_valid = false;
        VMAT_LAUNCH_CHECK();
    }
    const double v[3] = {y0 < y_lo ? y_lo : (y0 > y_hi ? y_hi : y0), y_lo, y_hi};
    VMAT_CUDA(cudaMemcpyAsync(h->y + k, &v[0], 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaMemcpyAsync(h->lo + k, &v[1], 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaMemcpyAsync(h->hi + k, &v[2], 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaStreamSynchronize(s));                     // v lives on this stack frame
    h->m = k + 1;
    return VMAT_OK;
}

int vmat_mp_set_fluence(vmat_mp *h, const double *y_host, void *stream)
{
    REQUIRE(h && y_host, "NULL argument");
    if (h->m > 0) {
        VMAT_CUDA(cudaMemcpyAsync(h->y, y_host, (size_t)h->m * 8, cudaMemcpyHostToDevice, (cudaStream_t)stream));
        VMAT_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    }
    return VMAT_OK;
}

int vmat_mp_solve(vmat_mp *h, const uint8_t *voxel_struct, int32_t n_struct, const float *T, const float *w_over,
                  const float *w_under, int32_t max_iter, double eps_F, double eps_y, float *z, double *y_host,
                  double *F_host, int32_t *n_iter_host, int32_t *reason_host, void *stream)
{
    REQUIRE(h && T && w_over && w_under, "NULL argument");
    REQUIRE(h->n_voxels == 0 || voxel_struct, "voxel_struct is NULL");
    REQUIRE(n_struct >= 1 && n_struct <= 256, "n_struct must be in 1..256");
    REQUIRE(h->m >= 1, "no aperture has been added");
    REQUIRE(max_iter >= 0 && max_iter <= (1 << 24), "max_iter out of range");
    REQUIRE(eps_F >= 0.0 && eps_y >= 0.0, "negative tolerance");
    cudaStream_t s = (cudaStream_t)stream;
    g_vmat_launches = 0;
    // resident CTAs per SM of the pass kernel that m selects; fixed by m, so every summation order is fixed by m
    h->n_cta = h->n_sm * (h->m <= 256 ? 3 : 2);
    // the voxels some aperture reaches, ascending; F of the others (their dose is 0 whatever y)
    if (!h->active_valid) {
        h->n_active = 0;
        if (h->n_voxels > 0) {
            size_t tb = h->select_tmp_bytes;
            VMAT_CUDA(cub::DeviceSelect::Flagged(h->select_tmp, tb, thrust::counting_iterator<int32_t>(0), h->row_flag,
                                                 h->active, h->n_active_dev, h->n_voxels, s));
            g_vmat_launches += 2;
            VMAT_CUDA(cudaMemcpyAsync(&h->n_active, h->n_active_dev, 4, cudaMemcpyDeviceToHost, s));
            VMAT_CUDA(cudaStreamSynchronize(s));
        }
        h->active_valid = true;
    }
    k_mp_unreached_F<<<1, 1024, 0, s>>>(h->n_voxels, h->row_flag, voxel_struct, T, w_over, w_under, h->F_unreached);
    VMAT_LAUNCH_CHECK();
    if (z && h->n_voxels > 0) VMAT_CUDA(cudaMemsetAsync(z, 0, (size_t)h->n_voxels * 4, s));   // unreached voxels: z = 0
    if (max_iter + 1 > h->hist_cap) {
        if (h->F_hist) cudaFree(h->F_hist);
        if (h->delta_hist) cudaFree(h->delta_hist);
        h->F_hist = h->delta_hist = nullptr;
        h->hist_cap = 0;
        VMAT_CUDA(cudaMalloc((void **)&h->F_hist, ((size_t)max_iter + 1) * 8));
        VMAT_CUDA(cudaMalloc((void **)&h->delta_hist, ((size_t)max_iter + 1) * 8));
        h->hist_cap = max_iter + 1;
    }
    MpState init = {};
    init.max_iter = max_iter; init.eps_F = eps_F; init.eps_y = eps_y;
    VMAT_CUDA(cudaMemcpyAsync(h->st, &init, sizeof(init), cudaMemcpyHostToDevice, s));
    k_mp_clip<<<(h->m + 127) / 128, 128, 0, s>>>(h->m, h->y, h->lo, h->hi);          // the start must be feasible (C16)
    VMAT_LAUNCH_CHECK();
    // iteration 0: gradient pass, step A, curvature pass, step B
    mp_launch_pass<false>(h, voxel_struct, n_struct, T, w_over, w_under, z, s); VMAT_LAUNCH_CHECK();
    mp_launch_step<0>(h, s); VMAT_LAUNCH_CHECK();
    mp_launch_pass<true>(h, voxel_struct, n_struct, T, w_over, w_under, nullptr, s); VMAT_LAUNCH_CHECK();
    mp_launch_step<1>(h, s); VMAT_LAUNCH_CHECK();
    MpState cur;
    const int BATCH = 8;                                     // iterations enqueued between two looks at the stop flag
    for (;;) {
        VMAT_CUDA(cudaMemcpyAsync(&cur, h->st, sizeof(cur), cudaMemcpyDeviceToHost, s));
        VMAT_CUDA(cudaStreamSynchronize(s));
        if (cur.reason != 0) break;
        for (int b = 0; b < BATCH; ++b) {                    // kernels after the stop are no-ops (they read the flag)
            mp_launch_pass<false>(h, voxel_struct, n_struct, T, w_over, w_under, z, s); VMAT_LAUNCH_CHECK();
            mp_launch_step<2>(h, s); VMAT_LAUNCH_CHECK();
        }
    }
    h->last_n_iter = cur.it;
    if (y_host) VMAT_CUDA(cudaMemcpyAsync(y_host, h->y, (size_t)h->m * 8, cudaMemcpyDeviceToHost, s));
    VMAT_CUDA(cudaStreamSynchronize(s));
    if (F_host) *F_host = cur.F;
    if (n_iter_host) *n_iter_host = cur.it;
    if (reason_host) *reason_host = cur.reason;
    return VMAT_OK;
}

int vmat_mp_history(const vmat_mp *h, double *F_hist, double *delta_hist)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(h->F_hist != nullptr, "no solve has run");
    VMAT_CUDA(cudaDeviceSynchronize());
    if (F_hist) VMAT_CUDA(cudaMemcpy(F_hist, h->F_hist, ((size_t)h->last_n_iter + 1) * 8, cudaMemcpyDeviceToHost));
    if (delta_hist && h->last_n_iter > 0)
        VMAT_CUDA(cudaMemcpy(delta_hist, h->delta_hist, (size_t)h->last_n_iter * 8, cudaMemcpyDeviceToHost));
    return VMAT_OK;
}

// The column-generation loop of PAPER.md L56 / Figure 1(a), every step on the device; the host only reads the
// chosen control point (4 bytes) per outer iteration and the master problem's stop flag.
int vmat_column_generation(vmat_ddc *h, vmat_mp *mp, const uint8_t *voxel_struct, int32_t n_struct, const float *T,
                           const float *w_over, const float *w_under, int32_t max_apertures, double y_lo, double y_hi,
                           int32_t mp_max_iter, double eps_F, double eps_y, float *z, int32_t *L, int32_t *R,
                           int32_t *n_apertures_host, int32_t *angles_host, double *y_host, double *F_hist_host,
                           double *aperture_price_host, int32_t *mp_iters_host, int32_t *stop_host, void *stream)
{
    return vmat_column_generation_ex(h, mp, voxel_struct, n_struct, T, w_over, w_under, max_apertures, y_lo, y_hi,
                                     mp_max_iter, eps_F, eps_y, 0, -1, 0, nullptr, z, L, R, n_apertures_host, angles_host,
                                     y_host, F_hist_host, aperture_price_host, mp_iters_host, stop_host, stream);
}

// With interdigitation != 0 or max_leaf_travel >= 0 the pricing step is: price kernel, leaf-travel windows from the
// occupied control points (reading C25), constrained selection (constrained.cu).
int vmat_column_generation_ex(vmat_ddc *h, vmat_mp *mp, const uint8_t *voxel_struct, int32_t n_struct, const float *T,
                              const float *w_over, const float *w_under, int32_t max_apertures, double y_lo, double y_hi,
                              int32_t mp_max_iter, double eps_F, double eps_y, int32_t interdigitation,
                              int32_t max_leaf_travel, int32_t n_arcs, const int32_t *arc_angle_offset, float *z,
                              int32_t *L, int32_t *R, int32_t *n_apertures_host, int32_t *angles_host, double *y_host,
                              double *F_hist_host, double *aperture_price_host, int32_t *mp_iters_host,
                              int32_t *stop_host, void *stream)
{
    REQUIRE(h && mp && T && w_over && w_under && n_apertures_host, "NULL argument");
    REQUIRE(h->n_voxels == mp->n_voxels, "the DDC handle and the master problem differ in n_voxels");
    REQUIRE(h->n_voxels == 0 || (voxel_struct && z), "NULL voxel vector");
    REQUIRE(h->n_leaf_rows == 0 || (L && R), "NULL leaf-row output");
    REQUIRE(max_apertures >= 0 && max_apertures <= mp->m_cap, "max_apertures exceeds the master problem's capacity");
    REQUIRE(n_struct >= 1 && n_struct <= 256, "n_struct must be in 1..256");
    REQUIRE(y_lo <= y_hi, "y_lo > y_hi");
    const bool constrained = interdigitation != 0 || max_leaf_travel >= 0;
    REQUIRE(!constrained || h->leafrow_pos0 != nullptr, "constraints need vmat_ddc_set_leaf_geometry");
    REQUIRE(max_leaf_travel < 0 || (n_arcs >= 1 && arc_angle_offset != nullptr), "max_leaf_travel needs the arcs");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t nv = (size_t)(h->n_voxels > 0 ? h->n_voxels : 1), nb = (size_t)(h->n_beamlets > 0 ? h->n_beamlets : 1);
    const size_t nr = (size_t)(h->n_leaf_rows > 0 ? h->n_leaf_rows : 1), na = (size_t)(h->n_angles > 0 ? h->n_angles : 1);
    // scratch of the pricing step, freed on every exit path
    struct Scratch {
        float *g = nullptr, *p = nullptr, *xs = nullptr, *DA = nullptr;
        int32_t *Lw = nullptr, *Rw = nullptr, *best = nullptr, *win = nullptr;
        double *row_price = nullptr, *angle_price = nullptr, *F = nullptr;
        uint8_t *mask = nullptr;
        ~Scratch() { for (void *q : {(void *)g, (void *)p, (void *)xs, (void *)DA, (void *)Lw, (void *)Rw, (void *)best, (void *)win,
                                     (void *)row_price, (void *)angle_price, (void *)F, (void *)mask}) if (q) cudaFree(q); }
    } w;
    VMAT_CUDA(cudaMalloc((void **)&w.g, nv * 4)); VMAT_CUDA(cudaMalloc((void **)&w.DA, nv * 4));
    VMAT_CUDA(cudaMalloc((void **)&w.p, nb * 4)); VMAT_CUDA(cudaMalloc((void **)&w.xs, nb * 4));
    VMAT_CUDA(cudaMalloc((void **)&w.Lw, nr * 4)); VMAT_CUDA(cudaMalloc((void **)&w.Rw, nr * 4));
    VMAT_CUDA(cudaMalloc((void **)&w.row_price, nr * 8)); VMAT_CUDA(cudaMalloc((void **)&w.angle_price, na * 8));
    VMAT_CUDA(cudaMalloc((void **)&w.best, 4)); VMAT_CUDA(cudaMalloc((void **)&w.F, 8));
    VMAT_CUDA(cudaMalloc((void **)&w.mask, na));
    if (max_leaf_travel >= 0) VMAT_CUDA(cudaMalloc((void **)&w.win, nr * 16));              // L_lo, L_hi, R_lo, R_hi
    VMAT_CUDA(cudaMemsetAsync(w.mask, 0, na, s));
    VMAT_CUDA(cudaMemsetAsync(z, 0, nv * 4, s));                                         // L56: start with z = 0 ...
    if (h->n_leaf_rows > 0) {
        VMAT_CUDA(cudaMemsetAsync(L, 0, nr * 4, s));
        VMAT_CUDA(cudaMemsetAsync(R, 0, nr * 4, s));
    }
    { int rcf = mp_forget(mp, s); if (rcf != VMAT_OK) return rcf; }                      // ... and no apertures
    int launches = 0, count = 0, stop = 1;
    if (F_hist_host) {                                                                   // F(z = 0)
        double F0 = 0.0;
        int rc0 = vmat_launch_objective(h, z, voxel_struct, n_struct, T, w_over, w_under, w.g, w.F, s);
        if (rc0 != VMAT_OK) return rc0;
        VMAT_CUDA(cudaMemcpyAsync(&F0, w.F, 8, cudaMemcpyDeviceToHost, s));
        VMAT_CUDA(cudaStreamSynchronize(s));
        F_hist_host[0] = F0;
    }
    while (count < max_apertures) {
        // PP1: gradient at the current dose, beamlet prices; PP2: best opening per leaf row, best control point
        int rc = vmat_launch_objective(h, z, voxel_struct, n_struct, T, w_over, w_under, w.g, w.F, s);
        if (!constrained) {
            if (rc == VMAT_OK) rc = vmat_launch_price_select(h, w.g, w.mask, w.p, w.Lw, w.Rw, w.row_price, s, true);   // k not in C only (L58)
            if (rc == VMAT_OK) rc = vmat_launch_angle_price(h, w.row_price, w.mask, w.angle_price, w.best, s);
        } else {
            int32_t *wl[4] = {nullptr, nullptr, nullptr, nullptr};
            if (rc == VMAT_OK) rc = vmat_launch_price_unoccupied(h, w.g, w.mask, w.p, s);                 // k not in C only (L58)
            if (rc == VMAT_OK && max_leaf_travel >= 0) {
                for (int q = 0; q < 4; ++q) wl[q] = w.win + (size_t)q * nr;
                rc = vmat_launch_leaf_windows(h, w.mask, L, R, n_arcs, arc_angle_offset, max_leaf_travel, wl[0], wl[1],
                                              wl[2], wl[3], s);
            }
            if (rc == VMAT_OK) rc = vmat_launch_select_constrained(h, w.p, w.mask, interdigitation, wl[0], wl[1], wl[2],
                                                                   wl[3], w.Lw, w.Rw, w.row_price, w.angle_price, w.best, s);
        }
        if (rc != VMAT_OK) return rc;
        int32_t best = -1;
        double F = 0.0;
        VMAT_CUDA(cudaMemcpyAsync(&best, w.best, 4, cudaMemcpyDeviceToHost, s));
        VMAT_CUDA(cudaStreamSynchronize(s));
        launches += g_vmat_launches;
        if (best < 0) { stop = 0; break; }                                               // nothing decreases F any more
        const int32_t r0 = h->h_angle_row_offset[best], r1 = h->h_angle_row_offset[best + 1];
        if (r1 > r0) {
            VMAT_CUDA(cudaMemcpyAsync(L + r0, w.Lw + r0, (size_t)(r1 - r0) * 4, cudaMemcpyDeviceToDevice, s));
            VMAT_CUDA(cudaMemcpyAsync(R + r0, w.Rw + r0, (size_t)(r1 - r0) * 4, cudaMemcpyDeviceToDevice, s));
        }
        if (aperture_price_host)
            VMAT_CUDA(cudaMemcpyAsync(aperture_price_host + count, w.angle_price + best, 8, cudaMemcpyDeviceToHost, s));
        // Eq. (5): the aperture's dose vector; then the master problem over all apertures so far (warm start)
        rc = vmat_aperture_dose(h, best, w.Lw, w.Rw, w.xs, w.DA, s);
        launches += g_vmat_launches;
        if (rc == VMAT_OK) rc = vmat_mp_add_aperture(mp, w.DA, 0.0, y_lo, y_hi, s);
        launches += g_vmat_launches;
        if (rc != VMAT_OK) return rc;
        VMAT_CUDA(cudaMemsetAsync(w.mask + best, 1, 1, s));
        int32_t nit = 0, reason = 0;
        rc = vmat_mp_solve(mp, voxel_struct, n_struct, T, w_over, w_under, mp_max_iter, eps_F, eps_y, z, nullptr, &F,
                           &nit, &reason, s);
        launches += g_vmat_launches;
        if (rc != VMAT_OK) return rc;
        if (angles_host) angles_host[count] = best;
        if (F_hist_host) F_hist_host[count + 1] = F;
        if (mp_iters_host) mp_iters_host[count] = nit;
        ++count;
    }
    if (y_host && count > 0) VMAT_CUDA(cudaMemcpyAsync(y_host, mp->y, (size_t)count * 8, cudaMemcpyDeviceToHost, s));
    VMAT_CUDA(cudaStreamSynchronize(s));
    *n_apertures_host = count;
    if (stop_host) *stop_host = stop;
    g_vmat_launches = launches;
    return VMAT_OK;
}

int vmat_mp_reached_voxels(const vmat_mp *h, int32_t *n_reached)
{
    REQUIRE(h != nullptr && n_reached != nullptr, "NULL argument");
    REQUIRE(h->active_valid, "no solve has run since the last aperture was added");
    *n_reached = h->n_active;
    return VMAT_OK;
}

int vmat_mp_pass_geometry(const vmat_mp *h, int32_t m, int32_t *n_cta, int32_t *rows_per_grid_step)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(m >= 1 && m <= h->m_cap, "m must be in 1..max_apertures");
    // mirrors mp_launch_pass: lanes per row 2^LOG, 16-byte chunks per lane NC, rows per lane group and step 2^RBL
    const int LOG = m <= 32 ? 3 : (m <= 64 ? 4 : 5), NC = m <= 128 ? 1 : (m <= 256 ? 2 : 3);
    const int cta = h->n_sm * (m <= 256 ? 3 : 2);
    if (n_cta) *n_cta = cta;
    if (rows_per_grid_step) *rows_per_grid_step = cta * MP_WARPS * ((1 << mp_rbl(NC)) * (32 >> LOG));
    return VMAT_OK;
}

int vmat_mp_size(const vmat_mp *h, int32_t *n_apertures, int32_t *max_apertures)
{
    REQUIRE(h != nullptr, "handle is NULL");
    if (n_apertures) *n_apertures = h->m;
    if (max_apertures) *max_apertures = h->m_cap;
    return VMAT_OK;
}

}  // extern "C"
