// master.cu - NEXT-2: the master problem (MP) of the column-generation loop, Eq. (6)-(10) L70-L101
// and the four BB steps of L139: fluence rates y_k in [lo_k, hi_k] of the apertures chosen so far that minimise
// F(z), z = sum_k DA(A_k) y_k, by the Barzilai-Borwein iteration with the subspace step rule.
// Readings C15-C20: DESIGN.md section 2.
//
// Storage: DA is dense (the paper's aperture dose vectors are "dense-ish", <= 0.15 % of the DDC matrix, L264), in
// COLUMN BLOCKS of 32 apertures: float [column block][voxel][32].  A run of consecutive voxels is then one
// contiguous piece of memory per column block, whatever the capacity of the handle and however many apertures
// exist so far, and a pipeline stage of the solve kernel (R consecutive voxels) is ceil(m / 32) bulk copies of
// R x 128 bytes.  One BB iteration needs ONE pass over DA: the row dot gives z_i (step 4 of L139), the voxel's
// gradient follows (Eq. (1)), and every lane adds DA_ik * dF/dz_i to its own entries of the aperture gradient g_A
// (step 1) - no second read, no atomics.  HBM-bound: 4 m n_reached bytes per iteration.  Only BLOCKS of R
// consecutive voxels of which some aperture reaches at least one are visited.
// All sums are FP64 in a fixed order (FP32 storage of DA, T, weights): deterministic, and a trajectory differs
// from the FP64 oracle's by summation order only.
#include "common.cuh"
#include <cooperative_groups.h>
#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>
#include <new>
#include <stdlib.h>
#include <vector>

constexpr int MP_THREADS = 512;             // ONE persistent CTA per SM, 16 warps
constexpr int MP_WARPS = MP_THREADS / 32;
constexpr int MP_MAX_NC = 12;                 // up to 12 x 32 = 384 apertures
constexpr int MP_MAX_M = MP_MAX_NC * 32;
constexpr int MP_HIST = 6;                    // objective values the "last five changes" rule looks at

struct MpState {                              // device-resident scalars of one solve (written once, when it stops)
    int it;                                   // iterations done
    int reason;                               // 1 stationary, 2 objective, 3 step, 4 max_iter (C19)
    double delta;                             // last step size
    double F;                                 // objective at the returned iterate
};

struct vmat_mp {
    int32_t n_voxels = 0, m_cap = 0, m = 0;
    int64_t n_vox_pad = 0;                    // voxels rounded up to a multiple of 16 (rows beyond n_voxels stay 0)
    int n_cta = 0, n_sm = 0, device = 0;      // n_cta: CTAs of the solve kernel = SMs (one persistent CTA each)
    float *DA = nullptr;                      // [ceil(m_cap / 32)][n_vox_pad][32]
    double *y = nullptr, *g = nullptr, *lo = nullptr, *hi = nullptr;   // [m_cap]
    double *gpart = nullptr;                  // [m_cap][n_cta] per-CTA partials of g_A
    double *gsum = nullptr;                   // [m_cap] g_A of the current iterate, after the subspace rule
    double *spart = nullptr;                  // [n_cta][2]: F partial, curvature partial
    MpState *st = nullptr;
    double *F_hist = nullptr, *delta_hist = nullptr;   // [hist_cap + 1]
    int32_t hist_cap = 0;
    int32_t last_n_iter = 0;
    // the voxels some aperture reaches (rows of DA with a non-zero), and the blocks of R consecutive voxels that
    // hold at least one of them: only those blocks are visited by the passes
    uint8_t *row_flag = nullptr;              // [n_voxels] set by vmat_mp_add_aperture
    uint8_t *blk_flag = nullptr;              // [n_vox_pad / 2] per block of active_R voxels
    int32_t *active = nullptr;                // [n_vox_pad / 2] indices of the flagged blocks, ascending
    int32_t *n_active_dev = nullptr;          // [2]: flagged blocks, reached voxels
    void *select_tmp = nullptr;               // scratch of the compaction
    size_t select_tmp_bytes = 0;
    int32_t n_active = 0;                     // flagged blocks
    int32_t n_reached = 0;                    // reached voxels
    int32_t active_R = 0;                     // block size the list was built for; 0 = stale
    double *upart = nullptr;                  // [n_cta] partials of F over the voxels outside the flagged blocks
    double *stage3 = nullptr;                 // pinned host [3]: y0, lo, hi of the aperture being added
    cudaEvent_t stage3_free = nullptr;        // recorded after the copies that read stage3
    // scratch of the column-generation loop (allocated on first use, sized by the DDC handle it ran with)
    void *cg_scratch = nullptr;
    size_t cg_scratch_bytes = 0;
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

// column k of DA; a voxel that any aperture reaches is flagged: only blocks with such a voxel are ever read again
__global__ void k_mp_set_column(int n_voxels, int64_t n_vox_pad, int k, const float *__restrict__ col,
                                float *__restrict__ DA, uint8_t *__restrict__ row_flag)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_voxels) {
        const float v = col[i];
        DA[((size_t)(k >> 5) * n_vox_pad + i) * 32 + (k & 31)] = v;
        if (v != 0.f) row_flag[i] = 1;
    }
}

// flags of the blocks of R consecutive voxels (R = 4, 8 or 16) that hold a reached voxel; counts the reached voxels
__global__ void k_mp_block_flags(int n_voxels, int R, const uint8_t *__restrict__ row_flag, uint8_t *__restrict__ blk_flag,
                                 int32_t *__restrict__ n_reached)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    int cnt = 0;
    if ((int64_t)b * R < n_voxels) {
        for (int r = 0; r < R; ++r) {
            const int64_t i = (int64_t)b * R + r;
            if (i < n_voxels && row_flag[i]) ++cnt;
        }
        blk_flag[b] = cnt > 0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(n_reached, cnt);      // integer: order-free
}

// ---------------------------------------------------------------- the whole BB solve: one persistent kernel
// One CTA of 16 warps per SM, launched cooperatively; the BB iteration (the four steps of L139) runs on the device
// until a stopping rule fires.  Per iteration:
//   pass    z = DA y, F, dF/dz, per-CTA partials of g_A = DA^T dF/dz (steps 4 and 1), DA read from HBM once;
//   sync    grid barrier;
//   reduce  one warp per aperture sums that aperture's partials in a fixed order, applies the subspace rule
//           Eq. (9)/(10) with the sign of C15, publishes g_A;
//   sync    grid barrier;
//   step    EVERY CTA forms F, the stopping rules (C19), the step size Eq. (7)/(8) (C17 at iteration 0, after one
//           extra "curvature" pass) and the clipped update of y from the same published numbers by the same
//           instructions in the same order, so all CTAs hold bit-identical y, y_prev, g_prev in their own shared
//           memory and agree on when to stop; CTA 0 alone writes the trace and the result.
// No kernel launch and no host round trip per iteration (the first version launched a pass and a one-CTA step kernel
// per iteration and let the host look at the stop flag every 8: 61 us per launch on average over a plan).
//
// The pass.  A warp owns one flagged block of R consecutive voxels per pipeline stage, prefetched STAGES - 1 stages
// ahead by 1-D bulk copies (cp.async.bulk, SASS UBLKCP: one per column block, R x 128 contiguous bytes each, issued
// by different lanes; completion counted in bytes on the stage's mbarrier): no per-lane address arithmetic, no
// registers held across the flight.  LZ lanes share a row, each CZ 16-byte chunks interleaved by LZ; an entry is
// converted to FP64 ONCE (F2F runs on the 16-lane XU pipe: converting twice made it the busiest pipe), the row dot
// needs log2(LZ) plain shuffle steps for 32 / LZ rows at once, every lane of the row then forms dF/dz_i itself and
// adds DA_ik dF/dz_i to the accumulators of ITS columns from the same registers; the row groups of a warp and the
// warps are summed once per pass.  The block indices and structure ids a stage needs are loaded when the stage is
// ISSUED and ride along in registers: a load on the critical path would queue behind the whole bulk stream.
// ~30 warp instructions per 512 bytes of DA instead of 64 (ncu: profiles/r2_mp_solve.md).
// All sums are FP64 in a fixed order given (m, SM count): deterministic.
template <int V> struct MpCfg;
//                                    column blocks of 32 | lanes per row, 16-byte chunks per lane | voxels per block
//                                    (= rows per stage) | stages
template <> struct MpCfg<0> { static constexpr int NCB = 1,  LZ = 2,  CZ = 4, R = 16, STAGES = 4; };
template <> struct MpCfg<1> { static constexpr int NCB = 2,  LZ = 4,  CZ = 4, R = 8,  STAGES = 4; };
template <> struct MpCfg<2> { static constexpr int NCB = 4,  LZ = 8,  CZ = 4, R = 8,  STAGES = 3; };
template <> struct MpCfg<3> { static constexpr int NCB = 8,  LZ = 16, CZ = 4, R = 4,  STAGES = 3; };
template <> struct MpCfg<4> { static constexpr int NCB = 12, LZ = 32, CZ = 3, R = 4,  STAGES = 2; };
static inline int mp_variant(int m) { return m <= 32 ? 0 : (m <= 64 ? 1 : (m <= 128 ? 2 : (m <= 256 ? 3 : 4))); }
template <int V> __host__ __device__ constexpr size_t mp_ring_bytes()
{
    return (size_t)MP_WARPS * MpCfg<V>::STAGES * MpCfg<V>::R * MpCfg<V>::NCB * 128;
}
template <int V> __host__ __device__ constexpr size_t mp_accs_bytes() { return (size_t)MP_WARPS * (MpCfg<V>::NCB * 32) * 8; }
template <int V> __host__ __device__ constexpr size_t mp_ring_alloc()   // the FP64 accumulators of a CTA reuse the ring
{
    return mp_ring_bytes<V>() > mp_accs_bytes<V>() ? mp_ring_bytes<V>() : mp_accs_bytes<V>();
}
template <int V> __host__ __device__ constexpr size_t mp_smem_bytes() { return mp_ring_alloc<V>() + (size_t)MP_WARPS * MpCfg<V>::STAGES * 8; }

struct MpArgs {
    int n;                      // flagged blocks to visit
    const int32_t *active;      // their indices, ascending (block b = voxels b R .. b R + R - 1)
    int n_voxels;
    int64_t n_vox_pad;
    int m;
    const float *DA;
    double *y, *g;              // in: start; out: returned iterate and its g_A after the subspace rule
    const double *lo, *hi;
    const uint8_t *vstruct;
    int sid_aligned;            // vstruct is 16-byte aligned: the structure ids of a block can travel by cp.async
    int n_struct;
    const float *T, *w_over, *w_under;
    float *z_out;               // or NULL
    double *gpart, *spart, *gsum;
    MpState *st;
    double *F_hist, *delta_hist;
    const uint8_t *blk_flag;    // per block of R voxels: visited by the passes
    double *upart;              // [n_cta] partials of F over the voxels outside the flagged blocks
    int max_iter;
    double eps_F, eps_y;
};

__device__ __forceinline__ uint32_t mp_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mp_mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mp_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mp_mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
// 1-D bulk copy global -> shared (the TMA unit; SASS UBLKCP), completion in bytes on an mbarrier
// L2 policy: DA is far larger than L2 and read once per pass -> evict_first, so that the small per-row tables
// (evict_last) stay L2-resident from pass to pass; a table load that misses queues behind the whole bulk stream.
__device__ __forceinline__ void mp_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ uint64_t mp_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t mp_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ int mp_ld_keep_i32(const int32_t *p, uint64_t pol)
{
    int r;
    asm volatile("ld.global.nc.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ uint32_t mp_ld_keep_u8(const uint8_t *p, uint64_t pol)
{
    uint32_t r;
    asm volatile("ld.global.nc.L2::cache_hint.u8 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ void mp_fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ float4 mp_lds128(uint32_t addr)
{
    float4 e;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(e.x), "=f"(e.y), "=f"(e.z), "=f"(e.w) : "r"(addr));
    return e;
}

template <int BYTES>
__device__ __forceinline__ void mp_cp_async(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" :: "r"(dst), "l"(src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void mp_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void mp_cp_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void mp_sts_u8(uint32_t dst, uint8_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" :: "r"(dst), "r"((uint32_t)v) : "memory");
}
__device__ __forceinline__ uint32_t mp_lds_u8(uint32_t addr)
{
    uint32_t r;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}

// per-warp pipeline bookkeeping that lives across the passes of a solve
struct MpPipe {
    uint32_t phases;            // bit s: parity the next wait on stage s must see
    int cstage;                 // next stage to consume
};

// One pass over the flagged blocks.  CURV = false: z = DA y, F, dF/dz, g_A partials (acc).  CURV = true: z = DA y,
// q = DA v, sum_i w_i q_i^2 (C17).  ssum: this thread's part of F (or of the curvature).
// sT2: per structure {T, 2 w_over, 2 w_under} in FP64.
template <int V, bool CURV>
__device__ __forceinline__ void mp_pass(const MpArgs &a, uint32_t ring_w, uint32_t bar_w, uint32_t sid_w, MpPipe &pp, const double *sy,
                                        const double *sv, const double *sT2, double (&acc)[MpCfg<V>::CZ][4], double &ssum)
{
    using C = MpCfg<V>;
    constexpr int LZ = C::LZ, CZ = C::CZ, R = C::R, STAGES = C::STAGES, NCB = C::NCB;
    constexpr int CB_BYTES = R * 128, STAGE_BYTES = NCB * CB_BYTES;
    constexpr int RZ = 32 / LZ, NSUB = R / RZ;
    static_assert(R % RZ == 0 && NSUB >= 1 && NSUB <= 4 && LZ * CZ == NCB * 8 && NCB <= 32, "mapping");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rz = lane / LZ, qz = lane % LZ;
    const int n = a.n;
    const int ncb = (a.m + 31) >> 5;                              // column blocks that hold apertures
    const int step = gridDim.x * MP_WARPS;
    int pos = blockIdx.x * MP_WARPS + warp;                       // position in the list of flagged blocks
    double yz[CZ][4];                                             // y of this lane's columns
#pragma unroll
    for (int j = 0; j < CZ; ++j)
#pragma unroll
        for (int k = 0; k < 4; ++k) yz[j][k] = sy[(j * LZ + qz) * 4 + k];   // 0 beyond m
    const uint64_t pol_stream = mp_policy_evict_first(), pol_keep = mp_policy_evict_last();
    // lane part of the shared-memory offset of this lane's chunks of row rz: chunk c = j LZ + qz lies in column
    // block c / 8 at 16-byte slot c % 8
    const uint32_t lane_off = (uint32_t)((qz >> 3) * CB_BYTES + (qz & 7) * 16 + rz * 128);
    // Block indices: lane l holds the index of the block this warp takes l steps after the start of the current batch
    // of 32 steps; the next batch is loaded 32 steps before its first use, so no step ever waits for such a load
    // (a load on the critical path would queue behind the whole bulk stream).  Structure ids: R bytes per block,
    // copied by cp.async into the stage's slot of a small shared-memory FIFO when the stage is issued.
    auto load_batch = [&](int p0) {
        const int64_t p = (int64_t)p0 + (int64_t)lane * step;
        return p < n ? mp_ld_keep_i32(a.active + p, pol_keep) : 0;
    };
    int batch_cur = load_batch(pos), batch_next = load_batch(pos + 32 * step);
    int bi = 0;                                                   // steps issued out of batch_cur
    int blk_q[STAGES];                                            // block indices of the stages in flight, oldest first
#pragma unroll
    for (int q = 0; q < STAGES; ++q) blk_q[q] = 0;
    int istage = pp.cstage;
    int ipos = pos;
    auto issue = [&]() {                                          // the block at list position ipos
        const int blk = __shfl_sync(0xffffffffu, batch_cur, bi);
        if (++bi == 32) {
            bi = 0;
            batch_cur = batch_next;
            batch_next = load_batch(ipos + step + 32 * step);
        }
        if (ipos < n) {
            const uint32_t bar = bar_w + 8u * istage;
            if (lane == 0) {
                mp_mbar_expect_tx(bar, (uint32_t)(ncb * CB_BYTES));
                const int nb = min(R, a.n_voxels - blk * R);      // the volume may end inside the last block
                if (nb == R && a.sid_aligned) mp_cp_async<R>(sid_w + (uint32_t)(istage * 16), a.vstruct + (size_t)blk * R);
                else for (int r = 0; r < nb; ++r) mp_sts_u8(sid_w + (uint32_t)(istage * 16 + r), a.vstruct[(size_t)blk * R + r]);
            }
            __syncwarp();
            if (lane < ncb)
                mp_bulk_g2s(ring_w + (uint32_t)(istage * STAGE_BYTES + lane * CB_BYTES),
                            a.DA + ((size_t)lane * a.n_vox_pad + (size_t)blk * R) * 32, CB_BYTES, bar, pol_stream);
        }
        mp_cp_commit();
#pragma unroll
        for (int q = 0; q < STAGES - 1; ++q) blk_q[q] = blk_q[q + 1];
        blk_q[STAGES - 1] = blk;
        ipos += step;
        if (++istage == STAGES) istage = 0;
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) issue();
#pragma unroll 1
    for (; pos < n; pos += step) {
        __syncwarp();                                             // every lane is done with the slot refilled now
        issue();
        const int blk = blk_q[0];                                 // the stage consumed now was issued STAGES - 1 steps ago
        const int cs = pp.cstage;
        mp_cp_wait<STAGES - 1>();                                 // lane 0: this stage's structure ids have landed
        __syncwarp();
        mp_mbar_wait(bar_w + 8u * cs, (pp.phases >> cs) & 1u);
        pp.phases ^= 1u << cs;
        if (++pp.cstage == STAGES) pp.cstage = 0;
        const uint32_t stg = ring_w + (uint32_t)(cs * STAGE_BYTES) + lane_off;
#pragma unroll
        for (int u = 0; u < NSUB; ++u) {
            // ---- row u RZ + rz of the block: this lane's CZ chunks, converted to FP64 once
            double e[CZ][4];
            double z4[4] = {0.0, 0.0, 0.0, 0.0}, q4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int j = 0; j < CZ; ++j) {
                const float4 f = mp_lds128(stg + (uint32_t)(u * RZ * 128 + ((j * LZ) >> 3) * CB_BYTES + ((j * LZ) & 7) * 16));
                e[j][0] = (double)f.x; e[j][1] = (double)f.y; e[j][2] = (double)f.z; e[j][3] = (double)f.w;
#pragma unroll
                for (int k = 0; k < 4; ++k) z4[k] = fma(e[j][k], yz[j][k], z4[k]);
                if (CURV) {
                    const double *v = sv + (j * LZ + qz) * 4;
#pragma unroll
                    for (int k = 0; k < 4; ++k) q4[k] = fma(e[j][k], v[k], q4[k]);
                }
            }
            double zs = (z4[0] + z4[1]) + (z4[2] + z4[3]), qs = (q4[0] + q4[1]) + (q4[2] + q4[3]);
#pragma unroll
            for (int o = LZ / 2; o > 0; o >>= 1) {                // every lane of the row ends with the row's sums
                zs += shfl_xor_d(zs, o);
                if (CURV) qs += shfl_xor_d(qs, o);
            }
            // ---- the voxel's term of F and dF/dz (Eq. (1), sign C1): with u = z - T and w2 = 2 w_over (u > 0) or
            //      2 w_under, dF/dz = w2 u and the term is w2 u^2 / 2
            const int vox = blk * R + u * RZ + rz;
            const bool live = vox < a.n_voxels;                   // the last block may reach beyond the volume
            const double *tp = sT2 + 3 * mp_lds_u8(sid_w + (uint32_t)(cs * 16 + u * RZ + rz));
            const double du = zs - tp[0];
            const double w2 = du > 0.0 ? tp[1] : tp[2];
            double gz = 0.0;
            if (live) {
                if (!CURV) {
                    gz = w2 * du;
                    if (qz == 0) {
                        ssum = fma(0.5 * gz, du, ssum);
                        if (a.z_out) a.z_out[vox] = (float)zs;
                    }
                } else if (qz == 0) {
                    ssum = fma(du != 0.0 ? 0.5 * w2 : 0.0, qs * qs, ssum);   // C17
                }
            }
            if (!CURV) {                                          // g_A += DA_i: * dF/dz_i, same lanes, same registers
#pragma unroll
                for (int j = 0; j < CZ; ++j)
#pragma unroll
                    for (int k = 0; k < 4; ++k) acc[j][k] = fma(e[j][k], gz, acc[j][k]);
            }
        }
    }
}

template <int V>
__global__ void __launch_bounds__(MP_THREADS, 1)
k_mp_solve(const MpArgs a)
{
    using C = MpCfg<V>;
    constexpr int LZ = C::LZ, CZ = C::CZ, STAGES = C::STAGES, COLS = C::NCB * 32;
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    extern __shared__ __align__(128) unsigned char mp_dyn[];      // ring [warp][stage][column block][row][128 B]; then the barriers
    __shared__ double red_s[MP_WARPS + 1];
    __shared__ double sy[MP_MAX_M], syp[MP_MAX_M], sg[MP_MAX_M], sgp[MP_MAX_M];
    __shared__ double sT2[3 * 256];
    __shared__ double sFh[MP_HIST];
    __shared__ int s_flag;
    __shared__ __align__(16) uint8_t s_sid[MP_WARPS][4][16];      // structure ids of the blocks in flight, per warp and stage
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, qz = lane % LZ;
    const int m = a.m, n_cta = gridDim.x;
    constexpr size_t RING = mp_ring_alloc<V>();
    uint64_t *bars = (uint64_t *)(mp_dyn + RING);
    for (int t = tid; t < (int)(RING / 16); t += MP_THREADS) ((float4 *)mp_dyn)[t] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int t = tid; t < a.n_struct; t += MP_THREADS) {
        sT2[3 * t] = (double)a.T[t]; sT2[3 * t + 1] = 2.0 * (double)a.w_over[t]; sT2[3 * t + 2] = 2.0 * (double)a.w_under[t];
    }
    for (int k = tid; k < MP_MAX_M; k += MP_THREADS) {
        sy[k] = k < m ? fmin(fmax(a.y[k], a.lo[k]), a.hi[k]) : 0.0;          // the start must be feasible (C16)
        syp[k] = 0.0; sg[k] = 0.0; sgp[k] = 0.0;
    }
    {   // F of the voxels outside the flagged blocks (z_i = 0 whatever y): their terms of Eq. (1) at z = 0, this CTA's
        // slice of the volume; summed over the CTAs in a fixed order after the first grid barrier
        const int per = (a.n_voxels + n_cta - 1) / n_cta, i0 = blockIdx.x * per, i1 = min(a.n_voxels, i0 + per);
        double us = 0.0;
        for (int i = i0 + tid; i < i1; i += MP_THREADS)
            if (!a.blk_flag[i / C::R]) {
                const int sid = a.vstruct[i];
                const double Ti = (double)a.T[sid], over = fmax(0.0 - Ti, 0.0), under = fmax(Ti - 0.0, 0.0);
                us += (double)a.w_over[sid] * over * over + (double)a.w_under[sid] * under * under;
            }
        const double tot = mp_block_sum(us, red_s);
        if (tid == 0) a.upart[blockIdx.x] = tot;
    }
    if (tid < MP_WARPS * STAGES) mp_mbar_init(mp_smem_u32(bars + tid), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mp_fence_async_proxy();
    __syncthreads();
    const uint32_t ring_w = mp_smem_u32(mp_dyn) + (uint32_t)(warp * STAGES * C::R * C::NCB * 128);
    const uint32_t bar_w = mp_smem_u32(bars + warp * STAGES);
    const uint32_t sid_w = mp_smem_u32(&s_sid[warp][0][0]);
    MpPipe pp = {0u, 0};
    int it = 0, reason = 0;
    double delta = 0.0, F = 0.0, F_unreached = 0.0;
    for (;;) {
        // ---- steps 4 + 1 of L139: the gradient pass
        double acc[CZ][4];
#pragma unroll
        for (int j = 0; j < CZ; ++j)
#pragma unroll
            for (int k = 0; k < 4; ++k) acc[j][k] = 0.0;
        double ssum = 0.0;
        mp_pass<V, false>(a, ring_w, bar_w, sid_w, pp, sy, sg, sT2, acc, ssum);
        // CTA partials in a fixed order: the row groups of a warp, then the warps (in the ring's memory, idle now)
        __syncthreads();
        double *accs = (double *)mp_dyn;                          // [MP_WARPS][COLS]
#pragma unroll
        for (int j = 0; j < CZ; ++j)
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                double v = acc[j][k];
#pragma unroll
                for (int o = LZ; o < 32; o <<= 1) v += shfl_xor_d(v, o);
                if (lane < LZ) accs[warp * COLS + (j * LZ + qz) * 4 + k] = v;
            }
        __syncthreads();
        for (int k = tid; k < m; k += MP_THREADS) {
            double sacc = 0.0;
            for (int w = 0; w < MP_WARPS; ++w) sacc += accs[w * COLS + k];
            a.gpart[(size_t)k * n_cta + blockIdx.x] = sacc;       // [m_cap][n_cta]
        }
        {
            const double tot = mp_block_sum(ssum, red_s);
            if (tid == 0) a.spart[2 * blockIdx.x] = tot;
        }
        // the accumulators overwrote bytes the passes rely on to be zero (beyond a row's apertures): restore, then
        // hand the ring back to the async proxy
        __syncthreads();
        for (int t = tid; t < (int)(mp_accs_bytes<V>() / 16); t += MP_THREADS) ((float4 *)mp_dyn)[t] = make_float4(0.f, 0.f, 0.f, 0.f);
        mp_fence_async_proxy();
        grid.sync();
        // ---- g_A = sum of the CTA partials (one warp per aperture, fixed order), subspace rule Eq. (9)/(10), C15
        for (int k = blockIdx.x * MP_WARPS + warp; k < m; k += n_cta * MP_WARPS) {
            const double *col = a.gpart + (size_t)k * n_cta;
            double s = 0.0;
            for (int c0 = lane; c0 < n_cta; c0 += 32) s += __ldcg(col + c0);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += shfl_xor_d(s, o);
            const double yk = sy[k];
            if ((yk <= a.lo[k] && s > 0.0) || (yk >= a.hi[k] && s < 0.0)) s = 0.0;
            if (lane == 0) a.gsum[k] = s;
        }
        {                                                         // F: every CTA, same order
            double fs = 0.0;
            for (int c = tid; c < n_cta; c += MP_THREADS) fs += __ldcg(a.spart + 2 * c);
            if (it == 0) {
                double us = 0.0;
                for (int c = tid; c < n_cta; c += MP_THREADS) us += __ldcg(a.upart + c);
                F_unreached = mp_block_sum(us, red_s);
            }
            F = mp_block_sum(fs, red_s) + F_unreached;
        }
        grid.sync();
        // ---- every CTA: stopping rules (C19), tested at the top of the iteration
        int nonzero = 0;
        double dy_max = 0.0;
        for (int k = tid; k < m; k += MP_THREADS) {
            const double gk = __ldcg(a.gsum + k);
            sg[k] = gk;
            nonzero |= gk != 0.0;
            if (it >= 1) dy_max = fmax(dy_max, fabs(sy[k] - syp[k]));
        }
        if (tid == 0) s_flag = 0;
        __syncthreads();
        if (nonzero) atomicOr(&s_flag, 1);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dy_max = fmax(dy_max, shfl_xor_d(dy_max, o));   // max: exact, order-free
        __syncthreads();
        if (lane == 0) red_s[warp] = dy_max;
        __syncthreads();
        if (tid == 0) {
            for (int i = 0; i < MP_WARPS; ++i) dy_max = fmax(dy_max, red_s[i]);
            for (int j = MP_HIST - 1; j > 0; --j) sFh[j] = sFh[j - 1];
            sFh[0] = F;
            int r = 0;
            if (!s_flag) r = 1;
            else {
                bool flat = it >= 5;
                for (int j = 0; flat && j < 5; ++j) flat = fabs(sFh[j] - sFh[j + 1]) <= a.eps_F * fabs(sFh[j + 1]);
                if (flat) r = 2;
                else if (it >= 1 && dy_max <= a.eps_y) r = 3;
                else if (it >= a.max_iter) r = 4;
            }
            s_flag = r;
            if (blockIdx.x == 0) a.F_hist[it] = F;
        }
        __syncthreads();
        reason = s_flag;
        __syncthreads();
        if (reason != 0) break;
        // ---- step 2: the step size
        if (it == 0) {                                            // C17: one more pass, q = DA g_A
            double csum = 0.0;
            mp_pass<V, true>(a, ring_w, bar_w, sid_w, pp, sy, sg, sT2, acc, csum);
            const double tot = mp_block_sum(csum, red_s);
            if (tid == 0) a.spart[2 * blockIdx.x + 1] = tot;
            grid.sync();
            double cs = 0.0, gg = 0.0;
            for (int c = tid; c < n_cta; c += MP_THREADS) cs += __ldcg(a.spart + 2 * c + 1);
            for (int k = tid; k < m; k += MP_THREADS) gg += sg[k] * sg[k];
            const double den = 2.0 * mp_block_sum(cs, red_s);
            const double num = mp_block_sum(gg, red_s);
            delta = den > 0.0 ? num / den : 1.0;
        } else {                                                  // Eq. (7) odd iterations, Eq. (8) even ones (C18)
            double ss = 0.0, st = 0.0, tt = 0.0;
            for (int k = tid; k < m; k += MP_THREADS) {
                const double s = sy[k] - syp[k], t = sg[k] - sgp[k];
                ss += s * s; st += s * t; tt += t * t;
            }
            ss = mp_block_sum(ss, red_s);
            st = mp_block_sum(st, red_s);
            tt = mp_block_sum(tt, red_s);
            if (st > 0.0 && tt > 0.0) delta = (it & 1) ? ss / st : st / tt;   // else: the previous delta is kept
        }
        // ---- step 3: update within the box (C16)
        for (int k = tid; k < m; k += MP_THREADS) {
            const double yk = sy[k], gk = sg[k];
            syp[k] = yk;
            sgp[k] = gk;
            sy[k] = fmin(fmax(yk - delta * gk, a.lo[k]), a.hi[k]);
        }
        if (blockIdx.x == 0 && tid == 0) a.delta_hist[it] = delta;
        ++it;
        __syncthreads();
    }
    if (blockIdx.x == 0) {                                        // the iterate at which the rule fired
        for (int k = tid; k < m; k += MP_THREADS) { a.y[k] = sy[k]; a.g[k] = sg[k]; }
        if (tid == 0) { a.st->it = it; a.st->reason = reason; a.st->delta = delta; a.st->F = F; }
    }
}

// ---------------------------------------------------------------- host side
template <int V>
static cudaError_t mp_launch_solve_v(const vmat_mp *h, const MpArgs &a, cudaStream_t s)
{
    void *args[] = {(void *)&a};
    return cudaLaunchCooperativeKernel((const void *)k_mp_solve<V>, dim3(h->n_cta), dim3(MP_THREADS), args, mp_smem_bytes<V>(), s);
}
static cudaError_t mp_launch_solve(const vmat_mp *h, const MpArgs &a, cudaStream_t s)
{
    switch (mp_variant(a.m)) {
    case 0: return mp_launch_solve_v<0>(h, a, s);
    case 1: return mp_launch_solve_v<1>(h, a, s);
    case 2: return mp_launch_solve_v<2>(h, a, s);
    case 3: return mp_launch_solve_v<3>(h, a, s);
    default: return mp_launch_solve_v<4>(h, a, s);
    }
}
static int mp_rows_per_stage(int m)
{
    switch (mp_variant(m)) {
    case 0: return MpCfg<0>::R;
    case 1: return MpCfg<1>::R;
    case 2: return MpCfg<2>::R;
    case 3: return MpCfg<3>::R;
    default: return MpCfg<4>::R;
    }
}
// dynamic shared memory of every variant; true if one CTA of each fits an SM
static bool mp_prepare_kernels()
{
    bool ok = true;
#define MP_PREP(V)                                                                                                    \
    {                                                                                                                 \
        ok = ok && cudaFuncSetAttribute(k_mp_solve<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mp_smem_bytes<V>()) == cudaSuccess; \
        int nb = 0;                                                                                                   \
        ok = ok && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_mp_solve<V>, MP_THREADS, mp_smem_bytes<V>()) == cudaSuccess && nb >= 1; \
    }
    MP_PREP(0) MP_PREP(1) MP_PREP(2) MP_PREP(3) MP_PREP(4)
#undef MP_PREP
    return ok;
}

#define REQUIRE(cond, msg)                                            \
    do {                                                              \
        if (!(cond)) { vmat_set_error("%s: %s", __func__, msg); return VMAT_ERR_INVALID_ARG; } \
    } while (0)

extern "C" {

int vmat_mp_destroy(vmat_mp *h)
{
    if (!h) return VMAT_OK;
    void *ptrs[] = {h->DA, h->y, h->g, h->lo, h->hi, h->gpart, h->spart, h->gsum, h->st, h->F_hist,
                    h->delta_hist, h->row_flag, h->blk_flag, h->active, h->n_active_dev, h->select_tmp, h->upart,
                    h->cg_scratch};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    if (h->stage3) cudaFreeHost(h->stage3);
    if (h->stage3_free) cudaEventDestroy(h->stage3_free);
    delete h;
    return VMAT_OK;
}

int vmat_mp_create(vmat_mp **out, int32_t n_voxels, int32_t max_apertures, void *stream)
{
    REQUIRE(out != nullptr, "out is NULL");
    REQUIRE(n_voxels >= 0, "negative n_voxels");
    REQUIRE(max_apertures >= 1 && max_apertures <= MP_MAX_M, "max_apertures must be in 1..384");
    vmat_mp *h = new (std::nothrow) vmat_mp();
    if (!h) { vmat_set_error("vmat_mp_create: host allocation failed"); return VMAT_ERR_OOM; }
    h->n_voxels = n_voxels;
    h->m_cap = (max_apertures + 7) / 8 * 8;
    h->n_vox_pad = ((int64_t)n_voxels + 15) / 16 * 16;       // whole voxel blocks of every size (4, 8, 16)
    cudaGetDevice(&h->device);
    int n_sm = 1, coop = 0;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, h->device);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
    if (!coop || !mp_prepare_kernels()) {
        cudaGetLastError();
        delete h;
        vmat_set_error("vmat_mp_create: the device cannot hold one cooperative CTA of the solve kernel per SM");
        return VMAT_ERR_CUDA;
    }
    h->n_sm = n_sm;
    h->n_cta = n_sm;                                          // one persistent CTA per SM
    cudaStream_t s = (cudaStream_t)stream;
    auto alloc = [&](void **p, size_t bytes) { return cudaMalloc(p, bytes > 0 ? bytes : 1) == cudaSuccess; };
    const size_t mc = (size_t)h->m_cap;
    const size_t da_bytes = (size_t)((h->m_cap + 31) / 32) * (size_t)h->n_vox_pad * 128;
    const size_t nblk_max = (size_t)(h->n_vox_pad / 4);       // the smallest blocks hold 4 voxels
    bool ok = alloc((void **)&h->DA, da_bytes) && alloc((void **)&h->y, mc * 8) &&
              alloc((void **)&h->g, mc * 8) && alloc((void **)&h->gsum, mc * 8) &&
              alloc((void **)&h->lo, mc * 8) && alloc((void **)&h->hi, mc * 8) &&
              alloc((void **)&h->gpart, (size_t)h->n_cta * mc * 8) && alloc((void **)&h->spart, (size_t)h->n_cta * 16) &&
              alloc((void **)&h->st, sizeof(MpState)) && alloc((void **)&h->row_flag, (size_t)n_voxels) &&
              alloc((void **)&h->blk_flag, nblk_max) &&
              alloc((void **)&h->active, nblk_max * 4) && alloc((void **)&h->n_active_dev, 8) &&
              alloc((void **)&h->upart, (size_t)h->n_cta * 8) &&
              cudaMallocHost((void **)&h->stage3, 3 * sizeof(double)) == cudaSuccess &&
              cudaEventCreateWithFlags(&h->stage3_free, cudaEventDisableTiming) == cudaSuccess;
    if (ok) {
        cub::DeviceSelect::Flagged(nullptr, h->select_tmp_bytes, thrust::counting_iterator<int32_t>(0), h->blk_flag, h->active,
                                   h->n_active_dev, (int)nblk_max, s);
        ok = alloc(&h->select_tmp, h->select_tmp_bytes);
    }
    if (!ok) {
        cudaGetLastError();
        vmat_mp_destroy(h);
        vmat_set_error("vmat_mp_create: device allocation failed (%lld voxels x %d apertures)", (long long)n_voxels, h->m_cap);
        return VMAT_ERR_OOM;
    }
    cudaMemsetAsync(h->DA, 0, da_bytes, s);
    cudaMemsetAsync(h->row_flag, 0, (size_t)(n_voxels > 0 ? n_voxels : 1), s);
    cudaMemsetAsync(h->y, 0, mc * 8, s);
    cudaMemsetAsync(h->spart, 0, (size_t)h->n_cta * 16, s);
    cudaEventRecord(h->stage3_free, s);
    VMAT_CUDA(cudaStreamSynchronize(s));
    *out = h;
    return VMAT_OK;
}

// forgets the apertures and the reached-voxel flags (on stream s)
static int mp_forget(vmat_mp *h, cudaStream_t s)
{
    h->m = 0;
    h->active_R = 0;
    if (h->n_voxels > 0) VMAT_CUDA(cudaMemsetAsync(h->row_flag, 0, (size_t)h->n_voxels, s));
    return VMAT_OK;
}

int vmat_mp_reset(vmat_mp *h, void *stream)
{
    REQUIRE(h != nullptr, "handle is NULL");
    return mp_forget(h, (cudaStream_t)stream);               // ordered on the caller's stream like every other call
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
        k_mp_set_column<<<(h->n_voxels + 255) / 256, 256, 0, s>>>(h->n_voxels, h->n_vox_pad, k, DA, h->DA, h->row_flag);
        h->active_R = 0;
        VMAT_LAUNCH_CHECK();
    }
    // y0 / lo / hi through the handle's pinned staging buffer: wait (normally not at all) until the copies of the
    // previous aperture have read it, no synchronisation with the stream otherwise
    VMAT_CUDA(cudaEventSynchronize(h->stage3_free));
    h->stage3[0] = y0 < y_lo ? y_lo : (y0 > y_hi ? y_hi : y0);
    h->stage3[1] = y_lo;
    h->stage3[2] = y_hi;
    VMAT_CUDA(cudaMemcpyAsync(h->y + k, h->stage3 + 0, 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaMemcpyAsync(h->lo + k, h->stage3 + 1, 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaMemcpyAsync(h->hi + k, h->stage3 + 2, 8, cudaMemcpyHostToDevice, s));
    VMAT_CUDA(cudaEventRecord(h->stage3_free, s));
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
    // the blocks of R consecutive voxels (R by the kernel variant m selects) with a voxel some aperture reaches,
    // ascending; F of the voxels outside them (their dose is 0 whatever y)
    const int R = mp_rows_per_stage(h->m);
    if (h->active_R != R) {
        h->n_active = h->n_reached = 0;
        if (h->n_voxels > 0) {
            const int nblk = (int)(((int64_t)h->n_voxels + R - 1) / R);
            VMAT_CUDA(cudaMemsetAsync(h->n_active_dev, 0, 8, s));
            k_mp_block_flags<<<(nblk + 255) / 256, 256, 0, s>>>(h->n_voxels, R, h->row_flag, h->blk_flag, h->n_active_dev + 1);
            VMAT_LAUNCH_CHECK();
            size_t tb = h->select_tmp_bytes;
            VMAT_CUDA(cub::DeviceSelect::Flagged(h->select_tmp, tb, thrust::counting_iterator<int32_t>(0), h->blk_flag,
                                                 h->active, h->n_active_dev, nblk, s));
            g_vmat_launches += 2;
            int32_t cnt[2] = {0, 0};
            VMAT_CUDA(cudaMemcpyAsync(cnt, h->n_active_dev, 8, cudaMemcpyDeviceToHost, s));
            VMAT_CUDA(cudaStreamSynchronize(s));
            h->n_active = cnt[0]; h->n_reached = cnt[1];
        }
        h->active_R = R;
    }
    if (z && h->n_voxels > 0) VMAT_CUDA(cudaMemsetAsync(z, 0, (size_t)h->n_voxels * 4, s));   // voxels outside the blocks: z = 0
    if (max_iter + 1 > h->hist_cap) {
        if (h->F_hist) cudaFree(h->F_hist);
        if (h->delta_hist) cudaFree(h->delta_hist);
        h->F_hist = h->delta_hist = nullptr;
        h->hist_cap = 0;
        const size_t cap = (size_t)max_iter + 1 < 4096 ? 4096 : (size_t)max_iter + 1;
        VMAT_CUDA(cudaMalloc((void **)&h->F_hist, cap * 8));
        VMAT_CUDA(cudaMalloc((void **)&h->delta_hist, cap * 8));
        h->hist_cap = (int32_t)cap;
    }
    // the whole BB iteration in one cooperative launch; the start is clipped into the box inside (C16)
    MpArgs a;
    a.n = h->n_active; a.active = h->active; a.n_voxels = h->n_voxels; a.n_vox_pad = h->n_vox_pad; a.m = h->m; a.DA = h->DA;
    a.y = h->y; a.g = h->g; a.lo = h->lo; a.hi = h->hi; a.vstruct = voxel_struct; a.sid_aligned = ((uintptr_t)voxel_struct & 15) == 0; a.n_struct = n_struct; a.T = T;
    a.w_over = w_over; a.w_under = w_under; a.z_out = z; a.gpart = h->gpart; a.spart = h->spart; a.gsum = h->gsum;
    a.st = h->st; a.F_hist = h->F_hist; a.delta_hist = h->delta_hist; a.blk_flag = h->blk_flag; a.upart = h->upart;
    a.max_iter = max_iter; a.eps_F = eps_F; a.eps_y = eps_y;
    VMAT_CUDA(mp_launch_solve(h, a, s));
    VMAT_LAUNCH_CHECK();
    MpState cur;
    VMAT_CUDA(cudaMemcpyAsync(&cur, h->st, sizeof(cur), cudaMemcpyDeviceToHost, s));
    if (y_host) VMAT_CUDA(cudaMemcpyAsync(y_host, h->y, (size_t)h->m * 8, cudaMemcpyDeviceToHost, s));
    VMAT_CUDA(cudaStreamSynchronize(s));
    h->last_n_iter = cur.it;
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
    // scratch of the pricing step: one allocation owned by the master-problem handle, kept between calls
    struct Scratch {
        float *g, *p, *xs, *DA;
        int32_t *Lw, *Rw, *best, *win;
        double *row_price, *angle_price, *F;
        uint8_t *mask;
    } w;
    {
        auto up = [](size_t b) { return (b + 255) / 256 * 256; };
        const size_t need = 2 * up(nv * 4) + 2 * up(nb * 4) + 2 * up(nr * 4) + up(nr * 8) + up(na * 8) + up(4) + up(8) +
                            up(na) + up(nr * 16);
        if (need > mp->cg_scratch_bytes) {
            if (mp->cg_scratch) { VMAT_CUDA(cudaStreamSynchronize(s)); cudaFree(mp->cg_scratch); }
            mp->cg_scratch = nullptr; mp->cg_scratch_bytes = 0;
            VMAT_CUDA(cudaMalloc(&mp->cg_scratch, need));
            mp->cg_scratch_bytes = need;
        }
        char *q = (char *)mp->cg_scratch;
        auto take = [&](size_t b) { char *r = q; q += up(b); return (void *)r; };
        w.g = (float *)take(nv * 4); w.DA = (float *)take(nv * 4);
        w.p = (float *)take(nb * 4); w.xs = (float *)take(nb * 4);
        w.Lw = (int32_t *)take(nr * 4); w.Rw = (int32_t *)take(nr * 4);
        w.row_price = (double *)take(nr * 8); w.angle_price = (double *)take(na * 8);
        w.best = (int32_t *)take(4); w.F = (double *)take(8);
        w.mask = (uint8_t *)take(na);
        w.win = (int32_t *)take(nr * 16);                                                // L_lo, L_hi, R_lo, R_hi
    }
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
        g_vmat_launches = 0;
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
    REQUIRE(h->active_R != 0, "no solve has run since the last aperture was added");
    *n_reached = h->n_reached;
    return VMAT_OK;
}

int vmat_mp_pass_geometry(const vmat_mp *h, int32_t m, int32_t *n_cta, int32_t *rows_per_grid_step)
{
    REQUIRE(h != nullptr, "handle is NULL");
    REQUIRE(m >= 1 && m <= h->m_cap, "m must be in 1..max_apertures");
    if (n_cta) *n_cta = h->n_cta;
    if (rows_per_grid_step) *rows_per_grid_step = h->n_cta * MP_WARPS * mp_rows_per_stage(m);   // one block per warp and step
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
