// dose.cu - A1 forward dose d = D x through the voxel-row CSR, with the
// objective / gradient (Eq. (1), Eq. (4)) fused into the row epilogue (A2).
//
// Voxel rows are ragged (0 ... ~18 k non-zeros, mean 10^2-10^3).  The ingest step cuts the row range
// into SEGMENTS, each owned by one warp (consecutive segments per CTA, so neighbouring voxels - which
// see nearly the same beamlets - share the x sectors cached in L1):
//   long row   (> DOSE_SEG_NNZ padded entries)  a segment of its own: the warp streams the row's
//              interleaved tiles with 256-bit loads and accumulates in registers, as the price kernel does;
//   short rows (consecutive rows, <= DOSE_SEG_NNZ padded entries together)  the warp streams the contiguous
//              range once, parks the products in its private slice of shared memory, then groups of
//              G lanes (G sized to the segment's mean row length) reduce one row each with shuffles
//              (pads hold 0 and belong to the row before them, so they change no sum).
// No block-wide barrier sits inside the streaming of a segment (the first version, one CTA per 4096-entry
// block, lost 21 % of its issue slots to barrier stalls - profiles/).  Everything is FP32 with a fixed summation
// order; the objective partials are FP64, one per ITEM (4 consecutive segments, the unit a CTA takes at a time),
// summed afterwards in a fixed order (no atomics).  Items reach the CTAs either one CTA per item or, where items
// are long and many, through per-SM queues drawn by a persistent grid (smqueue.cuh): same bits either way.
#include "spmv.cuh"
#include "smqueue.cuh"
#include <mutex>

// g_i and the voxel's term of F for dose v (Eq. (1); sign and factor 2: C1, C2)
__device__ __forceinline__ float voxel_grad(float v, float T, float wo, float wu, double &f)
{
    const float over = fmaxf(v - T, 0.f);
    const float under = fmaxf(T - v, 0.f);
    f += (double)wo * ((double)over * (double)over) + (double)wu * ((double)under * (double)under);
    return 2.f * wo * over - 2.f * wu * under;
}

// deterministic block sum of doubles; result valid in thread 0
template <int NT>
__device__ __forceinline__ double block_sum_double(double v, double *red /* [NT/32] */)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) red[w] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < NT / 32; ++i) s += red[i];
    return s;
}

// Item = DOSE_THREADS / 32 consecutive segments (one per warp); F_partial has one slot per item.
template <bool FUSE, int FMT>
__global__ void __launch_bounds__(DOSE_THREADS, VMAT_DOSE_MINB)
k_dose(const int64_t *__restrict__ pptr, const MatView A, const int32_t *__restrict__ seg_row, int n_seg,
       const float *__restrict__ x, float *__restrict__ d,
       const uint8_t *__restrict__ vstruct, const float *__restrict__ T,
       const float *__restrict__ w_over, const float *__restrict__ w_under, float *__restrict__ g,
       double *__restrict__ F_partial, const SmQueues Q)
{
    __shared__ float prod[DOSE_THREADS / 32][DOSE_SEG_NNZ];
    __shared__ double red_d[DOSE_THREADS / 32];
    __shared__ int s_item[3];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n_items = (n_seg + DOSE_THREADS / 32 - 1) / (DOSE_THREADS / 32);
    sq_init(Q, s_item);
#pragma unroll 1
    for (;;) {
        const int item = sq_next_item(Q, s_item);
        if (item < 0 || item >= n_items) break;
        const int sgi = item * (DOSE_THREADS / 32) + warp;
        double fsum = 0.0;
        auto epilogue = [&](int r, float v) {          // d, and the fused A2: g and the voxel's term of F
            d[r] = v;
            if (FUSE) {
                const int sid = vstruct[r];
                g[r] = voxel_grad(v, __ldg(T + sid), __ldg(w_over + sid), __ldg(w_under + sid), fsum);
            }
        };
        if (sgi < n_seg) {
            const int r0 = seg_row[sgi], r1 = seg_row[sgi + 1];
            const int nr = r1 - r0;
            const int64_t s = pptr[r0], e = pptr[r1];               // padded positions, multiples of 32
            if (nr == 1) {
                // ---- one row: register accumulation
                const float acc = warp_sum(segment_dot<FMT, VMAT_DOSE_DEPTH>(A, s, e, x, lane));
                if (lane == 0) epilogue(r0, acc);
            } else {
                // ---- several short rows: products into this warp's slice at their padded position k - s ...
                float *wp = prod[warp];
                VMAT_ASSERT(e - s <= DOSE_SEG_NNZ);                  // the run of short rows fits this warp's slice
                const int nt = (int)((e - s) >> 8);
                TileCursor<FMT> tc(A, s, lane);
#pragma unroll 1
                for (int ti = 0; ti < nt; ++ti, tc.advance()) {
                    TileRegs<FMT> tr;
                    tile_load<FMT>(A, tc, lane, tr);
                    int c[8];
                    tile_indices<FMT>(A, tc, tr, lane, c);
                    float *dst = wp + ti * TILE + lane;
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        VMAT_ASSERT_INDEX(A, c[t]);
                        dst[32 * t] = __uint_as_float(tr.v.w[t]) * ld_gather(x + c[t]);
                    }
                }
                const int64_t k0 = s + (int64_t)nt * TILE;
                float *dst = wp + nt * TILE + lane;
                tail_foreach<FMT>(A, k0, (int)((e - k0) >> 5), x, lane, [&](int t, float q_) { dst[32 * t] = q_; });
                __syncwarp();
                // ... then G lanes per row, G = power of two near (mean row length)/4, 1..32
                const int mean = (int)((e - s) / nr);
                int G = 1;
                while (G < 32 && G * 4 < mean) G <<= 1;
                const int grp = lane / G, gl = lane % G, n_grp = 32 / G;
                const int n_iter = (nr + n_grp - 1) / n_grp;        // uniform trip count: shuffles stay converged
                for (int it = 0; it < n_iter; ++it) {
                    const int r = r0 + grp + it * n_grp;
                    float acc = 0.f;
                    if (r < r1) {
                        const int b = (int)(pptr[r] - s), f = (int)(pptr[r + 1] - s);
                        VMAT_ASSERT(0 <= b && b <= f && f <= (int)(e - s));
                        for (int k = b + gl; k < f; k += G) acc += wp[k];
                    }
                    for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                    if (r < r1 && gl == 0) epilogue(r, acc);
                }
                __syncwarp();                                       // the slice is refilled by the next item
            }
        }
        if (FUSE) {
            const double tot = block_sum_double<DOSE_THREADS>(fsum, red_d);
            if (threadIdx.x == 0) F_partial[((volatile int *)s_item)[0]] = tot;     // re-read: no register held across the loop
        }
    }
}

// Standalone A2 (vmat_objective_grad): one thread per voxel, FP64 partial per block.
constexpr int OBJ_THREADS = 256;
__global__ void __launch_bounds__(OBJ_THREADS)
k_objective(int n_voxels, const float *__restrict__ d, const uint8_t *__restrict__ vstruct, int n_struct,
            const float *__restrict__ T, const float *__restrict__ w_over, const float *__restrict__ w_under,
            float *__restrict__ g, double *__restrict__ F_partial)
{
    __shared__ double red_d[OBJ_THREADS / 32];
    const int i = blockIdx.x * OBJ_THREADS + threadIdx.x;
    double f = 0.0;
    if (i < n_voxels) {
        const int sid = vstruct[i];
        g[i] = voxel_grad(d[i], __ldg(T + sid), __ldg(w_over + sid), __ldg(w_under + sid), f);
    }
    const double tot = block_sum_double<OBJ_THREADS>(f, red_d);
    if (threadIdx.x == 0) F_partial[blockIdx.x] = tot;
}

// F = sum of the per-block partials, fixed order: thread t sums part[t], part[t+1024], ...; then a tree.
constexpr int SUM_THREADS = 1024;
__global__ void __launch_bounds__(SUM_THREADS)
k_sum_partials(const double *__restrict__ part, int n, double *__restrict__ out)
{
    __shared__ double red_d[SUM_THREADS / 32];
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += SUM_THREADS) s += part[i];
    const double tot = block_sum_double<SUM_THREADS>(s, red_d);
    if (threadIdx.x == 0) out[0] = tot;
}

// x in the column order of CSR(D) (common.cuh: tiles of 8 columns x all leaf rows per control point)
__global__ void k_permute_x(int n, const int32_t *__restrict__ perm, const float *__restrict__ x, float *__restrict__ xp)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) xp[perm[j]] = x[j];
}

// Launch geometry: SM-affine queues -> a persistent grid of SM count x resident CTAs per SM; static -> one CTA per item.
template <bool FUSE, int FMT>
static int dose_grid(const vmat_ddc *h)
{
    if (h->queues_dose().nq == 0) return h->n_blocks;
    static std::atomic<int> occ[VMAT_MAX_DEVICES];                   // per kernel instance and device
    return min(h->n_blocks, h->n_sm * vmat_resident_ctas(k_dose<FUSE, FMT>, DOSE_THREADS, h->device, occ));
}
int vmat_dose_grid(const vmat_ddc *h, bool fuse)
{
    switch (fmt_of(h->D) + (fuse ? 3 : 0)) {
    case 0: return dose_grid<false, FMT_WIDE>(h);
    case 1: return dose_grid<false, FMT_NARROW>(h);
    case 2: return dose_grid<false, FMT_NARROW_1BASE>(h);
    case 3: return dose_grid<true, FMT_WIDE>(h);
    case 4: return dose_grid<true, FMT_NARROW>(h);
    default: return dose_grid<true, FMT_NARROW_1BASE>(h);
    }
}

int vmat_launch_dose(const vmat_ddc *h, const float *x, float *d, bool fuse,
                     const uint8_t *voxel_struct, int32_t n_struct, const float *T, const float *w_over,
                     const float *w_under, float *g, double *F, cudaStream_t st)
{
    if (fuse && h->prof_ev[0]) VMAT_CUDA(cudaEventRecord(h->prof_ev[0], st));
    if (h->col_perm != nullptr && h->n_blocks > 0) {
        k_permute_x<<<(h->n_beamlets + 255) / 256, 256, 0, st>>>(h->n_beamlets, h->col_perm, x, h->x_perm);
        VMAT_LAUNCH_CHECK();
        x = h->x_perm;
    }
    if (h->n_blocks > 0) {
        const MatView A = view_of(h->D);
        const SmQueues Q = h->queues_dose();
#define VMAT_DOSE_LAUNCH(FUSE_, FMT_, ...)                                                              \
        k_dose<FUSE_, FMT_><<<dose_grid<FUSE_, FMT_>(h), DOSE_THREADS, 0, st>>>(h->D.pptr, A, h->seg_row, h->n_seg, x, d, __VA_ARGS__, Q)
#define VMAT_DOSE_ARGS_FUSED voxel_struct, T, w_over, w_under, g, h->F_partial
#define VMAT_DOSE_ARGS_PLAIN nullptr, nullptr, nullptr, nullptr, nullptr, nullptr
        switch (fmt_of(h->D) + (fuse ? 3 : 0)) {
        case 0: VMAT_DOSE_LAUNCH(false, FMT_WIDE, VMAT_DOSE_ARGS_PLAIN); break;
        case 1: VMAT_DOSE_LAUNCH(false, FMT_NARROW, VMAT_DOSE_ARGS_PLAIN); break;
        case 2: VMAT_DOSE_LAUNCH(false, FMT_NARROW_1BASE, VMAT_DOSE_ARGS_PLAIN); break;
        case 3: VMAT_DOSE_LAUNCH(true, FMT_WIDE, VMAT_DOSE_ARGS_FUSED); break;
        case 4: VMAT_DOSE_LAUNCH(true, FMT_NARROW, VMAT_DOSE_ARGS_FUSED); break;
        default: VMAT_DOSE_LAUNCH(true, FMT_NARROW_1BASE, VMAT_DOSE_ARGS_FUSED); break;
        }
#undef VMAT_DOSE_LAUNCH
#undef VMAT_DOSE_ARGS_FUSED
#undef VMAT_DOSE_ARGS_PLAIN
        VMAT_LAUNCH_CHECK();
    }
    if (fuse && h->prof_ev[1]) VMAT_CUDA(cudaEventRecord(h->prof_ev[1], st));
    if (fuse) {
        k_sum_partials<<<1, SUM_THREADS, 0, st>>>(h->F_partial, h->n_blocks, F);
        VMAT_LAUNCH_CHECK();
    }
    return VMAT_OK;
}

int vmat_launch_objective(const vmat_ddc *h, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                          const float *T, const float *w_over, const float *w_under, float *g, double *F,
                          cudaStream_t st)
{
    if (h->n_obj_blocks > 0) {
        k_objective<<<h->n_obj_blocks, OBJ_THREADS, 0, st>>>(h->n_voxels, d, voxel_struct, n_struct, T, w_over,
                                                             w_under, g, h->F_partial_obj);
        VMAT_LAUNCH_CHECK();
    }
    k_sum_partials<<<1, SUM_THREADS, 0, st>>>(h->F_partial_obj, h->n_obj_blocks, F);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// vmat_objective_grad_static (include/vmat.h): A2 without a handle and without a single allocation.
//
// Who needs this: code that is not allowed to call cudaMalloc at the moment it wants F and g.  Examples are a treatment
// planning host that hands the GPU's whole memory to its own pool at start-up, so that a later driver allocation fails
// or eats into that pool's headroom; a real-time control loop that must not take the driver's allocation lock
// (cudaMalloc can wait for all work on the device); and a plug-in whose host forbids driver allocations once it is
// initialised.  The handle-based vmat_objective_grad cannot serve them: its scratch (one FP64 partial sum of F per block
// of 256 voxels) belongs to a vmat_ddc, and vmat_ddc_create allocates.
//
// Here that scratch is the file-scope array below.  It is part of the library image: every GPU on which libvmat.so
// gets loaded holds its 256 KiB from the moment the CUDA module is loaded until the process exits, whether this entry
// point is ever called or not.  That is why the maximum is modest: VMAT_OBJECTIVE_STATIC_MAX_VOXELS = 2^23 voxels
// (config 3 of BASELINE.json, the largest, has 1.24 million).
//
// In host code `g_static_F_partial` is only a host-side shadow of the symbol: handing that name to a kernel would give it
// a host address.  The device address is asked for with cudaGetSymbolAddress, once per device, with that device current,
// and kept in g_static_F_partial_dev[device]; the kernels get that pointer.
static __device__ __align__(256) double g_static_F_partial[VMAT_OBJECTIVE_STATIC_MAX_VOXELS / OBJ_THREADS];

constexpr int STATIC_MAX_DEVICES = 64;
static double *g_static_F_partial_dev[STATIC_MAX_DEVICES];   // device address of the array on device i; NULL = not set up
static std::mutex g_static_mu;

extern "C" int vmat_objective_grad_static(int32_t n_voxels, const float *d, const uint8_t *voxel_struct, int32_t n_struct,
                                          const float *T, const float *w_over, const float *w_under, float *g, double *F,
                                          void *stream)
{
    static_assert(VMAT_OBJECTIVE_STATIC_MAX_VOXELS % OBJ_THREADS == 0, "whole blocks");
    if (n_voxels < 0 || !F || !T || !w_over || !w_under || (n_voxels > 0 && (!d || !voxel_struct || !g))) {
        vmat_set_error("vmat_objective_grad_static: NULL argument or negative n_voxels");
        return VMAT_ERR_INVALID_ARG;
    }
    if (n_struct < 1 || n_struct > 256) {
        vmat_set_error("vmat_objective_grad_static: n_struct must be in 1..256");
        return VMAT_ERR_INVALID_ARG;
    }
    if (n_voxels > VMAT_OBJECTIVE_STATIC_MAX_VOXELS) {
        vmat_set_error("vmat_objective_grad_static: n_voxels = %d exceeds VMAT_OBJECTIVE_STATIC_MAX_VOXELS = %d, the size "
                       "the built-in scratch was compiled for; use vmat_objective_grad (handle-owned scratch) instead",
                       n_voxels, (int)VMAT_OBJECTIVE_STATIC_MAX_VOXELS);
        return VMAT_ERR_INVALID_ARG;
    }
    int dev = -1;
    VMAT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) {
        vmat_set_error("vmat_objective_grad_static: device ordinal %d beyond the %d this entry point keeps addresses for",
                       dev, STATIC_MAX_DEVICES);
        return VMAT_ERR_INVALID_ARG;
    }
    double *part = nullptr;
    {   // set-up, first call on this device only: no allocation, just the address of the array on the current device
        std::lock_guard<std::mutex> lk(g_static_mu);
        if (!g_static_F_partial_dev[dev]) {
            void *p = nullptr;
            VMAT_CUDA(cudaGetSymbolAddress(&p, g_static_F_partial));
            g_static_F_partial_dev[dev] = (double *)p;
        }
        part = g_static_F_partial_dev[dev];
    }
    cudaStream_t st = (cudaStream_t)stream;
    g_vmat_launches = 0;
    // Same two kernels, same block size and same summation order as vmat_objective_grad, hence the same bits.  Every
    // slot k_sum_partials reads was written by k_objective in this very call, so nothing of the array has to start at
    // zero and what an earlier (possibly larger) call left behind is never read.
    const int n_blocks = (n_voxels + OBJ_THREADS - 1) / OBJ_THREADS;
    if (n_blocks > 0) {
        k_objective<<<n_blocks, OBJ_THREADS, 0, st>>>(n_voxels, d, voxel_struct, n_struct, T, w_over, w_under, g, part);
        VMAT_LAUNCH_CHECK();
    }
    k_sum_partials<<<1, SUM_THREADS, 0, st>>>(part, n_blocks, F);
    VMAT_LAUNCH_CHECK();
    return VMAT_OK;
}
