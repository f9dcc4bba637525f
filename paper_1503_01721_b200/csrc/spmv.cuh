// spmv.cuh - the streaming building blocks of both SpMV kernels, and the tile-interleaved storage
// order they rely on.
//
// Why the layout is not plain CSR order.  A warp must read the (val, idx) streams with wide,
// coalesced loads (sm_100 has 256-bit loads: 32 lanes x 32 B = 1 KB per instruction), but the gather
// vec[idx] that follows wants CONSECUTIVE lanes on CONSECUTIVE non-zeros: indices come in runs (a
// beamlet's voxels are x-runs of the raster, a voxel's beamlets are runs along a leaf row), so 32
// consecutive non-zeros touch a handful of 32-byte sectors, while "lane l owns non-zeros 8l..8l+7"
// touches 32 sectors in every gather instruction - ncu showed exactly that (profiles/r1_v1_first_path.md:
// 2.78 G sectors for 2.78 G gathered floats, L1TEX at 77-83 %, HBM at 45-64 %).
//
// So a segment [s, e) of a layout (a beamlet row of D^T; a row block of D) is stored as
//     head   [s, a0)            plain order,  a0 = min(e, s rounded up to 8)   (<= 7 entries)
//     tiles  [a0, a0 + 256 nt)  nt = (e - a0) / 256 full tiles, each LANE-INTERLEAVED:
//                               stored word 8*l + t of a tile holds the tile's logical entry 32*t + l
//     tail   [a0 + 256 nt, e)   plain order  (< 256 entries)
// It is a permutation inside the segment: 8 B/nnz, row pointers unchanged.  Lane l's 256-bit load of a
// tile yields logical entries l, 32+l, ..., 224+l, so gather instruction t covers 32 consecutive entries.
#pragma once
#include "common.cuh"

constexpr int TILE = 256;

struct Segment {
    int64_t a0;   // first tile
    int64_t nt;   // number of full tiles
    int64_t t0;   // start of the plain tail
};
__host__ __device__ __forceinline__ Segment segment_of(int64_t s, int64_t e)
{
    Segment g;
    const int64_t up = (s + 7) & ~int64_t(7);
    g.a0 = up < e ? up : e;
    g.nt = (e - g.a0) / TILE;
    g.t0 = g.a0 + g.nt * TILE;
    return g;
}

// One interleaved tile starting at k: this lane's partial of sum val*vec[idx].
__device__ __forceinline__ float tile_dot(const float *__restrict__ val, const int32_t *__restrict__ idx,
                                          int64_t k, const float *__restrict__ vec, int lane)
{
    const Vec8 v = ld_stream_256(val + k + lane * 8);
    const Vec8 c = ld_stream_256(idx + k + lane * 8);
    float acc = 0.f;
#pragma unroll
    for (int t = 0; t < 8; ++t) acc = fmaf(__uint_as_float(v.w[t]), ld_gather(vec + c.w[t]), acc);
    return acc;
}

// The plain head [s, a0) and tail [t0, e) of a segment, spread over NT cooperating threads (thread t):
// calls f(k, val[k] * vec[idx[k]]) for this thread's entries.  At most 7 + 255 entries, so
// ceil(255 / NT) + 1 independent loads per thread, all issued before the gathers.
template <int NT, typename F>
__device__ __forceinline__ void plain_foreach(const float *__restrict__ val, const int32_t *__restrict__ idx,
                                              int64_t s, const Segment &sg, int64_t e,
                                              const float *__restrict__ vec, int t, F f)
{
    constexpr int N = (TILE - 1 + NT - 1) / NT;           // tail passes (8 for a warp, 1 for 256 threads)
    constexpr int B = N < 4 ? N : 4;                      // loads issued together
    const int n_tail = (int)(e - sg.t0);
#pragma unroll
    for (int i0 = 0; i0 < N; i0 += B) {
        float v[B];
        int c[B];
#pragma unroll
        for (int i = 0; i < B; ++i) {
            const int o = (i0 + i) * NT + t;
            const bool ok = i0 + i < N && o < n_tail;
            v[i] = ok ? ld_stream_f(val + sg.t0 + o) : 0.f;
            c[i] = ok ? ld_stream_i(idx + sg.t0 + o) : 0;
        }
#pragma unroll
        for (int i = 0; i < B; ++i) {
            const int o = (i0 + i) * NT + t;
            if (i0 + i < N && o < n_tail) f(sg.t0 + o, v[i] * ld_gather(vec + c[i]));
        }
    }
    if (s + t < sg.a0) {                                  // head: NT >= 8 > 7 entries
        const float v = ld_stream_f(val + s + t);
        const int c = ld_stream_i(idx + s + t);
        f(s + t, v * ld_gather(vec + c));
    }
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
