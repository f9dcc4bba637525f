// spmv.cuh - the streaming building blocks of both SpMV kernels, and the grouped, tile-interleaved
// storage order they rely on.
//
// Storage.  The rows of a layout are cut into SEGMENTS, one warp each (a beamlet row of D^T; a long voxel
// row or a run of short voxel rows of D).  A segment is a whole number of GROUPS of 32 entries and starts
// at a multiple of 32 padded positions; the last group of a segment (and, in the narrow format, a group
// closed early, below) is filled up with PADS: value 0, index of the entry before it.  Pads add 0 to the
// row they fall in.  Entries keep their canonical order (row-major, ascending secondary index), so every
// floating-point sum has a fixed order whatever the order of the input triplets.
//
// Why groups of 32 consecutive entries.  A warp must read the streams with wide coalesced loads (sm_100:
// 256-bit, 1 KB per warp instruction), but the gather vec[idx] that follows wants CONSECUTIVE lanes on
// CONSECUTIVE non-zeros: indices come in runs (a beamlet's voxels are x-runs of the raster, a voxel's
// beamlets are runs along a leaf row), so 32 consecutive non-zeros touch a handful of 32-byte sectors,
// while "lane l owns non-zeros 8l..8l+7" touches 32 sectors per gather instruction (measured:
// profiles/r1_v1_first_path.md, L1TEX at 77-83 %, HBM at 45-64 %).  So 8 consecutive groups of a segment
// form a TILE that is stored LANE-INTERLEAVED: stored word 8*l + t of the tile holds entry l of group t.
// Lane l's 256-bit load yields entry l of all 8 groups; gather instruction t covers group t.  The groups
// after the last full tile of a segment (0..7) are stored in plain order and read with scalar loads.
//
// Narrow indices (index_bits 16).  Within a group the secondary indices span little (the same runs), so a
// group stores one int32 BASE (its minimum index) and 32 u16 OFFSETS: 4 + 2 + 4/32 = 6.125 B per entry
// instead of the paper's 8 (Table 2).  The ingest step closes a group early when the next
// entry would stretch its span beyond 65535, so the format holds any matrix; it is chosen per layout only
// when it is smaller than the wide one (ingest.cu).  Measured on B200: the price kernel moves 23 % fewer
// bytes and runs 26 % faster (profiles/r1_v5_narrow_indices.md).
#pragma once
#include "common.cuh"

constexpr int GROUP = 32;
constexpr int TILE = 256;

// Stored position of padded logical position q of a segment that starts at S and holds G groups.
__host__ __device__ __forceinline__ int64_t stored_pos(int64_t S, int64_t G, int64_t q)
{
    const int64_t ql = q - S, gl = ql >> 5, slot = ql & 31;
    return gl < (G & ~int64_t(7)) ? S + ((gl >> 3) << 8) + 8 * slot + (gl & 7) : q;
}

// Secondary indices of this lane's 8 entries of the tile at padded position k (entry `lane` of groups 0..7).
template <bool NARROW>
__device__ __forceinline__ void tile_indices(const MatView &A, int64_t k, int lane, int (&c)[8])
{
    if (NARROW) {
        const Vec4 o = ld_stream_128((const uint16_t *)A.sec + k + lane * 8);
        const int b = ld_stream_i(A.base + (k >> 5) + (lane & 7));        // the tile's 8 bases, one 32-byte line
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            const int bt = __shfl_sync(0xffffffffu, b, t);
            c[t] = bt + (int)((t & 1) ? (o.w[t >> 1] >> 16) : (o.w[t >> 1] & 0xffffu));
        }
    } else {
        const Vec8 o = ld_stream_256((const int32_t *)A.sec + k + lane * 8);
#pragma unroll
        for (int t = 0; t < 8; ++t) c[t] = (int)o.w[t];
    }
}

// One interleaved tile at padded position k: this lane's partial of sum val*vec[idx].
template <bool NARROW>
__device__ __forceinline__ float tile_dot(const MatView &A, int64_t k, const float *__restrict__ vec, int lane)
{
    const Vec8 v = ld_stream_256(A.val + k + lane * 8);
    int c[8];
    tile_indices<NARROW>(A, k, lane, c);
    float acc = 0.f;
#pragma unroll
    for (int t = 0; t < 8; ++t) acc = fmaf(__uint_as_float(v.w[t]), ld_gather(vec + c[t]), acc);
    return acc;
}

// Entry `lane` of the plain-order group at padded position kg: value and secondary index.
template <bool NARROW>
__device__ __forceinline__ void group_entry(const MatView &A, int64_t kg, int lane, float &v, int &c)
{
    v = ld_stream_f(A.val + kg + lane);
    if (NARROW) c = ld_stream_i(A.base + (kg >> 5)) + ld_stream_u16((const uint16_t *)A.sec + kg + lane);
    else        c = ld_stream_i((const int32_t *)A.sec + kg + lane);
}

// The ngt (0..7) plain-order groups after the last full tile, starting at padded position k0:
// calls f(t, product) for this lane's entry of group t.  Four groups' loads are issued together.
template <bool NARROW, typename F>
__device__ __forceinline__ void tail_foreach(const MatView &A, int64_t k0, int ngt, const float *__restrict__ vec,
                                             int lane, F f)
{
#pragma unroll
    for (int t0 = 0; t0 < 8; t0 += 4) {
        if (t0 >= ngt) break;
        float v[4];
        int c[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[i] = 0.f; c[i] = 0;
            if (t0 + i < ngt) group_entry<NARROW>(A, k0 + 32 * (t0 + i), lane, v[i], c[i]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (t0 + i < ngt) f(t0 + i, v[i] * ld_gather(vec + c[i]));
    }
}

// A whole segment [s, e) (padded positions, multiples of 32) as one dot product: this lane's partial.
template <bool NARROW>
__device__ __forceinline__ float segment_dot(const MatView &A, int64_t s, int64_t e, const float *__restrict__ vec,
                                             int lane)
{
    const int nt = (int)((e - s) >> 8);
    float acc = 0.f;
#pragma unroll 1
    for (int ti = 0; ti < nt; ++ti) acc += tile_dot<NARROW>(A, s + (int64_t)ti * TILE, vec, lane);
    const int64_t k0 = s + (int64_t)nt * TILE;
    tail_foreach<NARROW>(A, k0, (int)((e - k0) >> 5), vec, lane, [&](int, float q) { acc += q; });
    return acc;
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
