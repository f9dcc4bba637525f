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
// Kernel variants by index format: int32 indices; u16 offsets with the per-tile check of the base flag; u16
// offsets of a layout in which EVERY full tile has one base (no check, no shuffle path compiled in).
enum { FMT_WIDE = 0, FMT_NARROW = 1, FMT_NARROW_1BASE = 2 };


// Stored position of padded logical position q of a segment that starts at S and holds G groups.
__host__ __device__ __forceinline__ int64_t stored_pos(int64_t S, int64_t G, int64_t q)
{
    const int64_t ql = q - S, gl = ql >> 5, slot = ql & 31;
    return gl < (G & ~int64_t(7)) ? S + ((gl >> 3) << 8) + 8 * slot + (gl & 7) : q;
}

// Base word of a group: the group's base index; bit 31 of the FIRST group of a full tile set = all 8 groups of
// the tile share this base (written by the ingest step whenever the tile's indices span <= 65535, which is
// the rule for these matrices): the warp then needs one broadcast load per tile instead of one base per group.
constexpr int TILE_UNIFORM_BIT = int(0x80000000u);
__host__ __device__ __forceinline__ int base_index(int word) { return word & 0x7fffffff; }

// This lane's position in a segment's interleaved tiles, in ONE register: units of 8 stored entries (32 bytes of
// values), u = s / 8 + lane + 32 * tile; the stream addresses are formed from it with one multiply-add each against
// the layout's base pointers (constant bank).  The first version kept three 64-bit pointers (6 registers), which at
// the kernels' 40 registers left none for the item loop of the persistent kernels.  P / 8 < 2^32 is checked at ingest.
template <int FMT>
struct TileCursor {
    uint32_t u;
    __device__ __forceinline__ TileCursor(const MatView &, int64_t s, int lane) : u((uint32_t)(s >> 3) + (uint32_t)lane) {}
    __device__ __forceinline__ void advance() { u += TILE / 8; }
    __device__ __forceinline__ const float *v(const MatView &A) const { return A.val + (size_t)u * 8; }   // 8 values
    __device__ __forceinline__ const char *i(const MatView &A) const                // 8 offsets (u16) or indices (i32)
    {
        return (const char *)A.sec + (size_t)u * (FMT != FMT_WIDE ? 16 : 32);
    }
    __device__ __forceinline__ const int32_t *b(const MatView &A, int lane) const   // the tile's 8 base words
    {
        return A.base + ((u - (uint32_t)lane) >> 2);
    }
    __device__ __forceinline__ int64_t pos(int lane) const { return (int64_t)(u - (uint32_t)lane) << 3; }   // padded position of the tile
};

// This lane's share of one tile's streams, in registers: loading and using are separate steps so that a loop
// can have the next tile's loads in flight while it gathers for the current one.
template <int FMT>
struct TileRegs {
    Vec8 v;                  // 8 values
    Vec8 o;                  // wide: 8 int32 indices; narrow: o.w[0..3] = 8 u16 offsets, o.w[4] = the tile's base word
};
template <int FMT>
__device__ __forceinline__ void tile_load(const MatView &A, const TileCursor<FMT> &tc, int lane, TileRegs<FMT> &r)
{
    VMAT_ASSERT_STREAM(A, (int64_t)tc.u * 8, 8);
    r.v = ld_stream_256(tc.v(A));
    if (FMT != FMT_WIDE) {
        const Vec4 o = ld_stream_128(tc.i(A));
        r.o.w[0] = o.w[0]; r.o.w[1] = o.w[1]; r.o.w[2] = o.w[2]; r.o.w[3] = o.w[3];
        r.o.w[4] = (uint32_t)ld_stream_i(tc.b(A, lane));                    // broadcast: one 128-byte wavefront
    } else {
        r.o = ld_stream_256(tc.i(A));
    }
}

// Secondary indices of this lane's 8 entries of the tile (entry `lane` of groups 0..7).
template <int FMT>
__device__ __forceinline__ void tile_indices(const MatView &A, const TileCursor<FMT> &tc, const TileRegs<FMT> &r, int lane,
                                             int (&c)[8])
{
    if (FMT != FMT_WIDE) {
        const int b0 = (int)r.o.w[4];
        if (FMT == FMT_NARROW_1BASE || b0 < 0) {                            // warp-uniform branch
            const int bb = base_index(b0);
#pragma unroll
            for (int t = 0; t < 8; ++t)
                c[t] = bb + (int)((t & 1) ? (r.o.w[t >> 1] >> 16) : (r.o.w[t >> 1] & 0xffffu));
        } else {                                                            // one base per group, by shuffles
            const int b = ld_stream_i(tc.b(A, lane) + (lane & 7));
#pragma unroll
            for (int t = 0; t < 8; ++t) {
                const int bt = __shfl_sync(0xffffffffu, b, t);
                c[t] = bt + (int)((t & 1) ? (r.o.w[t >> 1] >> 16) : (r.o.w[t >> 1] & 0xffffu));
            }
        }
    } else {
#pragma unroll
        for (int t = 0; t < 8; ++t) c[t] = (int)r.o.w[t];
    }
}

// One interleaved tile: this lane's partial of sum val*vec[idx].
template <int FMT>
__device__ __forceinline__ float tile_dot(const MatView &A, const TileCursor<FMT> &tc, const TileRegs<FMT> &r,
                                          const float *__restrict__ vec, int lane)
{
    int c[8];
    tile_indices<FMT>(A, tc, r, lane, c);
#pragma unroll
    for (int t = 0; t < 8; ++t) VMAT_ASSERT_INDEX(A, c[t]);
    float acc = 0.f;
#pragma unroll
    for (int t = 0; t < 8; ++t) acc = fmaf(__uint_as_float(r.v.w[t]), ld_gather(vec + c[t]), acc);
    return acc;
}

// Entry `lane` of the plain-order group at padded position kg: value and secondary index.
template <int FMT>
__device__ __forceinline__ void group_entry(const MatView &A, int64_t kg, int lane, float &v, int &c)
{
    VMAT_ASSERT_STREAM(A, kg + lane, 1);
    v = ld_stream_f(A.val + kg + lane);
    if (FMT != FMT_WIDE) c = base_index(ld_stream_i(A.base + (kg >> 5))) + ld_stream_u16((const uint16_t *)A.sec + kg + lane);
    else        c = ld_stream_i((const int32_t *)A.sec + kg + lane);
    VMAT_ASSERT_INDEX(A, c);
}

// The ngt (0..7) plain-order groups after the last full tile, starting at padded position k0:
// calls f(t, product) for this lane's entry of group t.  Four groups' loads are issued together.
template <int FMT, typename F>
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
            if (t0 + i < ngt) group_entry<FMT>(A, k0 + 32 * (t0 + i), lane, v[i], c[i]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (t0 + i < ngt) f(t0 + i, v[i] * ld_gather(vec + c[i]));
    }
}

// A whole segment [s, e) (padded positions, multiples of 32) as one dot product: this lane's partial.
// DEPTH = tiles whose stream loads are in flight or in registers at once (1: load, use, load ...; 2: the next tile's
// loads are issued before this tile's gathers; 3: two tiles ahead).  DEPTH register sets take turns (the loop body is
// unrolled DEPTH times), so nothing is copied.  Only the cursor, the counts and the sum live across the loop (s and e
// are dead once the counts are formed: the tail starts where the cursor stands).  Tiles are added in order whatever
// the depth: the result does not depend on it.
template <int FMT, int DEPTH>
__device__ __forceinline__ float segment_dot(const MatView &A, int64_t s, int64_t e, const float *__restrict__ vec,
                                             int lane)
{
    const int nt = (int)((e - s) >> 8);
    const int ngt = (int)((e - s) >> 5) & 7;
    float acc = 0.f;
    TileCursor<FMT> tc(A, s, lane);                              // the next tile to LOAD
    if (DEPTH == 2) {                                            // written out: one count, no spare register at 40
        if (nt > 0) {
            TileRegs<FMT> ra, rb;
            tile_load<FMT>(A, tc, lane, ra);
            int left = nt - 1;                                   // tiles not yet loaded
#pragma unroll 1
            for (; left >= 2; left -= 2) {
                TileCursor<FMT> t0 = tc;
                tc.advance();
                tile_load<FMT>(A, tc, lane, rb);
                acc += tile_dot<FMT>(A, t0, ra, vec, lane);
                t0 = tc;
                tc.advance();
                tile_load<FMT>(A, tc, lane, ra);
                acc += tile_dot<FMT>(A, t0, rb, vec, lane);
            }
            if (left == 1) {
                TileCursor<FMT> t0 = tc;
                tc.advance();
                tile_load<FMT>(A, tc, lane, rb);
                acc += tile_dot<FMT>(A, t0, ra, vec, lane);
                acc += tile_dot<FMT>(A, tc, rb, vec, lane);
            } else {
                acc += tile_dot<FMT>(A, tc, ra, vec, lane);
            }
            tc.advance();
        }
    } else if (DEPTH > 2) {
        TileRegs<FMT> r[DEPTH];
        int to_load = nt, to_use = nt;
#pragma unroll
        for (int j = 0; j < DEPTH - 1; ++j)
            if (to_load > 0) { tile_load<FMT>(A, tc, lane, r[j]); tc.advance(); --to_load; }
#pragma unroll 1
        while (to_use > 0) {
#pragma unroll
            for (int j = 0; j < DEPTH; ++j) {
                if (to_load > 0) { tile_load<FMT>(A, tc, lane, r[(j + DEPTH - 1) % DEPTH]); tc.advance(); --to_load; }
                if (to_use > 0) {
                    TileCursor<FMT> tu = tc;                     // the tile in r[j]: DEPTH - 1 (or fewer, at the end) behind
                    tu.u -= (uint32_t)((to_use - to_load) * (TILE / 8));
                    acc += tile_dot<FMT>(A, tu, r[j], vec, lane);
                    --to_use;
                }
            }
        }
    } else {
#pragma unroll 1
        for (int ti = 0; ti < nt; ++ti, tc.advance()) {
            TileRegs<FMT> r;
            tile_load<FMT>(A, tc, lane, r);
            acc += tile_dot<FMT>(A, tc, r, vec, lane);
        }
    }
    tail_foreach<FMT>(A, tc.pos(lane), ngt, vec, lane, [&](int, float q) { acc += q; });
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
