// spmv.cuh - the row-dot building block of both SpMV kernels.
//
// A CSR row [s, e) of (val, idx) is streamed with 256-bit loads: every cooperating thread takes
// 8 consecutive non-zeros per load (32 B of values + 32 B of indices), so a warp covers 1 KB + 1 KB
// of contiguous, 32-byte-aligned stream per load pair.  Rows start at arbitrary offsets: the
// stream is read from the 8-element boundary at or below s and the (at most 7 + 7) elements outside
// [s, e) are masked.  Two chunks per thread are kept in flight (4 x 32 B = 128 B per thread).
#pragma once
#include "common.cuh"

// sum over the 8 elements k..k+7 of val*vec[idx], restricted to [s, e)
__device__ __forceinline__ float chunk_dot(const Vec8 &v, const Vec8 &c, int64_t k, int64_t s, int64_t e,
                                           const float *__restrict__ vec)
{
    float acc = 0.f;
    if (k >= s && k + 8 <= e) {
#pragma unroll
        for (int t = 0; t < 8; ++t) acc = fmaf(__uint_as_float(v.w[t]), ld_gather(vec + c.w[t]), acc);
    } else {
#pragma unroll
        for (int t = 0; t < 8; ++t)
            if (k + t >= s && k + t < e) acc = fmaf(__uint_as_float(v.w[t]), ld_gather(vec + c.w[t]), acc);
    }
    return acc;
}

// Partial dot product of row [s, e) with vec, for thread t of NT cooperating threads.
// The caller reduces the partials (warp shuffles or a block reduction).
template <int NT>
__device__ __forceinline__ float strided_row_dot(const float *__restrict__ val, const int32_t *__restrict__ idx,
                                                 int64_t s, int64_t e, const float *__restrict__ vec, int t)
{
    const int64_t a = s & ~int64_t(7);
    float acc0 = 0.f, acc1 = 0.f;
    for (int64_t k = a + (int64_t)t * 8; k < e; k += (int64_t)NT * 16) {
        const int64_t k2 = k + (int64_t)NT * 8;
        const bool has2 = k2 < e;
        Vec8 v0 = ld_stream_256(val + k);
        Vec8 c0 = ld_stream_256(idx + k);
        Vec8 v1, c1;
        if (has2) {
            v1 = ld_stream_256(val + k2);
            c1 = ld_stream_256(idx + k2);
        }
        acc0 += chunk_dot(v0, c0, k, s, e, vec);
        if (has2) acc1 += chunk_dot(v1, c1, k2, s, e, vec);
    }
    return acc0 + acc1;
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
