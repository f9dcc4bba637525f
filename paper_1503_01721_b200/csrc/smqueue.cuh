// smqueue.cuh - SM-affine work distribution for the two streaming kernels (k_dose, k_price).
//
// Why.  Both kernels gather from a small vector (x, g) while they stream the matrix, and NEIGHBOURING work items
// gather nearly the same entries: 8 consecutive beamlets of a leaf row see cylinders through the body that overlap
// by 80-90 %, consecutive voxels of a raster line see the same beamlets of every control point.  With one CTA per
// work item the hardware hands consecutive CTAs to DIFFERENT SMs, so the CTAs resident on one SM at a time are
// ~148 items apart, share nothing, and every gather sector is fetched from L2 once per CTA: 0.85-0.9 G sectors per
// launch against 0.54 G for the matrix stream itself (profiles/r2_hot_kernels.md) - the L2 -> L1 traffic, and the
// power it costs under the 1 kW cap, is dominated by the gathers.  Here the item range is cut into one contiguous
// QUEUE per SM (equal stored bytes each), the kernels are persistent (SM count x resident CTAs per SM), and a CTA
// takes its next item from the queue of the SM it runs on (%smid): the CTAs resident on an SM work on adjacent
// items at the same time and find each other's gather lines in L1.  A CTA whose queue is empty takes items from
// the next non-empty queue (cyclic), so the tail is as balanced as with one CTA per item.
//
// Results do not depend on who processes an item (every item's sums have a fixed order and its outputs their own
// slots), so the schedule changes no bit of any output.
#pragma once
#include <stdint.h>

struct SmQueues {
    const int32_t *start;   // [nq + 1] first item of each queue; start[nq] = number of items
    uint32_t *next;         // [nq + 1] items handed out per queue (may run past the queue's size); next[nq] = CTAs
                            // that have finished - the last one zeroes everything for the next launch
    int nq;                 // 0 = static schedule: one CTA per item, CTA b takes item b
    int chunk;              // consecutive items a CTA takes per visit to a queue (one atomic per chunk)
};

__device__ __forceinline__ unsigned sq_smid()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned sq_peek(const uint32_t *p)
{
    unsigned r;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}

// Next chunk of items for this CTA: first item, or -1 when every queue is empty; n = items in it (1..Q.chunk).
// Called by ALL lanes of ONE warp of the CTA; q = the queue to try first (in: the CTA's current queue, out: the queue
// the chunk came from).
__device__ __forceinline__ int sq_fetch(const SmQueues &Q, int &q, int lane, int &n)
{
    unsigned i = 0;
    {
        const int s0 = Q.start[q], s1 = Q.start[q + 1];             // loaded before the atomic, not behind it
        if (lane == 0) i = atomicAdd(Q.next + q, (unsigned)Q.chunk);
        i = __shfl_sync(0xffffffffu, i, 0);
        if (i < (unsigned)(s1 - s0)) { n = min(Q.chunk, s1 - s0 - (int)i); return s0 + (int)i; }
    }
    for (int t0 = 1; t0 < Q.nq; t0 += 32) {                         // 32 queues looked at per round
        const int t = t0 + lane;
        int qq = q + t;
        if (qq >= Q.nq) qq -= Q.nq;
        const bool has = t < Q.nq && sq_peek(Q.next + qq) < (unsigned)(Q.start[qq + 1] - Q.start[qq]);
        unsigned m = __ballot_sync(0xffffffffu, has);
        while (m) {
            const int l = __ffs(m) - 1;
            m &= m - 1;
            int qv = q + t0 + l;
            if (qv >= Q.nq) qv -= Q.nq;
            const int s0 = Q.start[qv], s1 = Q.start[qv + 1];
            if (lane == 0) i = atomicAdd(Q.next + qv, (unsigned)Q.chunk);
            i = __shfl_sync(0xffffffffu, i, 0);
            if (i < (unsigned)(s1 - s0)) { q = qv; n = min(Q.chunk, s1 - s0 - (int)i); return s0 + (int)i; }
        }
    }
    if (lane == 0) {                                                // this CTA is done: the last one resets the counters
        __threadfence();
        if (atomicAdd(Q.next + Q.nq, 1u) == gridDim.x - 1) {
            for (int k = 0; k <= Q.nq; ++k) Q.next[k] = 0;
            __threadfence();
        }
    }
    n = 0;
    return -1;
}

// Next item of a CTA, -1 when there is none.  Static schedule (Q.nq == 0): the CTA's one item is blockIdx.x, then
// -1.  st: three ints of shared memory {item, current queue (static: items taken), items left in the chunk}, set up by
// sq_init.  All threads call it; the state lives in shared memory so that no register is held across the caller's
// streaming loop, and st[0] stays valid until the next call.
__device__ __forceinline__ void sq_init(const SmQueues &Q, int *st)
{
    if (threadIdx.x == 0) { st[1] = Q.nq > 0 ? (int)(sq_smid() % (unsigned)Q.nq) : 0; st[2] = 0; }
}
__device__ __forceinline__ int sq_next_item(const SmQueues &Q, int *st)
{
    __syncthreads();                      // everyone is done with the previous item: st[0] may be read all through it
    if (threadIdx.x < 32) {
        int left = st[2];
        if (left > 0) {                   // the next item of the chunk in hand
            if (threadIdx.x == 0) { st[0] = st[0] + 1; st[2] = left - 1; }
        } else {
            int q = st[1], it, n = 1;
            if (Q.nq > 0) it = sq_fetch(Q, q, (int)threadIdx.x, n);
            else it = q++ == 0 ? (int)blockIdx.x : -1;
            if (threadIdx.x == 0) { st[0] = it; st[1] = q; st[2] = n - 1; }
        }
    }
    __syncthreads();
    return st[0];
}
