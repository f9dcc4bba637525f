/*
 * vmat_probe.h - C ABI of libvmat_probe.so: a measurement aid for bench.py, NOT part of the product library libvmat
 * (include/vmat.h) and not needed to use it.
 */
#ifndef VMAT_PROBE_H
#define VMAT_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* GB/s of a kernel that does nothing but read `bytes` (>= 1 MiB, rounded down to 32 KiB) of a zeroed scratch buffer,
 * `reps` times back to back after one warm-up pass, with the 256-bit streaming loads of libvmat's dose and price
 * kernels: what a READ-ONLY stream reaches on the current device at the clock it runs at (MEASURED_PEAKS.json's hbm_gbs
 * is a copy: read + write).  Allocates and frees its buffer; synchronous.  gbs host [1] out; launches host [1] out or
 * NULL: kernels launched.  Returns 0, or a negative code (-1 bad argument, -4 out of memory, -5 CUDA error) with the
 * reason in vmat_probe_last_error() (thread-local, never NULL). */
int vmat_hbm_read_probe(int64_t bytes, int32_t reps, double *gbs, int32_t *launches, void *stream);
const char *vmat_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* VMAT_PROBE_H */
