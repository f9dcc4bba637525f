// read_probe.cu - libvmat_probe.so, a measurement aid kept OUT of libvmat (include/vmat_probe.h): what a read-only
// stream reaches on this device.  The streaming kernels of libvmat only READ the matrix, while the copy benchmark
// behind MEASURED_PEAKS.json reads and writes; this kernel reads a buffer with the same 256-bit L1::no_allocate /
// L2::evict_first loads (csrc/common.cuh), four per thread, and nothing else: the ceiling of that access pattern at the
// clock the device runs at.  bench.py reports it as roofline.read_only_stream, beside the copy peak, as context.
#include "../common.cuh"
#include "../../../include/vmat_probe.h"
#include <stdarg.h>

static thread_local char g_probe_err[256] = "";
static int probe_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_probe_err, sizeof(g_probe_err), fmt, ap);
    va_end(ap);
    return code;
}

__global__ void __launch_bounds__(256) k_read_probe(const char *__restrict__ buf, size_t n32, uint32_t *__restrict__ sink)
{
    const size_t i = (size_t)blockIdx.x * 1024 + threadIdx.x;
    if (i + 768 < n32) {
        Vec8 r[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) r[u] = ld_stream_256(buf + (i + (size_t)u * 256) * 32);
        uint32_t acc = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int k = 0; k < 8; ++k) acc ^= r[u].w[k];
        if (acc == 0x9e3779b9u) sink[0] = acc;                     // never true for a zeroed buffer: keeps the loads
    }
}

extern "C" const char *vmat_probe_last_error(void) { return g_probe_err; }

extern "C" int vmat_hbm_read_probe(int64_t bytes, int32_t reps, double *gbs, int32_t *launches, void *stream)
{
    if (gbs == nullptr || reps < 1 || bytes < ((int64_t)1 << 20))
        return probe_fail(-1, "vmat_hbm_read_probe: gbs is NULL, reps < 1 or bytes < 1 MiB");
    cudaStream_t st = (cudaStream_t)stream;
    char *buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    bytes &= ~(int64_t)32767;
    cudaError_t e = cudaMalloc((void **)&buf, (size_t)bytes + 4);
    if (e != cudaSuccess) { cudaGetLastError(); return probe_fail(-4, "vmat_hbm_read_probe: cudaMalloc -> %s", cudaGetErrorString(e)); }
    uint32_t *sink = (uint32_t *)(buf + bytes);
    e = cudaMemsetAsync(buf, 0, (size_t)bytes + 4, st);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    const size_t n32 = (size_t)bytes / 32;
    const unsigned grid = (unsigned)((n32 + 1023) / 1024);
    int n_launch = 0;
    if (e == cudaSuccess) { k_read_probe<<<grid, 256, 0, st>>>(buf, n32, sink); ++n_launch; e = cudaEventRecord(e0, st); }   // warm-up
    for (int r = 0; r < reps && e == cudaSuccess; ++r) { k_read_probe<<<grid, 256, 0, st>>>(buf, n32, sink); ++n_launch; }
    if (e == cudaSuccess) e = cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return probe_fail(-5, "vmat_hbm_read_probe: %s", cudaGetErrorString(e));
    *gbs = (double)bytes * reps / ((double)ms * 1e-3) / 1e9;
    if (launches) *launches = n_launch;
    return 0;
}
