// cp_probe.cu -- measurement aids of libcrosspool (`bench.py --probe ...`): tiny kernels that
// have no part in the hot path but make the numbers DESIGN.md quotes reproducible from committed sources.
#include <cuda_runtime.h>
#include <cstdint>
#include "../../include/crosspool.h"
#include "cp_device_common.cuh"

namespace cp {

__global__ void cp_probe_globaltimer_kernel(unsigned long long *out) { *out = global_timer_ns(); }

// Read-only streaming of a contiguous buffer with 16-byte loads, grid-stride, `unroll` loads in flight per
// thread: the HBM read ceiling a TMA-free kernel reaches (SURVEY 8(d) asks for a read-only figure next to
// the copy bandwidth of MEASURED_PEAKS.json).
__global__ void __launch_bounds__(512) cp_probe_read_kernel(const uint4 *src, uint64_t n_vec, unsigned int *sink)
{
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    unsigned int acc = 0;
    for (; i + 7 * stride < n_vec; i += 8 * stride) {
        uint4 v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                         : "=r"(v[k].x), "=r"(v[k].y), "=r"(v[k].z), "=r"(v[k].w) : "l"(src + i + k * stride));
#pragma unroll
        for (int k = 0; k < 8; ++k) acc ^= v[k].x ^ v[k].y ^ v[k].z ^ v[k].w;
    }
    for (; i < n_vec; i += stride) {
        const uint4 v = __ldg(src + i);
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    if (acc == 0x9e3779b9u) *sink = acc;          // keeps the loads alive; practically never taken
}

}  // namespace cp

extern "C" {

cp_status cp_probe_globaltimer(uint64_t *stamp_dev, void *stream)
{
    if (!stamp_dev || ((uintptr_t)stamp_dev & 7u)) return CP_ERR_INVALID_ARG;
    cp::cp_probe_globaltimer_kernel<<<1, 1, 0, (cudaStream_t)stream>>>((unsigned long long *)stamp_dev);
    return cudaGetLastError() == cudaSuccess ? CP_OK : CP_ERR_CUDA;
}

cp_status cp_probe_read_stream(const void *src_dev, uint64_t bytes, int32_t n_ctas, uint32_t *sink_dev, void *stream)
{
    if (!src_dev || !sink_dev || ((uintptr_t)src_dev & 15u) || bytes < 16 || n_ctas < 1) return CP_ERR_INVALID_ARG;
    cp::cp_probe_read_kernel<<<n_ctas, 512, 0, (cudaStream_t)stream>>>((const uint4 *)src_dev, bytes / 16, sink_dev);
    return cudaGetLastError() == cudaSuccess ? CP_OK : CP_ERR_CUDA;
}

}  // extern "C"
