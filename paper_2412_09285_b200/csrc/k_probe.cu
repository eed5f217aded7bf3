// Measurement helper behind fem_probe_l2_read (include/fem.h): the L2 -> SM read rate of this device, the roof the
// L2-resident kernels (Max-SAT step, cfg 3) are compared with in bench.py.  Not on the hot path.
#include "fem_internal.cuh"

namespace fem {

// every thread streams 16-byte loads that bypass L1 (ld.global.cg) over a buffer that fits in L2, `repeats` times
__global__ void __launch_bounds__(256) l2_read_probe_kernel(const float4 *buf, size_t count, int repeats, float *sink) {
    float acc = 0.0f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int rep = 0; rep < repeats; ++rep) {
        size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; k + 3 * stride < count; k += 4 * stride) {  // four loads in flight per thread
            const float4 a = __ldcg(buf + k), b = __ldcg(buf + k + stride), c = __ldcg(buf + k + 2 * stride),
                         d = __ldcg(buf + k + 3 * stride);
            acc += (a.x + b.y) + (c.z + d.w);
        }
        for (; k < count; k += stride) acc += __ldcg(buf + k).x;
    }
    if (acc == 1.2345e-30f) *sink = acc;  // keeps the loads alive; never true for the zero-filled buffer
}

// random-row gather: every warp reads 8 independent, pseudo-randomly chosen rows of `row_bytes` per iteration (16 bytes per
// lane, 32 / (row_bytes / 16) rows per warp instruction), the access pattern of the neighbour gathers of the step kernels
__device__ __forceinline__ uint32_t probe_mix(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}
__global__ void __launch_bounds__(256) l2_gather_probe_kernel(const float4 *buf, uint32_t nrows, int lanes_per_row, int iters, float *sink) {
    const int lane = threadIdx.x & 31;
    const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int rows_per_instr = 32 / lanes_per_row, sub = lane / lanes_per_row, l = lane % lanes_per_row;
    float acc = 0.0f;
    uint32_t ctr = warp * 7919u;
    for (int it = 0; it < iters; ++it) {
        float4 v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t r = probe_mix((ctr++) * (uint32_t)rows_per_instr + (uint32_t)sub) % nrows;
            v[k] = __ldg(buf + (size_t)r * lanes_per_row + l);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += v[k].x + v[k].w;
    }
    if (acc == 1.2345e-30f) *sink = acc;
}

}  // namespace fem

extern "C" fem_status fem_probe_l2_gather(void *buffer, size_t bytes, int32_t row_bytes, int32_t repeats, void *cuda_stream,
                                          double *gigabytes_per_second) {
    using namespace fem;
    if (!buffer || !gigabytes_per_second || bytes < (1u << 20) || bytes > ((size_t)1 << 30) || (bytes & 511) || repeats < 1 ||
        (row_bytes != 64 && row_bytes != 128 && row_bytes != 256 && row_bytes != 512) || (reinterpret_cast<uintptr_t>(buffer) & 15))
        return FEM_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
        return FEM_ECUDA;
    const uint32_t nrows = (uint32_t)((bytes - 512) / (size_t)row_bytes);  // the last 512 bytes hold the sink
    float *sink = reinterpret_cast<float *>(static_cast<char *>(buffer) + bytes - 512);
    if (cudaMemsetAsync(buffer, 0, bytes, st) != cudaSuccess) return FEM_ECUDA;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return FEM_ECUDA;
    const unsigned grid = (unsigned)sms * 8;
    const int lpr = row_bytes / 16;
    l2_gather_probe_kernel<<<grid, 256, 0, st>>>(static_cast<const float4 *>(buffer), nrows, lpr, repeats, sink);  // warm L2
    cudaEventRecord(e0, st);
    l2_gather_probe_kernel<<<grid, 256, 0, st>>>(static_cast<const float4 *>(buffer), nrows, lpr, repeats, sink);
    cudaEventRecord(e1, st);
    float ms = 0.f;
    const bool ok = cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.f;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (!ok) return FEM_ECUDA;
    *gigabytes_per_second = (double)grid * 8.0 * repeats * 8.0 * 512.0 / ((double)ms * 1e-3) / 1e9;  // warps x iterations x rows x 512 B
    return FEM_OK;
}

extern "C" fem_status fem_probe_l2_read(void *buffer, size_t bytes, int32_t repeats, void *cuda_stream, double *gigabytes_per_second) {
    using namespace fem;
    if (!buffer || !gigabytes_per_second || bytes < (1u << 20) || bytes > ((size_t)96 << 20) || (bytes & 15) || repeats < 1 ||
        (reinterpret_cast<uintptr_t>(buffer) & 15))
        return FEM_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
        return FEM_ECUDA;
    const size_t count = (bytes - 16) / 16;  // the last 16 bytes hold the sink
    float *sink = reinterpret_cast<float *>(static_cast<char *>(buffer) + count * 16);
    if (cudaMemsetAsync(buffer, 0, bytes, st) != cudaSuccess) return FEM_ECUDA;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return FEM_ECUDA;
    const unsigned grid = (unsigned)sms * 8;
    l2_read_probe_kernel<<<grid, 256, 0, st>>>(static_cast<const float4 *>(buffer), count, 2, sink);  // warm L2
    cudaEventRecord(e0, st);
    l2_read_probe_kernel<<<grid, 256, 0, st>>>(static_cast<const float4 *>(buffer), count, repeats, sink);
    cudaEventRecord(e1, st);
    float ms = 0.f;
    const bool ok = cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.f;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (!ok) return FEM_ECUDA;
    *gigabytes_per_second = (double)count * 16.0 * repeats / ((double)ms * 1e-3) / 1e9;
    return FEM_OK;
}
