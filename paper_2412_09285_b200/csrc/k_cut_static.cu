// fem_cut_static: cut values (Eq.6) of a batch of two-state configurations WITHOUT ANY ALLOCATION, for
// callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// It is a variant of the readout's energy_graph_kernel (k_readout.cu): a warp covers 32 configurations (lane =
// configuration, so the loads of a variable's row coalesce), the 8 warps of a CTA are 8 chunks that stride over the
// variables, every chunk writes one partial sum per configuration and a second kernel adds the chunks in ascending order
// (integer sums: exact whatever the order).  The existing path keeps those partials in the workspace the caller hands to
// fem_create; here they live in a file-scope `static __device__` array of kCutStaticScratchBytes (2 MiB), which every GPU
// that loads the library holds until the process exits.
//
// In host code the array's NAME is a host-side stand-in, not a device address, so the kernels are given the address that
// cudaGetSymbolAddress returns -- looked up once per device, with that device current, on the first call there.
//
// Every call on a device shares the array and finds in it what the previous call left.  Nothing has to start at zero: the
// first kernel writes every partial the second one reads, so no clearing is needed.  Two calls whose kernels can overlap on
// the GPU (different streams without an ordering between them, or two host threads on different streams) RACE on the
// array; calls on one stream are ordered and safe.
#include <mutex>
#include <string>

#include "fem_internal.cuh"

namespace fem {

constexpr size_t kCutStaticScratchBytes = (size_t)FEM_CUT_STATIC_SCRATCH_BYTES;
constexpr int kCutStaticMaxDevices = 64;

static __device__ __align__(256) unsigned char g_cut_static_scratch[kCutStaticScratchBytes];

static std::mutex g_cut_static_mutex;
static void *g_cut_static_ptr[kCutStaticMaxDevices] = {};  // device address of the array, per device ordinal
static thread_local std::string g_cut_static_error;

// partial cut of chunk `chunk` for configuration a: every edge once (j > i), weights rounded to integers as in the readout
__global__ void __launch_bounds__(kThreads) cut_static_partial_kernel(const int *__restrict__ row_ptr, const int *__restrict__ col,
                                                                       const float *__restrict__ w, const int8_t *__restrict__ sigma,
                                                                       int n, int count, int nchunks, long long *part) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.y * 32 + lane;
    const int chunk = blockIdx.x * 8 + warp;
    if (a >= count) return;
    long long acc = 0;
    for (int i = chunk; i < n; i += nchunks) {
        const int ci = sigma[(int64_t)i * count + a];
        const int e0 = __ldg(row_ptr + i), e1 = __ldg(row_ptr + i + 1);
        for (int e = e0; e < e1; ++e) {
            const int j = __ldg(col + e);
            if (j <= i) continue;
            const int cj = sigma[(int64_t)j * count + a];
            if (ci != cj) acc += w ? llrintf(__ldg(w + e)) : 1ll;
        }
    }
    part[(int64_t)chunk * count + a] = acc;
}

// one warp per configuration: the chunks' partials, lanes striding over the chunks, then a butterfly
__global__ void __launch_bounds__(kThreads) cut_static_sum_kernel(const long long *__restrict__ part, int count, int nchunks,
                                                                   long long *__restrict__ cut) {
    const int a = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (a >= count) return;  // warp-uniform
    long long s = 0;
    for (int c = lane; c < nchunks; c += 32) s += part[(int64_t)c * count + a];
#pragma unroll
    for (int k = 16; k > 0; k >>= 1) s += __shfl_xor_sync(0xffffffffu, s, k);
    if (lane == 0) cut[a] = s;
}

static fem_status cut_static_fail(fem_status st, const std::string &msg) {
    g_cut_static_error = msg;
    return st;
}

// device address of the scratch array on the current device (looked up once per device)
static fem_status cut_static_scratch(long long **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cut_static_fail(FEM_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kCutStaticMaxDevices) return cut_static_fail(FEM_EINVAL, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_cut_static_mutex);
    if (!g_cut_static_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_cut_static_scratch);
        if (e != cudaSuccess || !ptr)
            return cut_static_fail(FEM_ECUDA, std::string("cudaGetSymbolAddress(scratch): ") + cudaGetErrorString(e));
        g_cut_static_ptr[dev] = ptr;
    }
    *out = reinterpret_cast<long long *>(g_cut_static_ptr[dev]);
    return FEM_OK;
}

}  // namespace fem

extern "C" {

fem_status fem_cut_static(int32_t n, const int32_t *row_ptr, const int32_t *col_idx, const float *weight, const int8_t *sigma,
                          int32_t count, int64_t *cut, void *cuda_stream) {
    using namespace fem;
    if (n < 1) return cut_static_fail(FEM_EINVAL, "fem_cut_static: n must be >= 1");
    if (count < 1) return cut_static_fail(FEM_EINVAL, "fem_cut_static: count must be >= 1");
    if (count > FEM_CUT_STATIC_MAX_COUNT)
        return cut_static_fail(FEM_EINVAL, "fem_cut_static: count " + std::to_string(count) + " exceeds FEM_CUT_STATIC_MAX_COUNT = " +
                                               std::to_string(FEM_CUT_STATIC_MAX_COUNT) + " (the static scratch array holds " +
                                               std::to_string(kCutStaticScratchBytes) + " bytes of partial sums); split the batch");
    if (!row_ptr || !col_idx || !sigma || !cut) return cut_static_fail(FEM_EINVAL, "fem_cut_static: null pointer");
    long long *part = nullptr;
    const fem_status st = cut_static_scratch(&part);
    if (st != FEM_OK) return st;
    // chunks: 8 per CTA, at most 148 CTAs (one per SM), at least 16 variables per chunk, and what the array holds
    const int64_t cap_chunks = (int64_t)(kCutStaticScratchBytes / 8) / count;  // >= 64 at the maximum count
    int64_t blocks = std::min<int64_t>(148, ceil_div(n, 8 * 16));
    blocks = std::max<int64_t>(1, std::min<int64_t>(blocks, cap_chunks / 8));
    const int nchunks = (int)blocks * 8;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    const dim3 grid((unsigned)blocks, (unsigned)ceil_div(count, 32));
    cut_static_partial_kernel<<<grid, kThreads, 0, stream>>>(row_ptr, col_idx, weight, sigma, n, count, nchunks, part);
    cut_static_sum_kernel<<<(unsigned)ceil_div(count, kThreads / 32), kThreads, 0, stream>>>(part, count, nchunks,
                                                                                           reinterpret_cast<long long *>(cut));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cut_static_fail(FEM_ECUDA, std::string("fem_cut_static launch: ") + cudaGetErrorString(e));
    return FEM_OK;
}

const char *fem_cut_static_error(void) { return fem::g_cut_static_error.c_str(); }

}  // extern "C"
