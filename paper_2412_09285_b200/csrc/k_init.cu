// Initial fields, layout transposes and the marginals hook.
#include "device_math.cuh"

namespace fem {

// Device offset of logical element (replica a, row = i*F + s).
__device__ __forceinline__ int64_t dev_off(int a, int64_t row, int Rb, int64_t blk_stride) {
    const int b = a / Rb;
    return (int64_t)b * blk_stride + row * Rb + (a - b * Rb);
}

__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

// h(0) = scale * N(0,1) from the counter-based generator of DESIGN.md section 3
// (R4): keyed on the LOGICAL index c = a*n*F + row, so replica a does not depend on R or on the layout.
__global__ void __launch_bounds__(kThreads) init_fields_kernel(float *h, unsigned long long seed, double scale, int R,
                                                               int64_t nF, int Rb, int64_t blk_stride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= nF * R) return;
    // thread order follows the device layout so stores coalesce: idx = (b*nF + row)*Rb + r
    const int64_t per = nF * Rb;
    const int b = (int)(idx / per);
    const int64_t rem = idx - (int64_t)b * per;
    const int64_t row = rem / Rb;
    const int r = (int)(rem - row * Rb);
    const int a = b * Rb + r;
    const unsigned long long G = 0x9E3779B97F4A7C15ULL;
    const unsigned long long x = mix64(seed + G);
    const unsigned long long c = (unsigned long long)a * (unsigned long long)nF + (unsigned long long)row;
    const unsigned long long r1 = mix64(x + (2ULL * c + 1ULL) * G);
    const unsigned long long r2 = mix64(x + (2ULL * c + 2ULL) * G);
    const double U1 = ((double)(r1 >> 11) + 1.0) * 0x1.0p-53;
    const double U2 = (double)(r2 >> 11) * 0x1.0p-53;
    const double z = sqrt(-2.0 * log(U1)) * cos(6.283185307179586476925286766559 * U2);
    h[(int64_t)b * blk_stride + rem] = (float)(scale * z);
}

// logical [R][nF] <-> device layout
template <typename TS, typename TT, bool IN>
__global__ void __launch_bounds__(kThreads) transpose_kernel(const TS *src, TT *dst, int R, int64_t nF, int Rb,
                                                             int64_t blk_stride) {
    __shared__ TT tile[32][33];
    // tile over (row, a): 32 rows x 32 replicas
    const int64_t row0 = (int64_t)blockIdx.x * 32;
    const int a0 = blockIdx.y * 32;
    const int tx = threadIdx.x % 32, ty = threadIdx.x / 32;  // 32 x 8
    if (IN) {
        for (int k = ty; k < 32; k += 8) {  // read logical: contiguous in row
            const int a = a0 + k;
            const int64_t row = row0 + tx;
            if (a < R && row < nF) tile[k][tx] = (TT)src[(int64_t)a * nF + row];
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {  // write device: contiguous in a
            const int64_t row = row0 + k;
            const int a = a0 + tx;
            if (a < R && row < nF) dst[dev_off(a, row, Rb, blk_stride)] = tile[tx][k];
        }
    } else {
        for (int k = ty; k < 32; k += 8) {
            const int64_t row = row0 + k;
            const int a = a0 + tx;
            if (a < R && row < nF) tile[tx][k] = (TT)src[dev_off(a, row, Rb, blk_stride)];
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {
            const int a = a0 + k;
            const int64_t row = row0 + tx;
            if (a < R && row < nF) dst[(int64_t)a * nF + row] = tile[k][tx];
        }
    }
}

__global__ void __launch_bounds__(kThreads) zero_kernel(float *a, float *b, int64_t count) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx < count) {
        a[idx] = 0.f;
        b[idx] = 0.f;
    }
}

// Two-state marginals P(state 1) = sigmoid(h) in the device layout, written as fp32.
template <typename T>
__global__ void __launch_bounds__(kThreads) sigmoid_kernel(const T *h, float *out, int64_t per, int nblocks,
                                                           int64_t blk_stride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= per * nblocks) return;
    const int64_t b = idx / per;
    const int64_t off = b * blk_stride + (idx - b * per);  // skips the pad row of every block
    out[off] = (float)sigmoid_of(h[off]);
}

// wide phase entry: fp64 copy of the fields, zero fp64 moments
__global__ void __launch_bounds__(kThreads) widen_kernel(const float *h, double *hW, double *m1W, double *m2W,
                                                         int64_t count) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx < count) {
        hW[idx] = (double)h[idx];
        m1W[idx] = 0.0;
        m2W[idx] = 0.0;
    }
}

// wide phase exit: round the fp64 state to the fp32 arrays the bulk of the anneal runs on
__global__ void __launch_bounds__(kThreads) narrow_kernel(const double *hW, const double *m1W, const double *m2W,
                                                          const double *gW, float *h, float *m1, float *m2, float *g,
                                                          float *g_other, int64_t count, int fields_only) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx < count) {
        h[idx] = (float)hW[idx];
        if (fields_only != 1) {
            m1[idx] = (float)m1W[idx];
            m2[idx] = (float)m2W[idx];
            if (fields_only == 0) {  // 2: the gather arrays hold bytes shared by both precisions (manipulated gradients)
                g[idx] = (float)gW[idx];
                g_other[idx] = (float)gW[idx];  // carries the constant-1 pad rows into both buffers
            }
        }
    }
}

void launch_init_fields(Handle *hd, uint64_t seed, double scale) {
    const int64_t nF = (int64_t)hd->dp.n * hd->dp.F;
    const int64_t total = nF * hd->R;
    init_fields_kernel<<<(unsigned)ceil_div(total, kThreads), kThreads, 0, hd->stream>>>(
        hd->h, seed, scale, hd->R, nF, hd->Rb, hd->rows * hd->Rb);
    hd->launches++;
}

void launch_zero_moments(Handle *hd) {
    const int64_t count = hd->rows * (int64_t)hd->R;
    zero_kernel<<<(unsigned)ceil_div(count, kThreads), kThreads, 0, hd->stream>>>(hd->m1, hd->m2, count);
    hd->launches++;
}

void launch_widen(Handle *hd) {
    const int64_t count = hd->rows * (int64_t)hd->R;
    widen_kernel<<<(unsigned)ceil_div(count, kThreads), kThreads, 0, hd->stream>>>(hd->h, hd->hW, hd->m1W, hd->m2W, count);
    hd->launches++;
}

void launch_narrow(Handle *hd, bool fields_only) {
    const int64_t count = hd->rows * (int64_t)hd->R;
    narrow_kernel<<<(unsigned)ceil_div(count, kThreads), kThreads, 0, hd->stream>>>(
        hd->hW, hd->m1W, hd->m2W, hd->gW[hd->cur], hd->h, hd->m1, hd->m2, hd->g[hd->cur], hd->g[hd->cur ^ 1], count,
        fields_only ? 1 : (hd->gather_disc ? 2 : 0));
    hd->launches++;
}

void launch_transpose_in(Handle *hd, const float *logical_dev, float *dst) {
    const int64_t nF = (int64_t)hd->dp.n * hd->dp.F;
    dim3 grid((unsigned)ceil_div(nF, 32), (unsigned)ceil_div(hd->R, 32));
    transpose_kernel<float, float, true><<<grid, kThreads, 0, hd->stream>>>(logical_dev, dst, hd->R, nF, hd->Rb,
                                                                            hd->rows * hd->Rb);
    hd->launches++;
}

void launch_transpose_out(Handle *hd, const float *src, float *logical_dev) {
    const int64_t nF = (int64_t)hd->dp.n * hd->dp.F;
    dim3 grid((unsigned)ceil_div(nF, 32), (unsigned)ceil_div(hd->R, 32));
    transpose_kernel<float, float, false><<<grid, kThreads, 0, hd->stream>>>(src, logical_dev, hd->R, nF, hd->Rb,
                                                                             hd->rows * hd->Rb);
    hd->launches++;
}

void launch_transpose_out_wide(Handle *hd, const double *src, float *logical_dev) {
    const int64_t nF = (int64_t)hd->dp.n * hd->dp.F;
    dim3 grid((unsigned)ceil_div(nF, 32), (unsigned)ceil_div(hd->R, 32));
    transpose_kernel<double, float, false><<<grid, kThreads, 0, hd->stream>>>(src, logical_dev, hd->R, nF, hd->Rb,
                                                                              hd->rows * hd->Rb);
    hd->launches++;
}

void launch_sigmoid(Handle *hd, float *out) {
    const int64_t per = (int64_t)hd->dp.n * hd->dp.F * hd->Rb;
    const int nb = hd->R / hd->Rb;
    const unsigned grid = (unsigned)ceil_div(per * nb, kThreads);
    if (hd->wide_live)
        sigmoid_kernel<double><<<grid, kThreads, 0, hd->stream>>>(hd->hW, out, per, nb, hd->rows * hd->Rb);
    else
        sigmoid_kernel<float><<<grid, kThreads, 0, hd->stream>>>(hd->fields(), out, per, nb, hd->rows * hd->Rb);
    hd->launches++;
}

}  // namespace fem
