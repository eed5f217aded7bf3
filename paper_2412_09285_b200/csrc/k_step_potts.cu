// Fused annealing step for the q-state Potts kind (balanced minimum cut).
//
// One thread owns VEC consecutive replicas of one variable and all q of its states: softmax of the
// fields, the gather f_i(s) = sum_j W_ij D_j(s) of the centred marginals D = P - 1/q over the CSR row -- each neighbour is a
// row of q*Rb contiguous floats --, g^p from S26 (edge-once reading R1) with the balance
// term 2*lambda*[S_s - P_i(s)] (balance()) and the entropy term (h - lse)/beta, the chain
// rule S20, Adam, and the next marginals.  The column sums S_s = sum_i P_i(s) of the NEXT
// step are produced here as a by-product: per-thread partial sums over a fixed set of variables, a fixed
// shared-memory tree per block, fp64 partials per block, and a tiny second kernel that adds the blocks
// in order -- deterministic, no float atomics.
#include "device_math.cuh"

namespace fem {

template <typename T>
struct PottsParams {
    BlockArrays<T> a;
    DevProblem dp;
    Sc<T> sc;
    const double *S_in;  // [q][Rb] of this block (blockIdx.y stride q*Rb)
    double *partial;     // [gridDim.x][q*Rb] per block (blockIdx.y stride kColBlocks*q*Rb)
    int rv;              // Rb / VEC lanes per variable
    int npb;             // variables per CTA pass = kThreads / rv
};

template <typename T, int QMAX, int VEC, bool STEP>
__global__ void __launch_bounds__(kThreads) potts_kernel(const PottsParams<T> p) {
    using R = Row<T, VEC>;
    __shared__ double red[kThreads];
    const int q = p.dp.q, n = p.dp.n, Rb = p.a.Rb;
    const int nl = threadIdx.x / p.rv;
    const int c = (threadIdx.x - nl * p.rv) * VEC;
    const bool lane_ok = nl < p.npb;
    const int64_t blk = (int64_t)blockIdx.y * p.a.blk_stride;
    const T *__restrict__ gin = p.a.g_in + blk + c;
    const double *__restrict__ S = p.S_in + (int64_t)blockIdx.y * q * Rb;
    const Sc<T> &sc = p.sc;
    const T inv_q = (T)1 / (T)q;

    T colacc[QMAX][VEC];
#pragma unroll
    for (int s = 0; s < QMAX; ++s)
#pragma unroll
        for (int v = 0; v < VEC; ++v) colacc[s][v] = (T)0;

    for (int i = blockIdx.x * p.npb + nl; lane_ok && i < n; i += gridDim.x * p.npb) {
        const int64_t off = blk + (int64_t)i * q * Rb + c;
        T h[QMAX][VEC], P[QMAX][VEC];
#pragma unroll
        for (int s = 0; s < QMAX; ++s) {
            if (s < q) {
                const R r = R::ld_stream(p.a.h + off + (int64_t)s * Rb);
#pragma unroll
                for (int v = 0; v < VEC; ++v) h[s][v] = r.v[v];
            }
        }
        if (STEP) {
            // softmax and log-sum-exp of h(t)
            T lse[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                T mx = h[0][v];
#pragma unroll
                for (int s = 1; s < QMAX; ++s)
                    if (s < q) mx = fmax(mx, h[s][v]);
                T z = (T)0;
#pragma unroll
                for (int s = 0; s < QMAX; ++s)
                    if (s < q) {
                        P[s][v] = fexp(h[s][v] - mx);
                        z += P[s][v];
                    }
                const T rz = frcp(z);
#pragma unroll
                for (int s = 0; s < QMAX; ++s)
                    if (s < q) P[s][v] *= rz;
                lse[v] = mx + flog(z);
            }
            // coupling contraction f(s) = sum_j W_ij P_j(s)
            T f[QMAX][VEC];
#pragma unroll
            for (int s = 0; s < QMAX; ++s)
#pragma unroll
                for (int v = 0; v < VEC; ++v) f[s][v] = (T)0;
            int e0, e1;
            if (p.dp.uniform_deg > 0) {
                e0 = i * p.dp.uniform_deg;
                e1 = e0 + p.dp.uniform_deg;
            } else {
                e0 = __ldg(p.dp.row_ptr + i);
                e1 = __ldg(p.dp.row_ptr + i + 1);
            }
            for (int e = e0; e < e1; ++e) {
                const int j = __ldg(p.dp.col + e);
                const T wj = p.dp.w ? (T)__ldg(p.dp.w + e) : (T)1;
                const T *row = gin + (int64_t)j * q * Rb;
#pragma unroll
                for (int s = 0; s < QMAX; ++s)
                    if (s < q) {
                        const R r = R::ld(row + (int64_t)s * Rb);
#pragma unroll
                        for (int v = 0; v < VEC; ++v) f[s][v] += wj * r.v[v];
                    }
            }
            // g^p (S26, the "+1" of the entropy term cancels in S20), then g^h = P (g^p - <g^p>_P)
            T gbar[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) gbar[v] = (T)0;
#pragma unroll
            for (int s = 0; s < QMAX; ++s)
                if (s < q) {
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T Ss = (T)S[s * Rb + c + v];
                        f[s][v] = -f[s][v] + sc.two_lambda * (Ss - P[s][v]) + (h[s][v] - lse[v]) * sc.inv_beta;
                        gbar[v] += P[s][v] * f[s][v];
                    }
                }
            // Adam per state; h[s] becomes the new (fp32-rounded) field
#pragma unroll
            for (int s = 0; s < QMAX; ++s)
                if (s < q) {
                    R m1 = R::ld_stream(p.a.m1 + off + (int64_t)s * Rb);
                    R m2 = R::ld_stream(p.a.m2 + off + (int64_t)s * Rb);
                    R hn;
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T g = P[s][v] * (f[s][v] - gbar[v]);
                        hn.v[v] = adam_update(h[s][v], g, m1.v[v], m2.v[v], sc);
                        h[s][v] = hn.v[v];
                    }
                    hn.st_stream(p.a.h + off + (int64_t)s * Rb);
                    m1.st_stream(p.a.m1 + off + (int64_t)s * Rb);
                    m2.st_stream(p.a.m2 + off + (int64_t)s * Rb);
                }
        }
        // marginals of the (new) fields -> g_out, and their column sums
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            T mx = h[0][v];
#pragma unroll
            for (int s = 1; s < QMAX; ++s)
                if (s < q) mx = fmax(mx, h[s][v]);
            T z = (T)0;
#pragma unroll
            for (int s = 0; s < QMAX; ++s)
                if (s < q) {
                    P[s][v] = fexp(h[s][v] - mx);
                    z += P[s][v];
                }
            const T rz = frcp(z);
#pragma unroll
            for (int s = 0; s < QMAX; ++s)
                if (s < q) P[s][v] *= rz;
        }
#pragma unroll
        for (int s = 0; s < QMAX; ++s)
            if (s < q) {
                R po;
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    // centred marginal D = P - 1/q: constants in s cancel in S20, and near the uniform start
                    // the deviation is all the signal, so it is what gets stored and gathered
                    po.v[v] = P[s][v] - inv_q;
                    colacc[s][v] += po.v[v];  // sum what the next step will gather
                }
                po.st(p.a.g_out + off + (int64_t)s * Rb);
            }
    }

    // block reduction over the npb variable slots, fixed order, fp64; one partial row per CTA
    double *part = p.partial + ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * q * Rb;
#pragma unroll
    for (int s = 0; s < QMAX; ++s) {
        if (s < q) {  // q is uniform over the CTA, so the barriers below are too
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                __syncthreads();
                red[threadIdx.x] = lane_ok ? (double)colacc[s][v] : 0.0;
                __syncthreads();
                if (nl == 0 && lane_ok) {
                    double acc = 0.0;
                    for (int k = 0; k < p.npb; ++k) acc += red[k * p.rv + threadIdx.x];
                    part[s * Rb + c + v] = acc;
                }
            }
        }
    }
}

// S[s][a] = sum over CTAs of the partial rows, in CTA order (deterministic), fp64.
__global__ void __launch_bounds__(kThreads) potts_colsum_kernel(const double *partial, double *S, int nparts, int qR) {
    const int k = blockIdx.x * kThreads + threadIdx.x;
    if (k >= qR) return;
    const double *pp = partial + (int64_t)blockIdx.y * nparts * qR;
    double acc = 0.0;
    for (int b = 0; b < nparts; ++b) acc += pp[(int64_t)b * qR + k];
    S[(int64_t)blockIdx.y * qR + k] = acc;
}

template <typename T, int QMAX, int VEC>
static void launch_potts_t(Handle *hd, const PottsParams<T> &p, dim3 grid, bool step) {
    if (step)
        potts_kernel<T, QMAX, VEC, true><<<grid, kThreads, 0, hd->stream>>>(p);
    else
        potts_kernel<T, QMAX, VEC, false><<<grid, kThreads, 0, hd->stream>>>(p);
}

template <typename T>
static void launch_potts_q(Handle *hd, PottsParams<T> &p, dim3 grid, bool step, int vec) {
    const int q = hd->dp.q;
    if (q <= 4) {
        if (vec == 4) launch_potts_t<T, 4, 4>(hd, p, grid, step);
        else if (vec == 2) launch_potts_t<T, 4, 2>(hd, p, grid, step);
        else launch_potts_t<T, 4, 1>(hd, p, grid, step);
    } else if (q <= 8) {
        if (vec >= 2) launch_potts_t<T, 8, 2>(hd, p, grid, step);
        else launch_potts_t<T, 8, 1>(hd, p, grid, step);
    } else if (q <= 16) {
        launch_potts_t<T, 16, 1>(hd, p, grid, step);
    } else {
        launch_potts_t<T, 32, 1>(hd, p, grid, step);
    }
}

int potts_vec(const Handle *hd) {
    const int q = hd->dp.q, Rb = hd->Rb;
    if (q <= 4) return Rb % 4 == 0 ? 4 : (Rb % 2 == 0 ? 2 : 1);
    if (q <= 8) return Rb % 2 == 0 ? 2 : 1;
    return 1;
}

template <typename T>
static void launch_potts_typed(Handle *hd, const StepScalars &sc, bool step, int blk_begin, int blk_count) {
    using S = StateOf<T>;
    const int Rb = hd->Rb, q = hd->dp.q;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    PottsParams<T> p;
    p.a.h = S::h(hd) + base;
    p.a.m1 = S::m1(hd) + base;
    p.a.m2 = S::m2(hd) + base;
    p.a.g_in = S::g(hd, hd->cur) + base;
    p.a.g_out = (step ? S::g(hd, hd->cur ^ 1) : S::g(hd, hd->cur)) + base;
    p.a.blk_stride = hd->rows * Rb;
    p.a.Rb = Rb;
    p.dp = hd->dp;
    p.sc = Sc<T>(sc);
    p.S_in = hd->colsum[hd->cur] + (int64_t)blk_begin * q * Rb;
    p.partial = hd->colpart + (int64_t)blk_begin * kColBlocks * q * Rb;
    const int vec = potts_vec(hd);  // fem_anneal keeps Rb / vec <= kThreads (one variable inside one CTA pass)
    p.rv = Rb / vec;
    p.npb = kThreads / p.rv;
    const int nblk = (int)std::min<int64_t>(kColBlocks, ceil_div(hd->dp.n, p.npb));
    dim3 grid((unsigned)nblk, (unsigned)blk_count);
    launch_potts_q<T>(hd, p, grid, step, vec);
    double *S_out = (step ? hd->colsum[hd->cur ^ 1] : hd->colsum[hd->cur]) + (int64_t)blk_begin * q * Rb;
    dim3 g2((unsigned)ceil_div((int64_t)q * Rb, kThreads), (unsigned)blk_count);
    potts_colsum_kernel<<<g2, kThreads, 0, hd->stream>>>(p.partial, S_out, nblk, q * Rb);
    hd->launches += 2;
}

// step == false: centred marginals + column sums of the current fields into g[cur] / colsum[cur] (t = 0).
void launch_potts(Handle *hd, const StepScalars &sc, bool wide, bool step, int blk_begin, int blk_count) {
    if (wide) launch_potts_typed<double>(hd, sc, step, blk_begin, blk_count);
    else launch_potts_typed<float>(hd, sc, step, blk_begin, blk_count);
}

// Marginals hook: P = softmax(h) in the device layout, written as fp32.
template <typename T>
__global__ void __launch_bounds__(kThreads) potts_softmax_kernel(const T *h, float *out, int n, int q, int Rb,
                                                                 int nblocks, int64_t blk_stride) {
    const int64_t per = (int64_t)n * Rb;
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= per * nblocks) return;
    const int64_t b = idx / per, rem = idx - b * per;
    const int64_t i = rem / Rb, r = rem - i * Rb;
    const int64_t off = b * blk_stride + i * q * Rb + r;
    T mx = h[off];
    for (int s = 1; s < q; ++s) mx = fmax(mx, h[off + (int64_t)s * Rb]);
    T z = (T)0;
    for (int s = 0; s < q; ++s) z += fexp(h[off + (int64_t)s * Rb] - mx);
    for (int s = 0; s < q; ++s) out[off + (int64_t)s * Rb] = (float)(fexp(h[off + (int64_t)s * Rb] - mx) / z);
}

void launch_potts_softmax(Handle *hd, float *out) {
    const int nb = hd->R / hd->Rb;
    const int64_t total = (int64_t)hd->dp.n * hd->Rb * nb;
    const unsigned grid = (unsigned)ceil_div(total, kThreads);
    if (hd->wide_live)
        potts_softmax_kernel<double><<<grid, kThreads, 0, hd->stream>>>(hd->hW, out, hd->dp.n, hd->dp.q, hd->Rb, nb,
                                                                        hd->rows * hd->Rb);
    else
        potts_softmax_kernel<float><<<grid, kThreads, 0, hd->stream>>>(hd->h, out, hd->dp.n, hd->dp.q, hd->Rb, nb,
                                                                       hd->rows * hd->Rb);
    hd->launches++;
}

}  // namespace fem
