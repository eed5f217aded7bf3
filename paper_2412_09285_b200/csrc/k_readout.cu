// Readout: rounding (Eq.4), per-replica energies (Eq.6-8; Ising
// PAPER.md:43) and the best-replica argmin (Eq.5).  Integer work is exact; the two-level
// reduction (per-chunk partials, then chunks in order) makes the fp64 sums deterministic too.
//
// Mapping: a warp covers 32 consecutive replicas (lane = replica, so loads of a variable's row coalesce);
// the 8 warps of a CTA are 8 "chunks" that stride over variables / clauses / matrix rows.
#include "device_math.cuh"

namespace fem {

struct ReadoutParams {
    DevProblem dp;
    const int8_t *cfg;   // [blocks][n][Rb]
    int R, Rb;
    int64_t cstride;     // n * Rb
    int nchunks;
    long long *part_i;   // [nchunks][R]
    double *part_d;      // [nchunks][R]
    int *part_cnt;       // [nchunks][q][R]  (Potts)
};

__device__ __forceinline__ int64_t cfg_off(int a, int i, int Rb, int64_t cstride) {
    const int b = a / Rb;
    return (int64_t)b * cstride + (int64_t)i * Rb + (a - b * Rb);
}

// sigma from the fields: two-state 1 iff h > 0; Potts: lowest s among the maxima of h_i(.)  (reading R3)
template <typename T>
__global__ void __launch_bounds__(kThreads) round_kernel(const T *h, int8_t *cfg, int n, int F, int R, int Rb,
                                                         int64_t blk_stride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= (int64_t)n * R) return;
    const int64_t per = (int64_t)n * Rb;
    const int b = (int)(idx / per);
    const int64_t rem = idx - (int64_t)b * per;
    const int i = (int)(rem / Rb), r = (int)(rem - (int64_t)i * Rb);
    const T *hp = h + (int64_t)b * blk_stride + (int64_t)i * F * Rb + r;
    int best = 0;
    if (F == 1) {
        best = hp[0] > (T)0 ? 1 : 0;
    } else {
        T bv = hp[0];
        for (int s = 1; s < F; ++s) {
            const T v = hp[(int64_t)s * Rb];
            if (v > bv) {
                bv = v;
                best = s;
            }
        }
    }
    cfg[(int64_t)b * per + rem] = (int8_t)best;
}

template <int KIND>
__global__ void __launch_bounds__(kThreads) energy_graph_kernel(const ReadoutParams p) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.y * 32 + lane;
    const int chunk = blockIdx.x * 8 + warp;
    const bool ok = a < p.R;
    const int n = p.dp.n, q = p.dp.q;
    long long acc_i = 0;
    double acc_d = 0.0;
    int cnt[KIND == FEM_BMINCUT ? kMaxQ : 1];
#pragma unroll
    for (int k = 0; k < (KIND == FEM_BMINCUT ? kMaxQ : 1); ++k) cnt[k] = 0;
    const int8_t *cf = p.cfg + (ok ? cfg_off(a, 0, p.Rb, p.cstride) : 0);
    for (int i = chunk; ok && i < n; i += p.nchunks) {
        const int ci = cf[(int64_t)i * p.Rb];
        const int e0 = __ldg(p.dp.row_ptr + i), e1 = __ldg(p.dp.row_ptr + i + 1);
        for (int e = e0; e < e1; ++e) {
            const int j = __ldg(p.dp.col + e);
            if (j <= i) continue;  // every edge once
            const int cj = cf[(int64_t)j * p.Rb];
            const float w = p.dp.w ? __ldg(p.dp.w + e) : 1.0f;
            if (KIND == FEM_ISING) {
                const int ss = (2 * ci - 1) * (2 * cj - 1);
                acc_d -= (double)w * (double)ss;
            } else if (ci != cj) {
                acc_i += llrintf(w);
                acc_d += (double)w;
            }
        }
        if (KIND == FEM_BMINCUT) {
            const int vi = p.dp.vw ? (int)llrintf(__ldg(p.dp.vw + i)) : 1;  // part sizes are sums of node weights (S35)
#pragma unroll
            for (int k = 0; k < kMaxQ; ++k) cnt[k] += (ci == k) ? vi : 0;
        }
    }
    if (ok) {
        p.part_i[(int64_t)chunk * p.R + a] = acc_i;
        p.part_d[(int64_t)chunk * p.R + a] = acc_d;
        if (KIND == FEM_BMINCUT) {
#pragma unroll
            for (int k = 0; k < kMaxQ; ++k)
                if (k < q) p.part_cnt[((int64_t)chunk * q + k) * p.R + a] = cnt[k];
        }
    }
}

// number of clauses whose every literal is false (Eq.8)
__global__ void __launch_bounds__(kThreads) energy_sat_kernel(const ReadoutParams p) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.y * 32 + lane;
    const int chunk = blockIdx.x * 8 + warp;
    if (a >= p.R) return;
    const int8_t *cf = p.cfg + cfg_off(a, 0, p.Rb, p.cstride);
    long long unsat = 0;
    for (int c = chunk; c < p.dp.m; c += p.nchunks) {
        const int x0 = __ldg(p.dp.clause_ptr + c), x1 = __ldg(p.dp.clause_ptr + c + 1);
        bool sat = false;
        for (int x = x0; x < x1; ++x) {
            const int lit = __ldg(p.dp.lits + x);
            const int v = (lit > 0 ? lit : -lit) - 1;
            const int s = cf[(int64_t)v * p.Rb];
            // non-Boolean SAT: satisfied when some variable takes its clause value W_mi
            if (p.dp.lit_state) sat = sat || (s == __ldg(p.dp.lit_state + x));
            else sat = sat || ((lit > 0) == (s == 1));
        }
        unsat += sat ? 0 : 1;
    }
    p.part_i[(int64_t)chunk * p.R + a] = unsat;
    p.part_d[(int64_t)chunk * p.R + a] = (double)unsat;
}

// dense Ising: E = -sum_{i<j} J_ij s_i s_j in fp64
__global__ void __launch_bounds__(kThreads) energy_dense_kernel(const ReadoutParams p) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.y * 32 + lane;
    const int chunk = blockIdx.x * 8 + warp;
    if (a >= p.R) return;
    const int n = p.dp.n;
    const int8_t *cf = p.cfg + cfg_off(a, 0, p.Rb, p.cstride);
    double acc = 0.0;
    for (int i = chunk; i < n; i += p.nchunks) {
        const float *Ji = p.dp.J + (int64_t)i * n;
        double row = 0.0;
        for (int j = i + 1; j < n; ++j) {
            const int sj = 2 * cf[(int64_t)j * p.Rb] - 1;
            row += (double)__ldg(Ji + j) * (double)sj;
        }
        acc -= row * (double)(2 * cf[(int64_t)i * p.Rb] - 1);
    }
    p.part_i[(int64_t)chunk * p.R + a] = 0;
    p.part_d[(int64_t)chunk * p.R + a] = acc;
}

// Dense Ising on the fp64 tensor-core GEMM: S = +-1 spins as doubles, F = J * S (launch_dense_field_f64), then
// E_a = -1/2 sum_i S_ia F_ia (J symmetric with zero diagonal: sum_i s_i (J s)_i = 2 sum_{i<j} J_ij s_i s_j).
__global__ void __launch_bounds__(kThreads) spins_f64_kernel(const int8_t *cfg, double *S, int n, int R, int Rb, int64_t cstride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= (int64_t)n * R) return;
    const int i = (int)(idx / R), a = (int)(idx - (int64_t)i * R);
    S[idx] = (double)(2 * cfg[cfg_off(a, i, Rb, cstride)] - 1);
}

__global__ void __launch_bounds__(kThreads) energy_dense_reduce_kernel(const double *S, const double *F, int n, int R, int nchunks,
                                                                       long long *part_i, double *part_d) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = blockIdx.y * 32 + lane;
    const int chunk = blockIdx.x * 8 + warp;
    if (a >= R) return;
    double acc = 0.0;
    for (int i = chunk; i < n; i += nchunks) acc += S[(int64_t)i * R + a] * F[(int64_t)i * R + a];
    part_i[(int64_t)chunk * R + a] = 0;
    part_d[(int64_t)chunk * R + a] = -0.5 * acc;
}

void launch_dense_field_f64(Handle *hd, const double *M, double *C, int n, int R);  // k_step_q2.cu

struct FinalizeParams {
    int kind, n, q, R, nchunks, integral;
    double lambda;
    double vtotal;  // sum of the node weights (n without them)
    const long long *part_i;
    const double *part_d;
    const int *part_cnt;
    long long *e_int;
    double *e_real;
    int *part;  // [R][q]
};

// One warp per replica: lane l adds chunks l, l+32, ... in index order, then a fixed butterfly adds the 32 lane sums
// (a fixed order, so the fp64 sum is the same run to run; the integer sums do not depend on the order at all).
__global__ void __launch_bounds__(kThreads) energy_finalize_kernel(const FinalizeParams p) {
    const int a = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (a >= p.R) return;  // warp-uniform
    long long si = 0;
    double sd = 0.0;
    for (int c = lane; c < p.nchunks; c += 32) {
        si += p.part_i[(int64_t)c * p.R + a];
        sd += p.part_d[(int64_t)c * p.R + a];
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        si += __shfl_xor_sync(0xffffffffu, si, s);
        sd += __shfl_xor_sync(0xffffffffu, sd, s);
    }
    if (p.integral && p.kind != FEM_ISING) sd = (double)si;
    long long ei = 0;
    double er = 0.0;
    if (p.kind == FEM_MAXCUT) {
        ei = -si;
        er = -sd;
    } else if (p.kind == FEM_MAXSAT) {
        ei = si;
        er = sd;
    } else if (p.kind == FEM_ISING) {
        ei = 0;
        er = sd;
    } else {  // BMINCUT: cut + lambda * sum_k (n_k - n/q)^2, k ascending, no FMA contraction
        double pen = 0.0;
        const double target = __ddiv_rn(p.vtotal, (double)p.q);
        for (int k = 0; k < p.q; ++k) {
            int ck = 0;
            for (int c = lane; c < p.nchunks; c += 32) ck += p.part_cnt[((int64_t)c * p.q + k) * p.R + a];
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) ck += __shfl_xor_sync(0xffffffffu, ck, s);
            if (lane == 0) p.part[(int64_t)a * p.q + k] = ck;
            const double d = __dsub_rn((double)ck, target);
            pen = __dadd_rn(pen, __dmul_rn(d, d));
        }
        ei = si;
        er = __dadd_rn(sd, __dmul_rn(p.lambda, pen));
    }
    if (lane == 0) {
        p.e_int[a] = ei;
        p.e_real[a] = er;
    }
}

// argmin_a E_a, lowest a on ties; then the winner's configuration.  One CTA.
__global__ void __launch_bounds__(kThreads) argmin_kernel(const double *e, int R, int *best) {
    __shared__ double sv[kThreads];
    __shared__ int si[kThreads];
    double bv = 0.0;
    int bi = -1;
    for (int a = threadIdx.x; a < R; a += kThreads) {
        const double v = e[a];
        if (bi < 0 || v < bv) {  // ascending a within a thread: strict < keeps the lowest index
            bv = v;
            bi = a;
        }
    }
    sv[threadIdx.x] = bv;
    si[threadIdx.x] = bi;
    __syncthreads();
    for (int s = kThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            const int oi = si[threadIdx.x + s];
            const double ov = sv[threadIdx.x + s];
            const int mi = si[threadIdx.x];
            if (oi >= 0 && (mi < 0 || ov < sv[threadIdx.x] || (ov == sv[threadIdx.x] && oi < mi))) {
                sv[threadIdx.x] = ov;
                si[threadIdx.x] = oi;
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) best[0] = si[0];
}

__global__ void __launch_bounds__(kThreads) best_config_kernel(const int8_t *cfg, int *best, int n, int Rb,
                                                               int64_t cstride) {
    const int i = blockIdx.x * kThreads + threadIdx.x;
    if (i < n) best[1 + i] = cfg[cfg_off(best[0], i, Rb, cstride)];
}

// cfg in logical layout [count][n] int32 <-> device int8 [n][Rb]
__global__ void __launch_bounds__(kThreads) cfg_in_kernel(const int *src, int8_t *dst, int n, int R, int Rb,
                                                          int64_t cstride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= (int64_t)n * R) return;
    const int a = (int)(idx / n), i = (int)(idx - (int64_t)a * n);
    dst[cfg_off(a, i, Rb, cstride)] = (int8_t)src[idx];
}

__global__ void __launch_bounds__(kThreads) cfg_out_kernel(const int8_t *src, int *dst, int n, int R, int Rb,
                                                           int64_t cstride) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= (int64_t)n * R) return;
    const int a = (int)(idx / n), i = (int)(idx - (int64_t)a * n);
    dst[idx] = src[cfg_off(a, i, Rb, cstride)];
}

static void run_energy(Handle *hd, int R, int Rb, double lambda) {
    const DevProblem &dp = hd->dp;
    const int64_t units = dp.kind == FEM_MAXSAT ? dp.m : dp.n;
    const int nblocks = (int)std::max<int64_t>(1, std::min<int64_t>(kEnergyChunks / 8, ceil_div(units, 8 * 16)));
    ReadoutParams p;
    p.dp = dp;
    p.cfg = hd->cfg;
    p.R = R;
    p.Rb = Rb;
    p.cstride = (int64_t)dp.n * Rb;
    p.nchunks = nblocks * 8;
    p.part_i = hd->e_part_i;
    p.part_d = hd->e_part_d;
    p.part_cnt = hd->part_part;
    dim3 grid((unsigned)nblocks, (unsigned)ceil_div(R, 32));
    if (dp.kind == FEM_MAXSAT)
        energy_sat_kernel<<<grid, kThreads, 0, hd->stream>>>(p);
    else if (dp.kind == FEM_ISING && dp.J && dp.n >= 256 && R >= 64) {
        // scratch: the J*m buffer of the dense step and the gather array the next step overwrites (both n x R doubles)
        double *S = hd->gW[hd->cur ^ 1], *F = reinterpret_cast<double *>(hd->field);
        const int64_t tot = (int64_t)dp.n * R;
        spins_f64_kernel<<<(unsigned)ceil_div(tot, kThreads), kThreads, 0, hd->stream>>>(hd->cfg, S, dp.n, R, Rb, p.cstride);
        launch_dense_field_f64(hd, S, F, dp.n, R);
        energy_dense_reduce_kernel<<<grid, kThreads, 0, hd->stream>>>(S, F, dp.n, R, p.nchunks, p.part_i, p.part_d);
        hd->launches += 2;
    } else if (dp.kind == FEM_ISING && dp.J)
        energy_dense_kernel<<<grid, kThreads, 0, hd->stream>>>(p);
    else if (dp.kind == FEM_ISING)
        energy_graph_kernel<FEM_ISING><<<grid, kThreads, 0, hd->stream>>>(p);
    else if (dp.kind == FEM_BMINCUT)
        energy_graph_kernel<FEM_BMINCUT><<<grid, kThreads, 0, hd->stream>>>(p);
    else
        energy_graph_kernel<FEM_MAXCUT><<<grid, kThreads, 0, hd->stream>>>(p);
    FinalizeParams f;
    f.kind = dp.kind;
    f.n = dp.n;
    f.q = dp.q;
    f.R = R;
    f.nchunks = p.nchunks;
    f.integral = hd->integral_weights ? 1 : 0;
    f.lambda = lambda;
    f.vtotal = dp.vw ? dp.vtotal : (double)dp.n;
    f.part_i = hd->e_part_i;
    f.part_d = hd->e_part_d;
    f.part_cnt = hd->part_part;
    f.e_int = hd->e_int;
    f.e_real = hd->e_real;
    f.part = hd->part;
    energy_finalize_kernel<<<(unsigned)ceil_div(R, kThreads / 32), kThreads, 0, hd->stream>>>(f);
    hd->launches += 2;
}

void launch_readout(Handle *hd, double lambda) {
    const DevProblem &dp = hd->dp;
    const int64_t total = (int64_t)dp.n * hd->R;
    const unsigned rgrid = (unsigned)ceil_div(total, kThreads);
    if (hd->wide_live)
        round_kernel<double><<<rgrid, kThreads, 0, hd->stream>>>(hd->hW, hd->cfg, dp.n, dp.F, hd->R, hd->Rb,
                                                                 hd->rows * hd->Rb);
    else
        round_kernel<float><<<rgrid, kThreads, 0, hd->stream>>>(hd->fields(), hd->cfg, dp.n, dp.F, hd->R, hd->Rb,
                                                                hd->rows * hd->Rb);
    hd->launches++;
    run_energy(hd, hd->R, hd->Rb, lambda);
    argmin_kernel<<<1, kThreads, 0, hd->stream>>>(hd->e_real, hd->R, hd->best);
    best_config_kernel<<<(unsigned)ceil_div(dp.n, kThreads), kThreads, 0, hd->stream>>>(hd->cfg, hd->best, dp.n, hd->Rb,
                                                                                       (int64_t)dp.n * hd->Rb);
    hd->launches += 2;
}

void launch_energy_of(Handle *hd, int count, double lambda) { run_energy(hd, count, count, lambda); }

void launch_cfg_in(Handle *hd, const int *cfg_logical_dev, int count) {
    const int64_t total = (int64_t)hd->dp.n * count;
    cfg_in_kernel<<<(unsigned)ceil_div(total, kThreads), kThreads, 0, hd->stream>>>(cfg_logical_dev, hd->cfg, hd->dp.n,
                                                                                   count, count,
                                                                                   (int64_t)hd->dp.n * count);
    hd->launches++;
}

void launch_cfg_out(Handle *hd, int *cfg_logical_dev) {
    const int64_t total = (int64_t)hd->dp.n * hd->R;
    cfg_out_kernel<<<(unsigned)ceil_div(total, kThreads), kThreads, 0, hd->stream>>>(
        hd->cfg, cfg_logical_dev, hd->dp.n, hd->R, hd->Rb, (int64_t)hd->dp.n * hd->Rb);
    hd->launches++;
}

}  // namespace fem
