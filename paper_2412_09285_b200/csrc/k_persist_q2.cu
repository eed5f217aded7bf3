// Replica-persistent annealing kernel for SMALL two-state problems (MaxCut / sparse Ising / Max-SAT with clauses of at
// most 5 literals; at most 4096 variables per CTA of the cluster).
//
// The stepwise kernel (k_step_q2.cu) is launch- and latency-bound when n*R is a few tens of thousands of
// fields (BASELINE.json configs[0]: n = 800, R = 32: one launch per annealing step, 11 us each, 1% of HBM).
// Replicas are independent, so here ONE CLUSTER of CS CTAs owns ONE replica for a whole
// run of annealing steps: CTA c of the cluster owns the variables [c*chunk, (c+1)*chunk); their h, m1, m2 live in
// registers; every CTA keeps the replica's whole gathered vector m = tanh(h/2) double-buffered in its own shared
// memory and, after each step, stores its new m values into all CS copies through distributed shared memory;
// the only synchronisation per annealing step is one cluster barrier (__syncthreads() when CS = 1).  The CTA's
// rows of the CSR are staged once in shared memory as a sliced ELL (slot-major inside each warp: lane l of a
// warp reads index/weight slot j at [j*32 + l], conflict-free; 16-bit column indices).  HBM is touched at entry
// (load state) and exit (store state), so the per-step launch, DRAM and L2 round trips disappear; the binding
// resource is the shared-memory gather rate of the SMs a replica is spread over.
//
// Arithmetic is the stepwise kernel's, instruction for instruction (same device functions, same CSR-order sum),
// so the result is bit-identical to the stepwise path (tests/test_gpu_parity.py::test_persistent_bit_identical).
// Rows a1-a4 of DESIGN.md section 2: S30 coupling sum, S29 entropy gradient and
// chain rule, Adam; the per-step scalars 1/beta_t and the two bias corrections come from the
// host (double) in the kernel parameters, kChunk steps per launch.
#include <cooperative_groups.h>

#include "device_math.cuh"

namespace fem {

template <typename T>
struct PersistChunk {
    static constexpr int kSteps = sizeof(T) == 4 ? 256 : 96;  // 3 * kSteps * sizeof(T) <= 3 KB of kernel parameters
};

template <typename T>
struct PersistParams {
    T *h, *m1, *m2;      // state arrays (device layout, all replica blocks)
    const T *g_in;       // gather buffer holding m of the current fields
    T *g_out;            // gather buffer that must hold m of the final fields
    const int *row_ptr;
    const int *col;
    const float *w;      // nullptr = unit weights
    int n, Rb;
    int64_t blk_stride;
    int nsteps;
    int chunk;           // variables per CTA of the cluster (multiple of 32)
    int ell_cap;         // sliced-ELL entries reserved per CTA
    const double *rowsum;  // sum_j |W_ij| per node (manipulated gradients)
    const signed char *g8_in;  // manipulated gradients: sgn(m) as bytes in the gather arrays (device_math.cuh)
    signed char *g8_out;
    T eps, b1, b2, omb1, omb2, wd, gamma;
    int opt, disc;
    int kst;             // Max-SAT: ints per occurrence in `col` (k_max - 1 rounded up to a power of two)
    int first_step;      // index in this chunk of the anneal's step 0 (SGD momentum buffer starts there), or -1
    T inv_beta[PersistChunk<T>::kSteps];
    T step_size[PersistChunk<T>::kSteps];
    T rsqrt_bc2[PersistChunk<T>::kSteps];
};

constexpr int kPersistUnroll = 8;     // ELL rows are padded to a multiple of this: warp-uniform, remainder-free gather loops
constexpr int kPersistMaxUnits = 128;  // (items per thread) x (warps per CTA) <= 4 x 32

// IPT variables per thread: variable i = c*chunk + k*blockDim.x + threadIdx.x.  ISING: dU/dp = -2 sum_j J_ij m_j.
// SATK > 0: Max-SAT -- `row_ptr` / `col` are the variable -> occurrence table (fem_internal.cuh), SATK = k_max - 1 packed
// entries (var << 1 | negated) per occurrence, own sign in bit 31 of entry 0; the ELL keeps SATK 16-bit arrays and a sign
// byte per slot; slot n of the gathered vector is the constant 1 that pads short clauses.
template <typename T, int IPT, bool ISING, bool WEIGHTED, int SATK>
__global__ void __launch_bounds__(1024, 1) persist_q2_kernel(const __grid_constant__ PersistParams<T> p) {
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int unit_off[kPersistMaxUnits + 1];
    const int n = p.n;
    const int gn = n + 1;                                                  // slot n of each buffer stays 0: the ELL padding points at it
    T *gbuf = reinterpret_cast<T *>(smem_raw);                             // [2][n + 1]
    float *ws = reinterpret_cast<float *>(gbuf + 2 * (size_t)gn);         // [ell_cap] when WEIGHTED
    unsigned short *cs = reinterpret_cast<unsigned short *>(WEIGHTED ? (ws + p.ell_cap) : ws);  // [ell_cap] ([SATK][ell_cap])
    unsigned char *sgn = reinterpret_cast<unsigned char *>(cs + (size_t)(SATK > 0 ? SATK : 1) * p.ell_cap);  // SAT: [ell_cap]

    cg::cluster_group cluster = cg::this_cluster();
    const unsigned CS = cluster.num_blocks();
    const unsigned c = cluster.block_rank();
    const int r = blockIdx.x / CS;  // replica
    const int64_t base = (int64_t)(r / p.Rb) * p.blk_stride + (r % p.Rb);
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;
    const int v_begin = c * p.chunk, v_end = min(n, v_begin + p.chunk);

    // ---- state into registers, the whole gathered vector into this CTA's shared memory ----
    T h[IPT], m1[IPT], m2[IPT];
    int e0[IPT], deg[IPT], off[IPT], pdeg[IPT];  // pdeg: the unit's longest row rounded up to kPersistUnroll (warp-uniform)
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = v_begin + k * nt + tid;
        const bool ok = i < v_end;
        const int64_t o = base + (int64_t)(ok ? i : 0) * p.Rb;
        h[k] = ok ? p.h[o] : (T)0;
        m1[k] = ok ? p.m1[o] : (T)0;
        m2[k] = ok ? p.m2[o] : (T)0;
        e0[k] = ok ? p.row_ptr[i] : 0;
        deg[k] = ok ? p.row_ptr[i + 1] - e0[k] : 0;
        int mx = deg[k];
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, s));
        pdeg[k] = (mx + kPersistUnroll - 1) / kPersistUnroll * kPersistUnroll;
        if (lane == 0) unit_off[k * nwarps + warp + 1] = pdeg[k] * 32;
    }
    for (int i = tid; i < n; i += nt)
        gbuf[i] = p.disc ? (T)(int)p.g8_in[base + (int64_t)i * p.Rb] : p.g_in[base + (int64_t)i * p.Rb];
    if (tid == 0) {
        unit_off[0] = 0;
        gbuf[n] = SATK > 0 ? (T)1 : (T)0;
        gbuf[gn + n] = SATK > 0 ? (T)1 : (T)0;
    }
    __syncthreads();
    if (tid == 0)
        for (int u = 1; u <= IPT * nwarps; ++u) unit_off[u] += unit_off[u - 1];
    __syncthreads();
    // ---- this CTA's CSR rows as a sliced ELL: slot j of lane l of unit (k, warp) at unit_off + j*32 + l ----
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        off[k] = unit_off[k * nwarps + warp] + lane;
        for (int j = 0; j < pdeg[k]; ++j) {  // rows shorter than the unit are padded with (column n, weight 0): adds +0
            const bool real = j < deg[k];
            if (SATK > 0) {
                // padding occurrence: first factor 0.5 - 0.5 * 1 = 0, the others 1: contributes +-0
#pragma unroll
                for (int x = 0; x < (SATK > 0 ? SATK : 1); ++x) {
                    const unsigned pk = real ? (unsigned)p.col[(int64_t)(e0[k] + j) * p.kst + x] : (((unsigned)n << 1) | (x == 0 ? 0u : 1u));
                    cs[(size_t)x * p.ell_cap + off[k] + j * 32] = (unsigned short)(pk & 0xffffu);
                    if (x == 0) sgn[off[k] + j * 32] = (unsigned char)(pk >> 31);
                }
                continue;
            }
            cs[off[k] + j * 32] = real ? (unsigned short)p.col[e0[k] + j] : (unsigned short)n;
            if (WEIGHTED) ws[off[k] + j * 32] = real ? p.w[e0[k] + j] : 0.0f;
        }
    }
    if (CS > 1) cluster.sync();  // every CTA of the cluster is running before anyone stores into its shared memory
    else __syncthreads();

    Sc<T> sc;
    sc.eps = p.eps; sc.b1 = p.b1; sc.b2 = p.b2; sc.omb1 = p.omb1; sc.omb2 = p.omb2; sc.wd = p.wd;
    sc.two_lambda = (T)0;
    sc.gamma = p.gamma; sc.opt = p.opt; sc.disc = p.disc; sc.first = 0;
    // manipulated gradients: c_i = 1 / sum_j |W_ij| (Ising: |2 J_ij|), static, so it lives in a register
    T ci[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        ci[k] = (T)1;
        const int i = v_begin + k * nt + tid;
        if (p.disc && i < v_end) {
            const double rs = p.rowsum[i] * (ISING ? 2.0 : 1.0);
            ci[k] = rs > 0.0 ? (T)(1.0 / rs) : (T)0;
        }
    }
    int cur = 0;
    for (int t = 0; t < p.nsteps; ++t) {
        const T *__restrict__ gi = gbuf + (size_t)cur * gn;
        T *go = gbuf + (size_t)(cur ^ 1) * gn;
        sc.inv_beta = p.inv_beta[t];
        sc.step_size = p.step_size[t];
        sc.rsqrt_bc2 = p.rsqrt_bc2[t];
        sc.first = t == p.first_step;
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const int i = v_begin + k * nt + tid;
            if (i < v_end) {
                T dU = (T)0;
                const unsigned short *__restrict__ cp = cs + off[k];
                if (SATK > 0) {
                    // dU/dp_i = sum_{m ni i} s_mi prod_{k != i} u_mk (S28), occurrences in table order
                    const unsigned char *__restrict__ sp = sgn + off[k];
#pragma unroll 4
                    for (int j = 0; j < pdeg[k]; ++j) {
                        T prod = (T)1;
#pragma unroll
                        for (int x = 0; x < (SATK > 0 ? SATK : 1); ++x) {
                            const unsigned e = cp[(size_t)x * p.ell_cap + j * 32];
                            const T sg = (e & 1u) ? (T)0.5 : (T)-0.5;
                            prod *= fma(sg, gi[e >> 1], (T)0.5);
                        }
                        dU += sp[j * 32] ? -prod : prod;
                    }
                } else if (WEIGHTED) {
                    const float *__restrict__ wp = ws + off[k];
#pragma unroll kPersistUnroll
                    for (int j = 0; j < pdeg[k]; ++j) dU = fma((T)wp[j * 32], gi[cp[j * 32]], dU);
                } else {
#pragma unroll kPersistUnroll
                    for (int j = 0; j < pdeg[k]; ++j) dU += gi[cp[j * 32]];  // == fma(1, m_j, dU) of the stepwise kernel
                }
                if (ISING) dU = (T)-2 * dU;
                const T g = q2_grad(dU, ci[k], h[k], sc);
                h[k] = opt_update(h[k], g, m1[k], m2[k], sc);
                const T mg = sc.disc ? sign_of(h[k]) : mag_of(h[k]);
                if (CS > 1) {
                    for (unsigned pr = 0; pr < CS; ++pr) cluster.map_shared_rank(go, pr)[i] = mg;
                } else {
                    go[i] = mg;
                }
            }
        }
        // one barrier per step is enough with two buffers: step t+1 overwrites the buffer step t READ, and no
        // CTA starts step t+1 before all have finished step t
        if (CS > 1) cluster.sync();
        else __syncthreads();
        cur ^= 1;
    }

#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = v_begin + k * nt + tid;
        if (i < v_end) {
            const int64_t o = base + (int64_t)i * p.Rb;
            p.h[o] = h[k];
            p.m1[o] = m1[k];
            p.m2[o] = m2[k];
            if (p.disc) p.g8_out[o] = (signed char)(int)gbuf[(size_t)cur * gn + i];
            else p.g_out[o] = gbuf[(size_t)cur * gn + i];
        }
    }
}

// ---- host side ----
static constexpr size_t kSmemCap = 227 * 1024 - 1024;  // dynamic shared memory a CTA may ask for (static part reserved)
static const int kClusterSizes[4] = {1, 2, 4, 8};

struct PersistGeom {
    int chunk, ipt, threads;
};

// Variable -> (CTA, item, thread) mapping for a cluster of cs CTAs; shared by the ELL sizing below and the launch.
static bool persist_geometry(int n, int cs, PersistGeom *g) {
    g->chunk = (int)(ceil_div(ceil_div(n, cs), 32) * 32);
    if (g->chunk > 4096) return false;
    g->ipt = g->chunk <= 1024 ? 1 : (g->chunk <= 2048 ? 2 : 4);
    g->threads = (int)(ceil_div(ceil_div(g->chunk, g->ipt), 32) * 32);
    return true;
}

// Called by fem_create with the host CSR: sliced-ELL entries per CTA (max over the CTAs of a cluster) for each
// cluster size; -1 where the mapping does not apply.
void persist_prepare(Handle *hd, const int64_t *row_ptr) {
    const int n = hd->dp.n;
    for (int a = 0; a < 4; ++a) {
        hd->persist_ell[a] = -1;
        PersistGeom g;
        if (n > 65535 || !persist_geometry(n, kClusterSizes[a], &g)) continue;
        int64_t worst = 0;
        for (int c = 0; c < kClusterSizes[a]; ++c) {
            int64_t entries = 0;
            const int v_begin = c * g.chunk, v_end = std::min(n, v_begin + g.chunk);
            for (int k = 0; k < g.ipt; ++k)
                for (int w0 = 0; w0 < g.threads; w0 += 32) {
                    int64_t mx = 0;
                    for (int l = 0; l < 32; ++l) {
                        const int i = v_begin + k * g.threads + w0 + l;
                        if (i < v_end) mx = std::max<int64_t>(mx, row_ptr[i + 1] - row_ptr[i]);
                    }
                    entries += 32 * ((mx + kPersistUnroll - 1) / kPersistUnroll * kPersistUnroll);
                }
            worst = std::max(worst, entries);
        }
        hd->persist_ell[a] = worst;
    }
}

static size_t persist_smem_bytes(const Handle *hd, int a, size_t elt) {
    const size_t per_slot = hd->dp.kind == FEM_MAXSAT ? 2 * (size_t)hd->dp.kstride + 1 : (hd->dp.w ? 6 : 2);
    return 2 * ((size_t)hd->dp.n + 1) * elt + (size_t)hd->persist_ell[a] * per_slot + 16;
}

// Cluster size index for R replicas: spread a replica over as many SMs as the device has to spare (R * CS <= SMs),
// at least 64 variables per CTA, and the CTA's ELL + two copies of the gathered vector (fp64) must fit.
static int persist_choose(const Handle *hd, int R) {
    if (hd->opt_persistent == 0) return -1;
    const bool graph = hd->dp.kind == FEM_MAXCUT || (hd->dp.kind == FEM_ISING && !hd->dp.J);
    // Max-SAT: clause length <= 5 (one kernel per k_max - 1 = 1..4), packed entries (var << 1 | negated) in 16 bits
    const bool sat = hd->dp.kind == FEM_MAXSAT && !hd->dp.lit_state && hd->dp.kstride >= 1 && hd->dp.kstride <= 4 && hd->dp.n <= 32767;
    if (!graph && !sat) return -1;
    if (graph && hd->dp.n_long > 0 && hd->opt_long_rows) return -1;  // long rows: the stepwise kernel splits them over a CTA (k_step_q2.cu)
    int best = -1;
    for (int a = 0; a < 4; ++a) {
        if (hd->persist_ell[a] < 0 || persist_smem_bytes(hd, a, sizeof(double)) > kSmemCap) continue;
        if (hd->opt_persistent > 1) {  // forced cluster size (tests, experiments)
            if (kClusterSizes[a] == hd->opt_persistent - 1) return a;
            continue;
        }
        if (best < 0) best = a;  // the smallest size that fits
        const int sms = kClusterSizes[a] == 1 ? hd->sm_count : hd->sm_count - hd->sm_count % (2 * kClusterSizes[a]);
        if ((int64_t)R * kClusterSizes[a] <= sms && ceil_div(hd->dp.n, kClusterSizes[a]) >= 64) best = a;
    }
    // one CTA (cluster) per replica runs in waves over the SMs: beyond ~3 waves the stepwise kernel, which spreads every
    // step over the whole device, is faster (Max-SAT n = 300, m = 2600: R = 148 -> 2.0 vs 7.1 ms per 500-step anneal,
    // R = 400 -> 6.0 vs 7.8, R = 800 -> 11.8 vs 10.3)
    if (best >= 0 && (int64_t)R * kClusterSizes[best] > 3 * (int64_t)hd->sm_count) return -1;
    return best;
}

bool persist_eligible(const Handle *hd) { return persist_choose(hd, std::max(hd->R, 1)) >= 0; }

template <typename T, int IPT>
static cudaError_t persist_launch_ipt(Handle *hd, const PersistParams<T> &p, int cs, int threads, size_t smem) {
    auto launch = [&](auto kernel) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(hd->R * cs));
        cfg.blockDim = dim3((unsigned)threads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = hd->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)cs;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kernel, p);
    };
    const bool ising = hd->dp.kind == FEM_ISING, weighted = hd->dp.w != nullptr;
    if (hd->dp.kind == FEM_MAXSAT) {
        switch (hd->dp.kstride) {
            case 1: return launch(persist_q2_kernel<T, IPT, false, false, 1>);
            case 2: return launch(persist_q2_kernel<T, IPT, false, false, 2>);
            case 3: return launch(persist_q2_kernel<T, IPT, false, false, 3>);
            default: return launch(persist_q2_kernel<T, IPT, false, false, 4>);
        }
    }
    if (ising) return weighted ? launch(persist_q2_kernel<T, IPT, true, true, 0>) : launch(persist_q2_kernel<T, IPT, true, false, 0>);
    return weighted ? launch(persist_q2_kernel<T, IPT, false, true, 0>) : launch(persist_q2_kernel<T, IPT, false, false, 0>);
}

// Runs steps [t_begin, t_end) of the schedule for all replicas; `scalars(t)` gives the per-step scalars.
template <typename T, typename F>
static cudaError_t persist_run_t(Handle *hd, int t_begin, int t_end, F &&scalars) {
    using S = StateOf<T>;
    const int a = persist_choose(hd, hd->R);
    if (a < 0) return cudaErrorInvalidConfiguration;
    const int cs = kClusterSizes[a];
    PersistGeom g;
    persist_geometry(hd->dp.n, cs, &g);
    const size_t smem = persist_smem_bytes(hd, a, sizeof(T));
    for (int ta = t_begin; ta < t_end; ta += PersistChunk<T>::kSteps) {
        const int tb = std::min(t_end, ta + PersistChunk<T>::kSteps);
        PersistParams<T> p;
        p.h = S::h(hd);
        p.m1 = S::m1(hd);
        p.m2 = S::m2(hd);
        p.g_in = S::g(hd, hd->cur);
        const int cur_after = hd->cur ^ ((tb - ta) & 1);
        p.g_out = S::g(hd, cur_after);
        const bool sat = hd->dp.kind == FEM_MAXSAT;
        p.row_ptr = sat ? hd->dp.occ_ptr : hd->dp.row_ptr;
        p.col = sat ? hd->dp.occ : hd->dp.col;
        p.w = sat ? nullptr : hd->dp.w;
        p.kst = 1;
        while (p.kst < hd->dp.kstride) p.kst <<= 1;
        p.n = hd->dp.n;
        p.Rb = hd->Rb;
        p.blk_stride = hd->rows * hd->Rb;
        p.nsteps = tb - ta;
        p.chunk = g.chunk;
        p.ell_cap = (int)hd->persist_ell[a];
        p.rowsum = hd->rowsum;
        p.g8_in = reinterpret_cast<const signed char *>(hd->g[hd->cur]);
        p.g8_out = reinterpret_cast<signed char *>(hd->g[cur_after]);
        p.first_step = -1;
        for (int t = ta; t < tb; ++t) {
            const StepScalars s = scalars(t);
            if (t == ta) {
                const Sc<T> c(s);
                p.eps = c.eps; p.b1 = c.b1; p.b2 = c.b2; p.omb1 = c.omb1; p.omb2 = c.omb2; p.wd = c.wd;
                p.gamma = c.gamma; p.opt = c.opt; p.disc = c.disc;
            }
            if (s.first) p.first_step = t - ta;
            p.inv_beta[t - ta] = (T)s.inv_beta;
            p.step_size[t - ta] = (T)s.step_size;
            p.rsqrt_bc2[t - ta] = (T)s.rsqrt_bc2;
        }
        cudaError_t e;
        if (g.ipt == 1) e = persist_launch_ipt<T, 1>(hd, p, cs, g.threads, smem);
        else if (g.ipt == 2) e = persist_launch_ipt<T, 2>(hd, p, cs, g.threads, smem);
        else e = persist_launch_ipt<T, 4>(hd, p, cs, g.threads, smem);
        if (e != cudaSuccess) return e;
        hd->cur = cur_after;
        hd->launches++;
        hd->persist_launches++;
        hd->persist_cluster = cs;
    }
    return cudaSuccess;
}

cudaError_t persist_run(Handle *hd, bool wide, int t_begin, int t_end, StepScalars (*scalars)(void *, int), void *ctx) {
    auto f = [&](int t) { return scalars(ctx, t); };
    if (wide) return persist_run_t<double>(hd, t_begin, t_end, f);
    return persist_run_t<float>(hd, t_begin, t_end, f);
}

}  // namespace fem
