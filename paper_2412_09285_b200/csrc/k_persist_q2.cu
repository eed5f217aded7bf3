// Replica-persistent annealing kernel for SMALL two-state problems (MaxCut / sparse Ising / Max-SAT with clauses of at
// most 5 literals; at most 4096 variables per CTA of the cluster).
//
// The stepwise kernel (k_step_q2.cu) is launch- and latency-bound when n*R is a few tens of thousands of
// fields (BASELINE.json configs[0]: n = 800, R = 32: one launch per annealing step, 11 us each, 1% of HBM).
// Replicas are independent, so here ONE CLUSTER of CS CTAs owns ONE replica for a whole
// run of annealing steps: the warps of the cluster take the variables in turn along the degree-sorted processing order;
// their h, m1, m2 live in registers; every CTA keeps the replica's whole gathered vector m = tanh(h/2) double-buffered in
// its own shared memory, in slot order (what a CTA produces is one contiguous run), and after each step pushes its run
// into the peers' copies with one bulk copy per peer through distributed shared memory, completing on the peer's
// mbarrier: no cluster barrier and no per-lane remote store inside the step (__syncthreads() only when CS = 1).  The CTA's
// rows of the CSR are staged once per launch in shared memory as a sliced ELL of 16-bit slot columns (eight per lane and
// 16-byte load), or kept in registers (fp32 steps, unit weights, rows of at most 72 entries).  HBM is touched at entry
// (load state) and exit (store state), so the per-step launch, DRAM and L2 round trips disappear; what binds is the
// latency of the shared-memory gathers and of the exchange.
//
// Arithmetic is the stepwise kernel's, instruction for instruction (same device functions, same CSR-order sum),
// so the result is bit-identical to the stepwise path (tests/test_gpu_parity.py::test_persistent_bit_identical).
// Rows a1-a4 of DESIGN.md section 2: S30 coupling sum, S29 entropy gradient and
// chain rule, Adam; the per-step scalars 1/beta_t and the two bias corrections come from the
// host (double) in the kernel parameters, PersistChunk<T>::kSteps steps per launch.
#include <cooperative_groups.h>

#include "device_math.cuh"

namespace fem {

template <typename T>
struct PersistChunk {
    static constexpr int kSteps = sizeof(T) == 4 ? 2048 : 1024;  // 3 * kSteps * sizeof(T) = 24 KB of the 32 KB of kernel parameters
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
    const int *order;    // processing order of the variables (degree-sorted, fem_api.cu) or nullptr = identity
    const int *rank;     // inverse of `order` (position of each variable) or nullptr = identity
    int gn;              // slots per buffer of the gathered vector (persist_gn)
    int first_step;      // index in this chunk of the anneal's step 0 (SGD momentum buffer starts there), or -1
    T inv_beta[PersistChunk<T>::kSteps];
    T step_size[PersistChunk<T>::kSteps];
    T rsqrt_bc2[PersistChunk<T>::kSteps];
};

constexpr int kPersistUnroll = 8;     // ELL rows are padded to a multiple of this: warp-uniform, remainder-free gather loops
constexpr int kPersistRegGroups = 9;   // register-resident columns: the longest row they hold, in groups of 8 entries (72)
constexpr int kPersistMaxUnits = 128;  // (items per thread) x (warps per CTA) <= 4 x 32

// ---- mbarrier / bulk-copy primitives of the cluster exchange ----
__device__ __forceinline__ unsigned ps_smem(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned ps_mapa(unsigned addr, unsigned cta) {  // the same offset in the shared memory of CTA `cta`
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
__device__ __forceinline__ void ps_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nPS_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra PS_DONE_%=;\nbra PS_WAIT_%=;\nPS_DONE_%=:\n}" ::"r"(ps_smem(bar)), "r"(parity) : "memory");
}

// IPT variables per thread.  Unit u = k * (warps per CTA) + warp of CTA c takes the 32 positions starting at (u*CS + c)*32
// of the processing order (warps dealt out to the CTAs of the cluster in turn: with a degree-sorted order every CTA gets the
// same mix of short and long rows, and the rows of a warp have nearly the same length, so the padding of the sliced ELL is
// small).  The gathered vector is kept in SLOT order: the variable of thread tid, item k of CTA c sits at c*cw + k*nt + tid
// (cw = IPT * nt), so that what a CTA produces in a step is one contiguous run, and the ELL columns are slots.
//
// Exchange between the CTAs of a cluster, once per annealing step: every thread stores its new m into its own CTA's copy;
// after a CTA-wide barrier CS - 1 threads each push the CTA's run into one peer with a bulk copy through distributed shared
// memory (cp.async.bulk.shared::cluster.shared::cta) that completes, in bytes, on the PEER's mbarrier of that buffer; a CTA
// starts the next step when its own mbarrier has seen the CS - 1 runs.  No cluster barrier and no per-lane remote stores
// (measured at cfg 0, CS = 4: 0.32 - 0.66 us of a 1.7 us step went to the 4-byte remote stores, 0.18 to the cluster barrier).
// Two buffers are enough: a peer pushes its step-t run into the buffer I read in step t-1 only after it has received my
// step-(t-1) run, which I send after my last read of that buffer.
//
// ISING: dU/dp = -2 sum_j J_ij m_j.
// SATK > 0: Max-SAT -- `row_ptr` / `col` are the variable -> occurrence table (fem_internal.cuh), SATK = k_max - 1 packed
// entries (var << 1 | negated) per occurrence, own sign in bit 31 of entry 0; the ELL keeps SATK 16-bit arrays
// (slot << 1 | negated) and a sign byte per ELL entry (entry-major: entry j of lane l at [j*32 + l]); the last slot of the
// gathered vector is the constant 1 that pads short clauses.  Graph modes: eight 16-bit columns per lane and 16-byte load
// (entries 8g .. 8g+7 of lane l at [g*256 + l*8 ..]), the last slot is the constant 0.
// RG > 0 (graph modes, IPT = 1, rows of at most 8 * RG entries): the thread keeps its row's columns in registers (RG * 4
// packed words, padded with the constant slot) and the gather loop is unrolled in full: no column loads in the step and all
// gathers of a row in flight at once.
template <typename T, int IPT, bool ISING, bool WEIGHTED, int SATK, int RG>
__global__ void __launch_bounds__(RG > 0 ? 512 : 1024, 1) persist_q2_kernel(const __grid_constant__ PersistParams<T> p) {
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int unit_off[kPersistMaxUnits + 1];
    __shared__ __align__(8) unsigned long long bar[2];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned CS = cluster.num_blocks();
    const unsigned c = cluster.block_rank();
    const int n = p.n;
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;
    const int cw = IPT * nt;          // slots per CTA
    const int pad = (int)CS * cw;     // the constant slot the ELL padding points at
    const int gn = p.gn;              // slots per buffer, >= pad + 1, a multiple of 4 (16-byte alignment of what follows)
    T *gbuf = reinterpret_cast<T *>(smem_raw);                             // [2][gn]
    float *ws = reinterpret_cast<float *>(gbuf + 2 * (size_t)gn);         // [ell_cap] when WEIGHTED
    unsigned short *cs = reinterpret_cast<unsigned short *>(WEIGHTED ? (ws + p.ell_cap) : ws);  // [ell_cap] ([SATK][ell_cap])
    unsigned char *sgn = reinterpret_cast<unsigned char *>(cs + (size_t)(SATK > 0 ? SATK : 1) * p.ell_cap);  // SAT: [ell_cap]
    const int r = blockIdx.x / CS;  // replica
    const int64_t base = (int64_t)(r / p.Rb) * p.blk_stride + (r % p.Rb);
    auto slot_of = [&](int j) -> int {
        const int pos = p.rank ? p.rank[j] : j;
        const int gw = pos >> 5;
        return (gw % (int)CS) * cw + (gw / (int)CS) * 32 + (pos & 31);
    };

    // ---- state into registers, the whole gathered vector into this CTA's shared memory ----
    T h[IPT], m1[IPT], m2[IPT];
    int vi[IPT];                                 // the variable, -1 = none
    int e0[IPT], deg[IPT], off[IPT], pdeg[IPT];  // pdeg: the unit's longest row rounded up to kPersistUnroll (warp-uniform)
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int pos = ((k * nwarps + warp) * (int)CS + (int)c) * 32 + lane;
        const bool ok = pos < n;
        const int i = ok ? (p.order ? p.order[pos] : pos) : 0;
        vi[k] = ok ? i : -1;
        const int64_t o = base + (int64_t)i * p.Rb;
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
    for (int x = tid; x < 2 * gn; x += nt) gbuf[x] = (T)0;  // (slots of no variable travel with the runs: keep them defined)
    if (tid == 0) {
        unit_off[0] = 0;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ps_smem(&bar[0])));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ps_smem(&bar[1])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    for (int i = tid; i < n; i += nt)
        gbuf[slot_of(i)] = p.disc ? (T)(int)p.g8_in[base + (int64_t)i * p.Rb] : p.g_in[base + (int64_t)i * p.Rb];
    if (tid < 2) gbuf[tid * gn + pad] = SATK > 0 ? (T)1 : (T)0;
    if (tid == 0)
        for (int u = 1; u <= IPT * nwarps; ++u) unit_off[u] += unit_off[u - 1];
    __syncthreads();
    // ---- this CTA's CSR rows as a sliced ELL ----
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        off[k] = unit_off[k * nwarps + warp] + (SATK > 0 ? lane : lane * kPersistUnroll);
        for (int j = 0; j < pdeg[k]; ++j) {  // rows shorter than the unit are padded with (pad slot, weight 0): adds +0
            const bool real = j < deg[k];
            if (SATK > 0) {
                // padding occurrence: first factor 0.5 - 0.5 * 1 = 0, the others 1: contributes +-0
#pragma unroll
                for (int x = 0; x < (SATK > 0 ? SATK : 1); ++x) {
                    const unsigned pk = real ? (unsigned)p.col[(int64_t)(e0[k] + j) * p.kst + x] : (((unsigned)n << 1) | (x == 0 ? 0u : 1u));
                    const unsigned var = (pk & 0x7fffffffu) >> 1;
                    const unsigned sl = var >= (unsigned)n ? (unsigned)pad : (unsigned)slot_of((int)var);  // (short clauses are padded with variable n)
                    cs[(size_t)x * p.ell_cap + off[k] + j * 32] = (unsigned short)((sl << 1) | (pk & 1u));
                    if (x == 0) sgn[off[k] + j * 32] = (unsigned char)(pk >> 31);
                }
                continue;
            }
            cs[off[k] + (j / kPersistUnroll) * (32 * kPersistUnroll) + (j % kPersistUnroll)] = (unsigned short)(real ? slot_of(p.col[e0[k] + j]) : pad);
            if (WEIGHTED) ws[unit_off[k * nwarps + warp] + j * 32 + lane] = real ? p.w[e0[k] + j] : 0.0f;
        }
    }
    if (CS > 1) cluster.sync();  // every CTA of the cluster is running (and its mbarriers exist) before anyone pushes into it
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
        const int i = vi[k];
        if (p.disc && i >= 0) {
            const double rs = p.rowsum[i] * (ISING ? 2.0 : 1.0);
            ci[k] = rs > 0.0 ? (T)(1.0 / rs) : (T)0;
        }
    }
    unsigned creg[RG > 0 ? RG * 4 : 1];
    if (RG > 0) {
        __syncthreads();  // (the staged columns of this thread were written by this thread; the barrier is for tidiness only)
#pragma unroll
        for (int g = 0; g < RG; ++g) {
            uint4 pk = make_uint4(0u, 0u, 0u, 0u);
            if (g * kPersistUnroll < pdeg[0]) pk = *reinterpret_cast<const uint4 *>(cs + off[0] + g * kPersistUnroll * 32);
            else pk.x = pk.y = pk.z = pk.w = (unsigned)pad | ((unsigned)pad << 16);
            creg[g * 4 + 0] = pk.x; creg[g * 4 + 1] = pk.y; creg[g * 4 + 2] = pk.z; creg[g * 4 + 3] = pk.w;
        }
    }
    const unsigned run_bytes = (unsigned)cw * (unsigned)sizeof(T);
    unsigned phase[2] = {0u, 0u};
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
            if (vi[k] >= 0) {
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
                } else if (RG > 0 && !WEIGHTED) {
                    // no branches: every gather of the row is issued before the first add (rows shorter than 8 * RG read the
                    // constant slot, a broadcast)
                    T mv[RG > 0 ? RG * kPersistUnroll : 1];
#pragma unroll
                    for (int x = 0; x < RG * kPersistUnroll; ++x) mv[x] = gi[(creg[x >> 1] >> ((x & 1) * 16)) & 0xffffu];
#pragma unroll
                    for (int x = 0; x < RG * kPersistUnroll; ++x) dU += mv[x];  // (the padding adds +0 at the end: CSR order kept)
                } else {
                    // eight columns per 16-byte load; the sum runs in CSR order (== the stepwise kernel's fma(w, m_j, dU))
                    const float *__restrict__ wp = ws + unit_off[k * nwarps + warp] + lane;
#pragma unroll 2
                    for (int jg = 0; jg < pdeg[k]; jg += kPersistUnroll) {
                        const uint4 pk = *reinterpret_cast<const uint4 *>(cp + jg * 32);
                        const unsigned w4[4] = {pk.x, pk.y, pk.z, pk.w};
                        T mv[kPersistUnroll];
#pragma unroll
                        for (int x = 0; x < kPersistUnroll; ++x) mv[x] = gi[(w4[x >> 1] >> ((x & 1) * 16)) & 0xffffu];
#pragma unroll
                        for (int x = 0; x < kPersistUnroll; ++x) {
                            if (WEIGHTED) dU = fma((T)wp[(jg + x) * 32], mv[x], dU);
                            else dU += mv[x];
                        }
                    }
                }
                if (ISING) dU = (T)-2 * dU;
                const T g = q2_grad(dU, ci[k], h[k], sc);
                h[k] = opt_update(h[k], g, m1[k], m2[k], sc);
                go[(int)c * cw + k * nt + tid] = sc.disc ? sign_of(h[k]) : mag_of(h[k]);
            }
        }
        if (CS > 1) {
            const int b = cur ^ 1;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // my stores, before the bulk copies read them
            __syncthreads();
            if (tid == 0)
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ps_smem(&bar[b])), "r"((CS - 1) * run_bytes) : "memory");
            if (tid < (int)CS && tid != (int)c) {
                const unsigned src = ps_smem(go + (size_t)c * cw);
                asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                 ps_mapa(src, (unsigned)tid)),
                             "r"(src), "r"(run_bytes), "r"(ps_mapa(ps_smem(&bar[b]), (unsigned)tid))
                             : "memory");
            }
            ps_wait(&bar[b], phase[b]);
            phase[b] ^= 1u;
        } else {
            __syncthreads();
        }
        cur ^= 1;
    }
    if (CS > 1) cluster.sync();  // nobody leaves while a peer's last push may still be reading or writing here

#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = vi[k];
        if (i >= 0) {
            const int64_t o = base + (int64_t)i * p.Rb;
            p.h[o] = h[k];
            p.m1[o] = m1[k];
            p.m2[o] = m2[k];
            const T mg = gbuf[(size_t)cur * gn + (int)c * cw + k * nt + tid];
            if (p.disc) p.g8_out[o] = (signed char)(int)mg;
            else p.g_out[o] = mg;
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

// Slots per buffer of the gathered vector: IPT * threads per CTA of the cluster, the constant slot, rounded up to 4.
static int persist_gn(int n, int cs) {
    PersistGeom g;
    if (!persist_geometry(n, cs, &g)) return 0;
    return (cs * g.ipt * g.threads + 1 + 3) & ~3;
}

// Called by fem_create with the host CSR (or occurrence table) and the processing order (nullptr = identity): sliced-ELL
// entries per CTA (max over the CTAs of a cluster) for each cluster size, with the kernel's unit -> position mapping;
// -1 where the mapping does not apply.
void persist_prepare(Handle *hd, const int64_t *row_ptr, const int *order) {
    const int n = hd->dp.n;
    for (int a = 0; a < 4; ++a) {
        hd->persist_ell[a] = -1;
        PersistGeom g;
        const int cs = kClusterSizes[a];
        if (n > 65535 || !persist_geometry(n, cs, &g)) continue;
        const int units = g.ipt * (g.threads / 32);
        int64_t worst = 0;
        for (int c = 0; c < cs; ++c) {
            int64_t entries = 0;
            for (int u = 0; u < units; ++u) {
                int64_t mx = 0;
                for (int l = 0; l < 32; ++l) {
                    const int64_t pos = ((int64_t)u * cs + c) * 32 + l;
                    if (pos >= n) break;
                    const int i = order ? order[pos] : (int)pos;
                    mx = std::max<int64_t>(mx, row_ptr[i + 1] - row_ptr[i]);
                }
                entries += 32 * ((mx + kPersistUnroll - 1) / kPersistUnroll * kPersistUnroll);
            }
            worst = std::max(worst, entries);
        }
        hd->persist_ell[a] = worst;
    }
}

static size_t persist_smem_bytes(const Handle *hd, int a, size_t elt) {
    const bool sat = hd->dp.kind == FEM_MAXSAT;
    const size_t per_slot = sat ? 2 * (size_t)hd->dp.kstride + 1 : (hd->dp.w ? 6 : 2);
    (void)sat;
    return 2 * (size_t)persist_gn(hd->dp.n, kClusterSizes[a]) * elt + (size_t)hd->persist_ell[a] * per_slot + 16;
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
        if (persist_gn(hd->dp.n, kClusterSizes[a]) > (sat ? 32768 : 65536)) continue;  // slots (SAT: slot << 1 | negated) are 16-bit ELL columns
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
            case 1: return launch(persist_q2_kernel<T, IPT, false, false, 1, 0>);
            case 2: return launch(persist_q2_kernel<T, IPT, false, false, 2, 0>);
            case 3: return launch(persist_q2_kernel<T, IPT, false, false, 3, 0>);
            default: return launch(persist_q2_kernel<T, IPT, false, false, 4, 0>);
        }
    }
    if (IPT == 1 && sizeof(T) == 4 && !weighted && hd->dp.max_deg <= kPersistRegGroups * kPersistUnroll && threads <= 512) {
        // columns in registers, fp32 steps of unit-weight graphs: 24, 48 or 72 entries per row
        constexpr bool on = IPT == 1 && sizeof(T) == 4;
        const int groups = (hd->dp.max_deg + kPersistUnroll - 1) / kPersistUnroll;
        if (groups <= 3) return ising ? launch(persist_q2_kernel<T, IPT, true, false, 0, on ? 3 : 0>) : launch(persist_q2_kernel<T, IPT, false, false, 0, on ? 3 : 0>);
        if (groups <= 6) return ising ? launch(persist_q2_kernel<T, IPT, true, false, 0, on ? 6 : 0>) : launch(persist_q2_kernel<T, IPT, false, false, 0, on ? 6 : 0>);
        return ising ? launch(persist_q2_kernel<T, IPT, true, false, 0, on ? 9 : 0>) : launch(persist_q2_kernel<T, IPT, false, false, 0, on ? 9 : 0>);
    }
    if (ising) return weighted ? launch(persist_q2_kernel<T, IPT, true, true, 0, 0>) : launch(persist_q2_kernel<T, IPT, true, false, 0, 0>);
    return weighted ? launch(persist_q2_kernel<T, IPT, false, true, 0, 0>) : launch(persist_q2_kernel<T, IPT, false, false, 0, 0>);
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
    const int per_launch = hd->opt_persist_chunk > 0 ? (int)std::min<int64_t>(hd->opt_persist_chunk, PersistChunk<T>::kSteps) : PersistChunk<T>::kSteps;
    for (int ta = t_begin; ta < t_end; ta += per_launch) {
        const int tb = std::min(t_end, ta + per_launch);
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
        p.order = sat ? nullptr : hd->dp.order;
        p.rank = sat ? nullptr : hd->dp.rank;
        p.gn = persist_gn(hd->dp.n, cs);
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
