// Potts (balanced minimum cut) step, "a lane owns a replica": fp32, exact gradient, q <= 8, every degree <= 16,
// replica blocks of Rb = 8, 16 or 32 -- BASELINE.json configs[2] (q = 8, 10-regular, n = 100,000, R = 64).
//
// Why (profiles/r01_cfg2_step.md): the team kernels spread the q states of a variable over lanes, so
// every sum over states (two softmax normalisers, two maxima, the mean <g^p>_P of S20) is a butterfly of shuffles
// and every lane repeats the scalar work of its 4 fields: 634 warp instructions per 128 fields, issue-bound at 0.47
// of the HBM roof.  Here lane (g, r) of a warp owns ALL q states of replica r of variable i0 + g (G = 32 / Rb
// consecutive variables per warp iteration): the sums over states are register adds (no shuffles), the scalar work
// is done once per field, and the whole iteration is ~2.2 warp instructions per field.
//
// Memory side.  The HBM layout is unchanged (row of a variable = [state][replica], q * Rb floats), so a lane's q
// values sit Rb floats apart; they are read from SHARED memory, where the (3 + deg) rows each variable needs -- its
// h, m1, m2 rows and its neighbours' rows of D = P - 1/q -- are staged by 16-byte asynchronous copies (cp.async,
// LDGSTS: no registers held while the bytes are in flight) into a per-warp slot, ONE ITERATION AHEAD: a warp drains
// its slot into registers (neighbour sum + own rows: 4 q values), refills it at once for its next iteration, and only
// then runs softmax / chain rule / optimiser, which covers the fetch.  Rows of different variables are padded apart
// so that the 32 lanes of a shared-memory read hit 32 different banks.  Column indices (and weights) of the next
// iteration are read one iteration ahead and parked in the slot's tail.
//
// The arithmetic is potts_team_kernel's, operation for operation: the same device functions, the same CSR-order
// neighbour sum, and the sums over states are taken in the butterfly's tree order (a butterfly over the states gives
// every lane ((z0+z1)+(z2+z3))+((z4+z5)+(z6+z7)) up to commutativity, which is exact), so the two kernels are
// bit-identical (tests/test_gpu_parity.py::test_potts_lane_bit_identical_to_team_kernel) and results do not depend on
// the replica blocking.  Rows a1-a4 of DESIGN.md section 2: softmax, S26 coupling + balance terms
// (PAPER.md:636), chain rule S20, optimiser update.
#include <algorithm>

#include "device_math.cuh"

namespace fem {

struct PottsLaneParams {
    float *h, *m1, *m2;   // block base pointers (blockIdx.y walks replica blocks)
    const float *g_in;
    float *g_out;
    int64_t blk_stride;
    const int *col;
    const float *w;       // nullptr = unit weights
    const int *row_ptr;
    Sc<float> sc;
    const long long *S_in;
    long long *S_out, *S_zero;
    double fx_scale, fx_inv;
    int n;
    int deg;              // uniform degree, or 0: rows from row_ptr
    int max_deg;          // neighbour layers of the slot (1..16)
    int iters;            // warp iterations: ceil(n / G)
    int warp_floats;      // floats of shared memory per warp (slot + parked indices)
};

constexpr int kLaneMaxDeg = 16;
constexpr int kLaneMaxWarps = 16;

__device__ __forceinline__ void cp_async16(float *dst_smem, const float *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// shared-memory geometry of one warp (host and device agree through these)
template <int Q, int RB>
struct LaneShape {
    static constexpr int G = 32 / RB;        // variables per warp iteration
    static constexpr int ROW = Q * RB;       // floats of one variable's row
    static constexpr int CH = ROW / 4;       // 16-byte chunks of a row
    // rows of the G variables of a layer sit PITCH floats apart, PITCH = RB (mod 32): lane (g, r) reading element
    // s * RB + r of its row then hits bank (g * RB + r + s * RB) % 32 -- 32 different banks across the warp
    static constexpr int PITCH = G == 1 ? ROW : ROW + ((RB - ROW % 32) % 32 + 32) % 32;
    static constexpr int NJ = (G * CH + 31) / 32;  // 16-byte copies per lane and layer
    static constexpr int QPAD = Q <= 2 ? 2 : (Q <= 4 ? 4 : 8);
    static int warp_floats(int max_deg) { return (3 + max_deg) * G * PITCH + 64 + 64 + 4; }
};

// sum / maximum over the states in the butterfly's order (see the header); slots s >= Q hold the neutral element
template <int QPAD>
__device__ __forceinline__ float tree_sum(float (&t)[QPAD]) {
#pragma unroll
    for (int k = 1; k < QPAD; k <<= 1)
#pragma unroll
        for (int s = 0; s < QPAD; s += 2 * k) t[s] = t[s] + t[s + k];
    return t[0];
}
template <int QPAD>
__device__ __forceinline__ float tree_max(float (&t)[QPAD]) {
#pragma unroll
    for (int k = 1; k < QPAD; k <<= 1)
#pragma unroll
        for (int s = 0; s < QPAD; s += 2 * k) t[s] = fmax(t[s], t[s + k]);
    return t[0];
}

template <int Q, int RB, bool UNITW>
__global__ void __launch_bounds__(kLaneMaxWarps * 32, 1) potts_lane_kernel(const __grid_constant__ PottsLaneParams p) {
    using L = LaneShape<Q, RB>;
    constexpr int G = L::G, ROW = L::ROW, CH = L::CH, PITCH = L::PITCH, NJ = L::NJ, QPAD = L::QPAD;
    extern __shared__ __align__(16) float smem[];
    __shared__ unsigned long long cta_sum[ROW];
    pdl_trigger();
    const int n = p.n, MD = p.max_deg;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const int g = lane / RB, r = lane - g * RB;
    const int64_t blk = (int64_t)blockIdx.y * p.blk_stride;
    const Sc<float> &sc = p.sc;
    const float inv_q = 1.0f / (float)Q;
    const float fx_scale_t = (float)p.fx_scale;
    const int warps_total = gridDim.x * nwarps;
    const int warp_gid = blockIdx.x * nwarps + wib;

    float *slot = smem + (size_t)wib * p.warp_floats;
    int *cols_s = reinterpret_cast<int *>(slot + (3 + MD) * G * PITCH);  // [G][MD] column indices of the slot's variables
    float *w_s = reinterpret_cast<float *>(cols_s + 64);                 // [G][MD] their weights
    int *deg_s = reinterpret_cast<int *>(w_s + 64);                      // [G] their degrees

    // ---- lane constants of the copy mapping: chunk c = j * 32 + lane of a layer -> variable gj, 16-byte piece
    int cp_g[NJ], cp_dst[NJ], cp_src[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int c = j * 32 + lane;
        const int gg = c / CH, within = c - gg * CH;
        cp_g[j] = c < G * CH ? gg : -1;
        cp_dst[j] = gg * PITCH + within * 4;
        cp_src[j] = within * 4;
    }
    // ---- lane constants of the index loader: flat entries f = lane and lane + 32 of the [G][MD] tables
    int ld_g[2], ld_k[2];
#pragma unroll
    for (int x = 0; x < 2; ++x) {
        const int f = lane + 32 * x;
        ld_g[x] = f < G * MD ? f / MD : -1;
        ld_k[x] = f - (f / MD) * MD;
    }

    // CSR entries of iteration `it` (static problem structure: legal before pdl_wait)
    int m_col[2], m_deg[2];
    float m_w[2];
    auto load_meta = [&](int it) {
#pragma unroll
        for (int x = 0; x < 2; ++x) {
            m_col[x] = 0;
            m_deg[x] = 0;
            m_w[x] = 0.0f;
            const int i = it * G + ld_g[x];
            if (ld_g[x] >= 0 && it < p.iters && i < n) {
                int e0, d;
                if (p.deg > 0) {
                    e0 = i * p.deg;
                    d = p.deg;
                } else {
                    e0 = __ldg(p.row_ptr + i);
                    d = __ldg(p.row_ptr + i + 1) - e0;
                }
                m_deg[x] = d;
                if (ld_k[x] < d) {
                    m_col[x] = __ldg(p.col + e0 + ld_k[x]);
                    if (!UNITW) m_w[x] = __ldg(p.w + e0 + ld_k[x]);
                }
            }
        }
    };
    auto store_meta = [&]() {
#pragma unroll
        for (int x = 0; x < 2; ++x)
            if (ld_g[x] >= 0) {
                const int f = lane + 32 * x;
                cols_s[f] = m_col[x];
                if (!UNITW) w_s[f] = m_w[x];
                if (ld_k[x] == 0) deg_s[ld_g[x]] = m_deg[x];
            }
    };
    // asynchronous copies of iteration `it` into the slot: layers 0..2 = own rows of h, m1, m2, layer 3 + k = k-th neighbour
    const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();
    auto issue = [&](int it) {
        const int i0 = it * G;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            if (cp_g[j] < 0) continue;
            const int i = i0 + cp_g[j];
            if (i < n) {
                const int64_t own = blk + (int64_t)i * ROW + cp_src[j];
                cp_async16(slot + cp_dst[j], p.h + own);
                if (use_m1) cp_async16(slot + G * PITCH + cp_dst[j], p.m1 + own);
                if (use_m2) cp_async16(slot + 2 * G * PITCH + cp_dst[j], p.m2 + own);
            }
            const int d = deg_s[cp_g[j]];
            const int *cj = cols_s + cp_g[j] * MD;
            const float *src0 = p.g_in + blk + cp_src[j];
            float *dst = slot + 3 * G * PITCH + cp_dst[j];
#pragma unroll 2
            for (int k = 0; k < d; ++k) cp_async16(dst + k * (G * PITCH), src0 + (unsigned long long)(unsigned)cj[k] * (unsigned)(ROW));
        }
        cp_async_commit();
    };

    if (threadIdx.x < ROW) cta_sum[threadIdx.x] = 0ull;
    int it = warp_gid;
    load_meta(it);
    store_meta();
    __syncwarp();
    load_meta(it + warps_total);
    __syncthreads();
    pdl_wait();  // everything below reads or overwrites what the previous launch wrote

    float Ss[Q];
    {
        const long long *Sp = p.S_in + (int64_t)blockIdx.y * ROW + r;
#pragma unroll
        for (int s = 0; s < Q; ++s) Ss[s] = (float)((double)Sp[s * RB] * p.fx_inv);
    }
    if (blockIdx.x == 0)
        for (int k = threadIdx.x; k < ROW; k += blockDim.x) p.S_zero[(int64_t)blockIdx.y * ROW + k] = 0ll;

    long long colacc[Q];
#pragma unroll
    for (int s = 0; s < Q; ++s) colacc[s] = 0ll;

    if (it < p.iters) issue(it);

    for (; it < p.iters; it += warps_total) {
        const int i = it * G + g;
        const bool ok = i < n;
        cp_async_wait_all();
        __syncwarp();  // every lane's copies have landed
        // ---- drain the slot: coupling contraction f(s) = sum_j W_ij D_j(s) in CSR order, and the own rows
        float f[Q], h[Q], m1[Q], m2[Q];
#pragma unroll
        for (int s = 0; s < Q; ++s) f[s] = 0.0f;
        {
            const int mydeg = deg_s[g];
            const float *nb = slot + (3 * G + g) * PITCH + r;
            const float *wk = w_s + g * MD;
#pragma unroll 2
            for (int k = 0; k < mydeg; ++k, nb += G * PITCH) {
                if (UNITW) {
#pragma unroll
                    for (int s = 0; s < Q; ++s) f[s] += nb[s * RB];  // == fma(1, D_j, f)
                } else {
                    const float ww = wk[k];
#pragma unroll
                    for (int s = 0; s < Q; ++s) f[s] = fma(ww, nb[s * RB], f[s]);
                }
            }
            const float *own = slot + g * PITCH + r;
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                h[s] = own[s * RB];
                m1[s] = use_m1 ? own[G * PITCH + s * RB] : 0.0f;
                m2[s] = use_m2 ? own[2 * G * PITCH + s * RB] : 0.0f;
            }
        }
        __syncwarp();  // the slot is in registers: refill it with the warp's next iteration while this one is computed
        const int itn = it + warps_total;
        if (itn < p.iters) {
            store_meta();  // indices of iteration itn (read one iteration ago)
            __syncwarp();
            issue(itn);
            load_meta(itn + warps_total);
        }
        // ---- softmax of h(t) over the states
        float P[Q];
        {
            float t[QPAD];
#pragma unroll
            for (int s = 0; s < QPAD; ++s) t[s] = s < Q ? h[s] : -3.0e38f;
            const float mx = tree_max<QPAD>(t);
            float e[Q];
#pragma unroll
            for (int s = 0; s < Q; ++s) e[s] = fexp(h[s] - mx);
#pragma unroll
            for (int s = 0; s < QPAD; ++s) t[s] = s < Q ? e[s] : 0.0f;
            const float rz = frcp(tree_sum<QPAD>(t));
#pragma unroll
            for (int s = 0; s < Q; ++s) P[s] = e[s] * rz;
        }
        // ---- g^p (S26), g^h = P (g^p - <g^p>_P) (S20), optimiser
        {
            float gp[Q], t[QPAD];
#pragma unroll
            for (int s = 0; s < Q; ++s) gp[s] = fma(h[s], sc.inv_beta, fma(sc.two_lambda, Ss[s] - P[s], -f[s]));
#pragma unroll
            for (int s = 0; s < QPAD; ++s) t[s] = s < Q ? __fmul_rn(P[s], gp[s]) : 0.0f;  // (never contracted into the adds)
            const float gbar = tree_sum<QPAD>(t);
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                const float gh = sc.gamma * (P[s] * (gp[s] - gbar));
                h[s] = opt_update(h[s], gh, m1[s], m2[s], sc);
            }
        }
        const int64_t off = blk + (int64_t)(ok ? i : 0) * ROW + r;
        if (ok) {
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                __stcs(p.h + off + s * RB, h[s]);
                if (use_m1) __stcs(p.m1 + off + s * RB, m1[s]);
                if (use_m2) __stcs(p.m2 + off + s * RB, m2[s]);
            }
        }
        // ---- centred marginals of the new fields -> g_out, and their column sums (exact fixed point)
        {
            float t[QPAD], e[Q];
#pragma unroll
            for (int s = 0; s < QPAD; ++s) t[s] = s < Q ? h[s] : -3.0e38f;
            const float mx = tree_max<QPAD>(t);
#pragma unroll
            for (int s = 0; s < Q; ++s) e[s] = fexp(h[s] - mx);
#pragma unroll
            for (int s = 0; s < QPAD; ++s) t[s] = s < Q ? e[s] : 0.0f;
            const float rz = frcp(tree_sum<QPAD>(t));
            if (ok) {
#pragma unroll
                for (int s = 0; s < Q; ++s) {
                    const float po = fma(e[s], rz, -inv_q);
                    colacc[s] += __float2ll_rn(po * fx_scale_t);
                    p.g_out[off + s * RB] = po;
                }
            }
        }
    }

    // column sums: exact integer adds -- variable groups of the warp (shuffles) -> CTA (shared atomics) -> grid (global atomics)
#pragma unroll
    for (int s = 0; s < Q; ++s) {
#pragma unroll
        for (int o = RB; o < 32; o <<= 1) colacc[s] += __shfl_xor_sync(0xffffffffu, colacc[s], o);
    }
    if (g == 0) {
#pragma unroll
        for (int s = 0; s < Q; ++s)
            if (colacc[s] != 0ll) atomicAdd(&cta_sum[s * RB + r], (unsigned long long)colacc[s]);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < ROW; k += blockDim.x) {
        const unsigned long long v = cta_sum[k];
        if (v != 0ull) atomicAdd(reinterpret_cast<unsigned long long *>(p.S_out) + (int64_t)blockIdx.y * ROW + k, v);
    }
}

// ---- host side ----
bool potts_lane_applicable(const Handle *hd) {
    const int q = hd->dp.q, Rb = hd->Rb, deg = hd->dp.max_deg;
    if (hd->opt_potts_lane == 0 || hd->gather_disc) return false;
    if (q < 2 || q > 8 || (Rb != 8 && Rb != 16 && Rb != 32)) return false;
    return deg >= 1 && deg <= kLaneMaxDeg && hd->dp.nnz < ((int64_t)1 << 31);
}

template <int Q, int RB, bool UNITW>
static cudaError_t launch_lane_one(Handle *hd, PottsLaneParams &p, int blk_count) {
    using L = LaneShape<Q, RB>;
    p.warp_floats = L::warp_floats(p.max_deg);
    p.iters = (int)ceil_div(p.n, L::G);
    int smem_max = 0, dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return cudaErrorUnknown;
    smem_max -= (int)(L::ROW * sizeof(unsigned long long)) + 1024;  // static cta_sum + reserve
    const int nwarps = std::min<int64_t>(kLaneMaxWarps, smem_max / (p.warp_floats * (int)sizeof(float)));
    if (nwarps < 4) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)nwarps * p.warp_floats * sizeof(float);
    const void *fn = reinterpret_cast<const void *>(&potts_lane_kernel<Q, RB, UNITW>);
    if (!hd->attr_done.count(fn)) {
        cudaError_t e = cudaFuncSetAttribute(potts_lane_kernel<Q, RB, UNITW>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
        if (e != cudaSuccess) return e;
        hd->attr_done.insert(fn);
    }
    const unsigned gx = (unsigned)std::min<int64_t>(hd->sm_count, ceil_div(p.iters, nwarps));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(gx, (unsigned)blk_count);
    cfg.blockDim = dim3(nwarps * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = hd->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, potts_lane_kernel<Q, RB, UNITW>, p);
}

template <int Q>
static cudaError_t launch_lane_q(Handle *hd, PottsLaneParams &p, int blk_count) {
    const bool unit = p.w == nullptr;
    switch (hd->Rb) {
        case 8: return unit ? launch_lane_one<Q, 8, true>(hd, p, blk_count) : launch_lane_one<Q, 8, false>(hd, p, blk_count);
        case 16: return unit ? launch_lane_one<Q, 16, true>(hd, p, blk_count) : launch_lane_one<Q, 16, false>(hd, p, blk_count);
        default: return unit ? launch_lane_one<Q, 32, true>(hd, p, blk_count) : launch_lane_one<Q, 32, false>(hd, p, blk_count);
    }
}

// One fp32 exact-gradient Potts step of replica blocks [blk_begin, blk_begin + blk_count); false = not applicable.
bool launch_potts_lane(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count) {
    if (!potts_lane_applicable(hd)) return false;
    const int Rb = hd->Rb, q = hd->dp.q;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    PottsLaneParams p;
    p.h = hd->h + base;
    p.m1 = hd->m1 + base;
    p.m2 = hd->m2 + base;
    p.g_in = hd->g[hd->cur] + base;
    p.g_out = hd->g[hd->cur ^ 1] + base;
    p.blk_stride = hd->rows * Rb;
    p.col = hd->dp.col;
    p.w = hd->dp.w;
    p.row_ptr = hd->dp.row_ptr;
    p.sc = Sc<float>(sc);
    const int64_t so = (int64_t)blk_begin * q * Rb;
    const int t = sc.t;  // column-sum buffers rotate with the step number exactly as in launch_potts_typed
    p.S_in = hd->colsum[t % 3] + so;
    p.S_out = hd->colsum[(t + 1) % 3] + so;
    p.S_zero = hd->colsum[(t + 2) % 3] + so;
    p.fx_scale = hd->colsum_scale;
    p.fx_inv = 1.0 / hd->colsum_scale;
    p.n = hd->dp.n;
    p.deg = hd->dp.uniform_deg;
    p.max_deg = hd->dp.max_deg;
    cudaError_t e;
    switch (q) {
        case 2: e = launch_lane_q<2>(hd, p, blk_count); break;
        case 3: e = launch_lane_q<3>(hd, p, blk_count); break;
        case 4: e = launch_lane_q<4>(hd, p, blk_count); break;
        case 5: e = launch_lane_q<5>(hd, p, blk_count); break;
        case 6: e = launch_lane_q<6>(hd, p, blk_count); break;
        case 7: e = launch_lane_q<7>(hd, p, blk_count); break;
        default: e = launch_lane_q<8>(hd, p, blk_count); break;
    }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    hd->launches++;
    hd->lane_launches++;
    return true;
}

}  // namespace fem
