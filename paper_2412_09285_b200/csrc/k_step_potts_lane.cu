// Potts (balanced minimum cut) step, "a lane owns a replica": fp32, exact gradient, q <= 8, every degree <= 16,
// replica blocks of Rb = 8, 16 or 32 -- BASELINE.json configs[2] (q = 8, 10-regular, n = 100,000, R = 64).
//
// Why (profiles/r01_cfg2_step.md): the team kernels spread the q states of a variable over lanes, so
// every sum over states (two softmax normalisers, two maxima, the mean <g^p>_P of S20) is a butterfly of shuffles
// and every lane repeats the scalar work of its 4 fields: 634 warp instructions per 128 fields, issue-bound at 0.47
// of the HBM roof.  Here the ARITHMETIC runs with lane (g, r) of a warp owning ALL q states of replica r of variable
// i0 + g (G = 32 / Rb consecutive variables per warp iteration): the sums over states are register adds (no
// shuffles) and the scalar work is done once per field.
//
// Memory side.  The HBM layout is unchanged (row of a variable = [state][replica], q * Rb floats), so GLOBAL memory is
// accessed in the "row mapping": a lane holds 4 consecutive floats of a row, every load / store is a 16-byte vector and
// a warp instruction covers 512 contiguous bytes per row pair -- the own rows h, m1, m2 (read at the top of the
// iteration, consumed after the gather), the neighbours' rows of D = P - 1/q (summed in CSR order in this mapping,
// kGather rows in flight per lane) and the four output rows.  The two mappings meet in a small per-warp tile of SHARED
// memory (4 arrays x G rows): the row mapping writes it with 16-byte stores, the lane mapping reads it with 4-byte
// loads (rows PITCH = Rb (mod 32) floats apart: 32 different banks), and back for the outputs.  A first version that
// staged all (3 + deg) rows of an iteration in shared memory by cp.async was slower (111 us against 96 us for the
// TMA-staged team kernel on cfg 2): ptxas pads every LDGSTS with three dummy shared loads on sm_100a and the
// run-time loops over the degree cost as many instructions as the arithmetic (profiles/r02_cfg2_step.md).
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
    int max_deg;          // longest row (1..16)
    int iters;            // warp iterations: ceil(n / G)
    int warp_floats;      // floats of shared memory per warp
};

constexpr int kLaneMaxDeg = 16;
constexpr int kLaneMaxWarps = 8;   // warps per CTA (every warp works on its own)

__device__ __forceinline__ void cp_async16(float *dst_smem, const float *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// geometry of one warp iteration (host and device agree through these)
template <int Q, int RB>
struct LaneShape {
    static constexpr int G = 32 / RB;        // variables per warp iteration
    static constexpr int ROW = Q * RB;       // floats of one variable's row
    static constexpr int CH = ROW / 4;       // 16-byte pieces of a row
    // rows of the G variables sit PITCH floats apart in the shared tiles, PITCH = RB (mod 32): lane (g, r) reading
    // element s * RB + r of its row hits bank (g * RB + r + s * RB) % 32 -- 32 different banks across the warp
    static constexpr int PITCH = G == 1 ? ROW : ROW + ((RB - ROW % 32) % 32 + 32) % 32;
    static constexpr int NJ = (G * CH + 31) / 32;  // 16-byte pieces per lane in the row mapping
    static constexpr bool FULL = (G * CH) % 32 == 0;  // every lane holds a piece in every pass
    static constexpr int QPAD = Q <= 2 ? 2 : (Q <= 4 ? 4 : 8);
    static constexpr int TILE = G * PITCH;   // floats of one array's tile
    static constexpr int LAYER = NJ * 32 * 4;  // floats of one neighbour layer of the gather slot (piece c at c * 4)
    // 4 tiles, column indices, weights, degrees, then the gather slot: max_deg layers
    static int warp_floats(int max_deg) { return 4 * TILE + 64 + 64 + 4 + max_deg * LAYER; }
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

// DEG > 0: every row of the CSR has exactly DEG entries (regular graphs): the loops over the neighbours are unrolled
// and carry no predicates.  DEG = 0: rows of any length up to max_deg <= 16.
template <int Q, int RB, bool UNITW, int DEG>
__global__ void __launch_bounds__(kLaneMaxWarps * 32, 2) potts_lane_kernel(const __grid_constant__ PottsLaneParams p) {
    using L = LaneShape<Q, RB>;
    constexpr int G = L::G, ROW = L::ROW, CH = L::CH, PITCH = L::PITCH, NJ = L::NJ, QPAD = L::QPAD, TILE = L::TILE, LAYER = L::LAYER;
    extern __shared__ __align__(16) float smem[];
    __shared__ unsigned long long cta_sum[ROW];
    pdl_trigger();
    const int n = p.n;
    const int MD = DEG > 0 ? DEG : p.max_deg;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const int g = lane / RB, r = lane - g * RB;
    const int64_t blk = (int64_t)blockIdx.y * p.blk_stride;
    const Sc<float> &sc = p.sc;
    const float inv_q = 1.0f / (float)Q;
    const float fx_scale_t = (float)p.fx_scale;
    const int warps_total = gridDim.x * nwarps;
    const int warp_gid = blockIdx.x * nwarps + wib;
    const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();

    float *tile = smem + (size_t)wib * p.warp_floats;            // [4][G][PITCH]
    int *cols_s = reinterpret_cast<int *>(tile + 4 * TILE);      // [G][MD] column indices of the iteration's variables
    float *w_s = reinterpret_cast<float *>(cols_s + 64);         // [G][MD] their weights
    int *deg_s = reinterpret_cast<int *>(w_s + 64);              // [G] their degrees
    float *slot = reinterpret_cast<float *>(deg_s + 4);          // [MD][LAYER] neighbour rows, row mapping

    // ---- row mapping: piece c = j * 32 + lane -> variable rm_g[j], floats rm_off[j] .. +3 of its row
    int rm_g[NJ], rm_off[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int c = j * 32 + lane;
        const int gg = c / CH;
        rm_g[j] = (L::FULL || c < G * CH) ? gg : -1;
        rm_off[j] = (c - gg * CH) * 4;
    }
    // ---- index loader: flat entries f = lane and lane + 32 of the [G][MD] tables
    int ld_g[2], ld_k[2];
#pragma unroll
    for (int x = 0; x < 2; ++x) {
        const int f = lane + 32 * x;
        ld_g[x] = f < G * MD ? f / MD : -1;
        ld_k[x] = f - (f / MD) * MD;
    }
    int m_col[2], m_deg[2];
    float m_w[2];
    auto load_meta = [&](int it) {  // CSR entries of iteration `it` (static problem structure: legal before pdl_wait)
#pragma unroll
        for (int x = 0; x < 2; ++x) {
            m_col[x] = 0;
            m_deg[x] = 0;
            m_w[x] = 0.0f;
            const int i = it * G + ld_g[x];
            if (ld_g[x] >= 0 && it < p.iters && i < n) {
                int e0, d;
                if (DEG > 0) {
                    e0 = i * DEG;
                    d = DEG;
                } else if (p.deg > 0) {
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
                if (DEG == 0 && ld_k[x] == 0) deg_s[ld_g[x]] = m_deg[x];
            }
    };
    // asynchronous 16-byte copies of the neighbours' rows of the iteration whose indices are parked in cols_s:
    // layer k of the slot = k-th neighbour of every variable, pieces in row-mapping order (conflict-free to read back)
    const float *gsrc = p.g_in + blk;
    auto issue_gathers = [&]() {
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            if (rm_g[j] < 0) continue;
            const int *cj = cols_s + rm_g[j] * MD;
            const float *src0 = gsrc + rm_off[j];
            float *dst = slot + (j * 32 + lane) * 4;
            if (DEG > 0) {
#pragma unroll
                for (int k = 0; k < DEG; ++k)
                    cp_async16(dst + k * LAYER, src0 + (unsigned long long)(unsigned)cj[k] * (unsigned)ROW);
            } else {
                const int d = deg_s[rm_g[j]];
#pragma unroll 2
                for (int k = 0; k < d; ++k)
                    cp_async16(dst + k * LAYER, src0 + (unsigned long long)(unsigned)cj[k] * (unsigned)ROW);
            }
        }
        cp_async_commit();
    };

    if (threadIdx.x < ROW) cta_sum[threadIdx.x] = 0ull;
    int it = warp_gid;
    load_meta(it);
    store_meta();
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

    if (it < p.iters) issue_gathers();

    for (; it < p.iters; it += warps_total) {
        const int i0 = it * G;
        // ---- own rows in the row mapping (consumed after the neighbour sum)
        float4 own[3][NJ];
        int64_t roff[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const bool act = rm_g[j] >= 0 && i0 + rm_g[j] < n;
            roff[j] = act ? blk + (int64_t)(i0 + rm_g[j]) * ROW + rm_off[j] : -1;
            own[0][j] = own[1][j] = own[2][j] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (act) {
                own[0][j] = __ldcs(reinterpret_cast<const float4 *>(p.h + roff[j]));
                if (use_m1) own[1][j] = __ldcs(reinterpret_cast<const float4 *>(p.m1 + roff[j]));
                if (use_m2) own[2][j] = __ldcs(reinterpret_cast<const float4 *>(p.m2 + roff[j]));
            }
        }
        // ---- coupling contraction f(s) = sum_j W_ij D_j(s) in CSR order, row mapping, out of the gather slot
        cp_async_wait_all();
        __syncwarp();
        float4 facc[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            facc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (rm_g[j] < 0) continue;
            const float4 *src = reinterpret_cast<const float4 *>(slot + (j * 32 + lane) * 4);
            const float *wj = w_s + rm_g[j] * MD;
            auto add = [&](int k) {
                const float4 nb = src[k * (LAYER / 4)];
                if (UNITW) {  // == fma(1, D_j, f)
                    facc[j].x += nb.x; facc[j].y += nb.y; facc[j].z += nb.z; facc[j].w += nb.w;
                } else {
                    const float ww = wj[k];
                    facc[j].x = fma(ww, nb.x, facc[j].x); facc[j].y = fma(ww, nb.y, facc[j].y);
                    facc[j].z = fma(ww, nb.z, facc[j].z); facc[j].w = fma(ww, nb.w, facc[j].w);
                }
            };
            if (DEG > 0) {
#pragma unroll
                for (int k = 0; k < DEG; ++k) add(k);
            } else {
                const int d = deg_s[rm_g[j]];
#pragma unroll 2
                for (int k = 0; k < d; ++k) add(k);
            }
        }
        __syncwarp();
        // the slot and the index tables are free: park the next iteration's indices (read one iteration ago), start its
        // gathers -- they land while this iteration is computed -- and fetch the indices of the one after
        if (it + warps_total < p.iters) {
            store_meta();
            __syncwarp();
            issue_gathers();
            load_meta(it + 2 * warps_total);
        }
        // ---- row mapping -> shared tile -> lane mapping
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (rm_g[j] >= 0) {
                float *d = tile + rm_g[j] * PITCH + rm_off[j];
                *reinterpret_cast<float4 *>(d) = facc[j];
                *reinterpret_cast<float4 *>(d + TILE) = own[0][j];
                *reinterpret_cast<float4 *>(d + 2 * TILE) = own[1][j];
                *reinterpret_cast<float4 *>(d + 3 * TILE) = own[2][j];
            }
        __syncwarp();
        float f[Q], h[Q], m1[Q], m2[Q];
        {
            const float *src = tile + g * PITCH + r;
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                f[s] = src[s * RB];
                h[s] = src[TILE + s * RB];
                m1[s] = src[2 * TILE + s * RB];
                m2[s] = src[3 * TILE + s * RB];
            }
        }
        __syncwarp();
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
        // ---- centred marginals of the new fields and their column sums (exact fixed point)
        const bool ok = i0 + g < n;
        float po[Q];
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
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                po[s] = fma(e[s], rz, -inv_q);
                if (ok) colacc[s] += __float2ll_rn(po[s] * fx_scale_t);
            }
        }
        // ---- lane mapping -> shared tile -> row mapping -> 16-byte stores
        {
            float *dst = tile + g * PITCH + r;
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                dst[s * RB] = h[s];
                dst[TILE + s * RB] = m1[s];
                dst[2 * TILE + s * RB] = m2[s];
                dst[3 * TILE + s * RB] = po[s];
            }
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (roff[j] >= 0) {
                const float *src = tile + rm_g[j] * PITCH + rm_off[j];
                __stcs(reinterpret_cast<float4 *>(p.h + roff[j]), *reinterpret_cast<const float4 *>(src));
                if (use_m1) __stcs(reinterpret_cast<float4 *>(p.m1 + roff[j]), *reinterpret_cast<const float4 *>(src + TILE));
                if (use_m2) __stcs(reinterpret_cast<float4 *>(p.m2 + roff[j]), *reinterpret_cast<const float4 *>(src + 2 * TILE));
                *reinterpret_cast<float4 *>(p.g_out + roff[j]) = *reinterpret_cast<const float4 *>(src + 3 * TILE);
            }
        __syncwarp();
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
    if (hd->dp.vw) return false;  // node-weighted balance term: register path / state-innermost kernel only
    if (hd->opt_potts_lane == 0 || hd->gather_disc) return false;
    if (q < 2 || q > 8 || (Rb != 8 && Rb != 16 && Rb != 32)) return false;
    return deg >= 1 && deg <= kLaneMaxDeg && hd->dp.nnz < ((int64_t)1 << 31);
}

template <int Q, int RB, bool UNITW, int DEG>
static cudaError_t launch_lane_deg(Handle *hd, PottsLaneParams &p, int blk_count) {
    using L = LaneShape<Q, RB>;
    p.warp_floats = L::warp_floats(p.max_deg);
    p.iters = (int)ceil_div(p.n, L::G);
    auto kernel = potts_lane_kernel<Q, RB, UNITW, DEG>;
    const void *fn = reinterpret_cast<const void *>(kernel);
    int smem_sm = 0, dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev) != cudaSuccess) return cudaErrorUnknown;
    // two CTAs per SM (the kernel is compiled for 128 registers): as many warps per CTA as half the SM's shared memory holds
    const int per_cta = smem_sm / 2 - 1024 - (int)(L::ROW * sizeof(unsigned long long)) - 512;
    const int nwarps = (int)std::min<int64_t>(kLaneMaxWarps, per_cta / (p.warp_floats * (int)sizeof(float)));
    if (nwarps < 2) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)nwarps * p.warp_floats * sizeof(float);
    if (!hd->attr_done.count(fn)) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, per_cta);
        if (e != cudaSuccess) return e;
        hd->attr_done.insert(fn);
    }
    int &resident = hd->resident_ctas[{fn, smem}];
    if (resident == 0) {
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, nwarps * 32, smem) != cudaSuccess || occ < 1) occ = 1;
        resident = occ * hd->sm_count;
    }
    const unsigned gx = (unsigned)std::min<int64_t>(resident, ceil_div(p.iters, nwarps));
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
    return cudaLaunchKernelEx(&cfg, kernel, p);
}

// regular graphs of the common degrees get the unrolled, predicate-free instantiation
template <int Q, int RB, bool UNITW>
static cudaError_t launch_lane_one(Handle *hd, PottsLaneParams &p, int blk_count) {
    switch (p.deg) {
        case 3: return launch_lane_deg<Q, RB, UNITW, 3>(hd, p, blk_count);
        case 4: return launch_lane_deg<Q, RB, UNITW, 4>(hd, p, blk_count);
        case 6: return launch_lane_deg<Q, RB, UNITW, 6>(hd, p, blk_count);
        case 10: return launch_lane_deg<Q, RB, UNITW, 10>(hd, p, blk_count);
        default: return launch_lane_deg<Q, RB, UNITW, 0>(hd, p, blk_count);
    }
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
