// Potts (balanced minimum cut) step with the memory side on the TMA: fp32, exact gradient, every degree <= 16,
// one variable per warp (q * Rb / 4 == 32 lanes, q a power of two) -- BASELINE.json configs[2].
//
// Why: ncu on potts_team_kernel (profiles/r01_cfg2_step.md) shows nothing saturated -- DRAM 49%, issue ~50% -- with
// every warp spending ~5.5 us per variable in four dependent memory round trips (h, column indices, neighbour rows,
// m1/m2), and registers (64 per thread at 4 CTAs per SM) leave no room to keep more loads in flight per warp.  Here the
// rows a variable needs -- its own h, m1, m2 rows and its `deg` neighbour rows of D = P - 1/q, (3 + deg) * 512 B at
// cfg 2 -- are fetched by bulk asynchronous copies (cp.async.bulk, the 1-D TMA path) into a per-warp slot in shared
// memory, completion counted on an mbarrier, ONE VARIABLE AHEAD of the arithmetic: a warp drains its slot into
// registers (the neighbour sum and the three own rows: 16 values), refills it with its next variable at once, and
// only then does the softmax / chain rule / optimiser work, which covers the fetch.  The bytes in flight live in
// shared memory, not in registers: 64 registers per thread, four CTAs (32 warps, 32 slots of 6.5 KB) per SM.
// Measured on cfg 2: 116 us (register path) -> 101 us; a two-stage ring at 2 CTAs per SM gave 117 us
// (too few warps to cover the ALU latency), per-lane cp.async (LDGSTS) staging instead of bulk copies 105 us, L2
// cache hints on the bulk copies (evict-first own rows + evict-last neighbour rows 122 us, evict-first alone 101 us).  The column indices are read two variables ahead (one per lane, handed to the issuing lanes by a shuffle).
//
// The arithmetic is potts_team_kernel's, instruction for instruction (same device functions, same CSR-order sum),
// so the two kernels are bit-identical (tests/test_gpu_parity.py::test_potts_tma_bit_identical).  Rows a1-a4 of
// softmax, S26 coupling + balance terms, chain rule S20
// (PAPER.md:599), optimiser update.
#include <algorithm>
#include <map>

#include "device_math.cuh"

namespace fem {

struct PottsTmaParams {
    float *h, *m1, *m2;   // block base pointers (blockIdx.y walks replica blocks)
    const float *g_in;
    float *g_out;
    int64_t blk_stride;
    const int *col;
    const float *w;       // nullptr = unit weights
    Sc<float> sc;
    const long long *S_in;
    long long *S_out, *S_zero;
    double fx_scale, fx_inv;
    int n, q, Rb;
    int deg;              // uniform degree, or 0: rows from row_ptr, at most max_deg entries each
    int max_deg;          // rows of the slot reserved for neighbours
    const int *row_ptr;
    unsigned row_len;     // q * Rb floats = 128 (one float4 per lane)
    // manipulated gradients (DISC): neighbours enter as state ids, one byte per (variable, replica) (device_math.cuh)
    const signed char *g8_in;
    signed char *g8_out;
    const double *rowsum;
};

constexpr int kTmaWarps = 8;          // warps per CTA
constexpr int kTmaMaxDeg = 16;

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_addr(bar)),
        "r"(parity)
        : "memory");
}
// 1-D bulk copy global -> shared, completion in bytes on an mbarrier (size a multiple of 16, both addresses 16-aligned)
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr(dst)),
                 "l"(src), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}

template <int QPAD, bool UNITW, bool DISC>
__global__ void __launch_bounds__(kTmaWarps * 32, 4) potts_tma_kernel(const __grid_constant__ PottsTmaParams p) {
    constexpr int VEC = 4;
    using R = Row<float, VEC>;
    constexpr int kStages = QPAD == 32 ? 5 : QPAD == 16 ? 4 : QPAD == 8 ? 3 : QPAD == 4 ? 2 : 1;
    constexpr int lps = 32 / QPAD;  // lanes per state; Rb = 4 * lps
    extern __shared__ __align__(128) float ring[];                 // [warp][(3 + deg) rows][128 floats]
    __shared__ __align__(8) uint64_t full_bar[kTmaWarps];
    __shared__ unsigned long long cta_sum[32 * VEC];
    pdl_trigger();
    const int n = p.n;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int s = lane / lps, rl = lane - s * lps;
    int partner[kStages];
#pragma unroll
    for (int k = 0; k < kStages; ++k) partner[k] = (s ^ (1 << k)) * lps + rl;
    const int64_t blk = (int64_t)blockIdx.y * p.blk_stride;
    const unsigned lo = (unsigned)lane * VEC;  // this lane's float4 inside a 128-float row
    const Sc<float> &sc = p.sc;
    const float inv_q = 1.0f / (float)p.q;
    const float fx_scale_t = (float)p.fx_scale;
    const int warps_total = gridDim.x * kTmaWarps;
    const int warp_gid = blockIdx.x * kTmaWarps + wib;
    const int rows = 3 + p.max_deg;  // slot capacity
    const uint32_t row_bytes = 128 * sizeof(float);
    float *my_ring = ring + (size_t)wib * rows * 128;
    uint64_t *bar = &full_bar[wib];

    if (lane == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (threadIdx.x < 32 * VEC) cta_sum[threadIdx.x] = 0ull;
    __syncthreads();
    pdl_wait();  // everything below reads or overwrites what the previous launch wrote

    float Ss[VEC];
    {
        const long long *Sp = p.S_in + (int64_t)blockIdx.y * p.row_len + lo;
#pragma unroll
        for (int v = 0; v < VEC; ++v) Ss[v] = (float)((double)Sp[v] * p.fx_inv);
    }
    if (blockIdx.x == 0)
        for (unsigned k = threadIdx.x; k < p.row_len; k += kTmaWarps * 32) p.S_zero[(int64_t)blockIdx.y * p.row_len + k] = 0ll;

    long long colacc[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) colacc[v] = 0ll;

    // fetch of variable `i` into stage `st`: lane 0 posts the byte count, lanes 0..2 copy the h, m1, m2 rows,
    // lanes 3..3+deg-1 the neighbour rows (lane 3+k holds column index k after the shuffle)
    auto issue = [&](int i, int col_lane, int d) {
        const int c = __shfl_sync(0xffffffffu, col_lane, lane >= 3 ? lane - 3 : 0);
        float *dst = my_ring + (size_t)lane * 128;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the slot was read through the generic proxy
        const uint32_t id_bytes = (uint32_t)p.Rb;  // DISC: one id row = Rb bytes (a multiple of 16 on this path)
        if (lane == 0) mbar_expect_tx(bar, DISC ? 3 * row_bytes + (uint32_t)(d + 1) * id_bytes : (uint32_t)(3 + d) * row_bytes);
        __syncwarp();
        const int64_t own = blk + (int64_t)i * 128;
        if (lane == 0) bulk_g2s(dst, p.h + own, row_bytes, bar);
        else if (lane == 1) bulk_g2s(dst, p.m1 + own, row_bytes, bar);
        else if (lane == 2) bulk_g2s(dst, p.m2 + own, row_bytes, bar);
        else if (!DISC && lane < 3 + d) bulk_g2s(dst, p.g_in + blk + (int64_t)(unsigned)c * 128, row_bytes, bar);
        else if (DISC && lane <= 3 + d) {
            // id rows behind the three fp32 rows: neighbour k at byte 1536 + k*Rb, the variable's own ids after them
            signed char *d8 = reinterpret_cast<signed char *>(my_ring + 3 * 128) + (size_t)(lane - 3) * id_bytes;
            const int64_t var = lane < 3 + d ? (int64_t)(unsigned)c : (int64_t)i;
            bulk_g2s(d8, p.g8_in + blk + var * p.Rb, id_bytes, bar);
        }
    };
    // CSR row of variable i: first entry e0, degree d (warp-uniform), this lane's column index
    float cf_n = 1.0f, lamc_n = sc.two_lambda, shift_n = 0.0f;  // DISC: c^f, lambda c^a, sum_j W_ij / q of the row loaded last
    auto load_row = [&](int i, int &e0, int &d) -> int {
        e0 = 0;
        d = 0;
        if (i >= n) return 0;
        if (DISC) {  // S27, exactly as in potts_team_kernel
            const double rs = __ldg(p.rowsum + i);
            cf_n = rs > 0.0 ? (float)((double)p.q / rs) : 0.0f;
            lamc_n = rs > 0.0 ? (float)(0.5 * (double)sc.two_lambda * ((double)p.q / sqrt(rs))) : 0.0f;
            shift_n = (float)(rs / (double)p.q);
        }
        if (p.deg > 0) {
            e0 = i * p.deg;
            d = p.deg;
        } else {
            e0 = __ldg(p.row_ptr + i);
            d = __ldg(p.row_ptr + i + 1) - e0;
        }
        return lane < d ? __ldg(p.col + e0 + lane) : 0;
    };

    int i = warp_gid;
    int e0 = 0, deg = 0, e0_next = 0, deg_next = 0, col_next = 0;
    float cf = 1.0f, lam_c = sc.two_lambda, shift = 0.0f, cf_next = 1.0f, lamc_next = sc.two_lambda, shift_next = 0.0f;
    if (i < n) {
        const int c0 = load_row(i, e0, deg);
        cf = cf_n; lam_c = lamc_n; shift = shift_n;
        issue(i, c0, deg);
        col_next = load_row(i + warps_total, e0_next, deg_next);
        cf_next = cf_n; lamc_next = lamc_n; shift_next = shift_n;
    }
    for (int t = 0; i < n; ++t, i += warps_total) {
        const int in = i + warps_total;
        mbar_wait(bar, (uint32_t)(t & 1));
        const float *stage = my_ring + lo;
        const int64_t off = blk + (int64_t)i * 128 + lo;

        // coupling contraction f(s) = sum_j W_ij D_j(s), CSR order, rows already in shared memory
        float f[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) f[v] = 0.0f;
        unsigned own_ids = 0;
        if (DISC) {
            // one-hot neighbours: f(s) = sum_j W_ij [id_j == s], centred by sum_j W_ij / q; this lane's 4 replicas are
            // word rl of each Rb-byte id row
            const unsigned *ids = reinterpret_cast<const unsigned *>(my_ring + 3 * 128) + rl;
            const int words = p.Rb / 4;
            for (int k = 0; k < deg; ++k) {
                const unsigned w4 = ids[k * words];
                const float ww = UNITW ? 1.0f : __ldg(p.w + e0 + k);
#pragma unroll
                for (int v = 0; v < VEC; ++v) f[v] += ((w4 >> (8 * v)) & 0xffu) == (unsigned)s ? ww : 0.0f;
            }
            own_ids = ids[deg * words];
#pragma unroll
            for (int v = 0; v < VEC; ++v) f[v] -= shift;
        }
        for (int k = 0; k < (DISC ? 0 : deg); ++k) {
            const float4 nb = *reinterpret_cast<const float4 *>(stage + (3 + k) * 128);
            if (UNITW) {
                f[0] += nb.x; f[1] += nb.y; f[2] += nb.z; f[3] += nb.w;  // == fma(1, D_j, f)
            } else {
                const float ww = __ldg(p.w + e0 + k);
                f[0] = fma(ww, nb.x, f[0]); f[1] = fma(ww, nb.y, f[1]); f[2] = fma(ww, nb.z, f[2]); f[3] = fma(ww, nb.w, f[3]);
            }
        }
        float h[VEC];
        R m1, m2, hn;
        {
            const float4 a = *reinterpret_cast<const float4 *>(stage);
            const float4 b = *reinterpret_cast<const float4 *>(stage + 128);
            const float4 c = *reinterpret_cast<const float4 *>(stage + 256);
            h[0] = a.x; h[1] = a.y; h[2] = a.z; h[3] = a.w;
            m1.v[0] = b.x; m1.v[1] = b.y; m1.v[2] = b.z; m1.v[3] = b.w;
            m2.v[0] = c.x; m2.v[1] = c.y; m2.v[2] = c.z; m2.v[3] = c.w;
        }
        // the slot is in registers now: refill it with the warp's next variable while this one is computed
        __syncwarp();
        const int deg_issue = deg_next;
        const float cf_i = cf, lamc_i = lam_c;  // this variable's factors; the rotation below is for the next one
        e0 = e0_next;   // (the neighbour sum above is done with this variable's row)
        deg = deg_next;
        cf = cf_next; lam_c = lamc_next; shift = shift_next;
        if (in < n) {
            issue(in, col_next, deg_issue);
            col_next = load_row(in + warps_total, e0_next, deg_next);
            cf_next = cf_n; lamc_next = lamc_n; shift_next = shift_n;
        }
        // softmax of h(t) across the states
        float P[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            float mx = h[v];
#pragma unroll
            for (int k = 0; k < kStages; ++k) mx = fmax(mx, __shfl_sync(0xffffffffu, mx, partner[k]));
            const float e = fexp(h[v] - mx);
            float z = e;
#pragma unroll
            for (int k = 0; k < kStages; ++k) z += __shfl_sync(0xffffffffu, z, partner[k]);
            P[v] = e * frcp(z);
        }
        // g^p (S26), then g^h = P (g^p - <g^p>_P) (S20), optimiser
        const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            float gp;
            if (DISC) {
                const float own = ((((own_ids >> (8 * v)) & 0xffu) == (unsigned)s) ? 1.0f : 0.0f) - inv_q;
                gp = fma(h[v], sc.inv_beta, fma(lamc_i, Ss[v] - own, -(cf_i * f[v])));
            } else {
                gp = fma(h[v], sc.inv_beta, fma(sc.two_lambda, Ss[v] - P[v], -f[v]));
            }
            float gbar = P[v] * gp;
#pragma unroll
            for (int k = 0; k < kStages; ++k) gbar += __shfl_sync(0xffffffffu, gbar, partner[k]);
            const float g = sc.gamma * (P[v] * (gp - gbar));
            hn.v[v] = opt_update(h[v], g, m1.v[v], m2.v[v], sc);
            h[v] = hn.v[v];
        }
        hn.st_stream(p.h + off);
        if (use_m1) m1.st_stream(p.m1 + off);
        if (use_m2) m2.st_stream(p.m2 + off);
        // centred marginals of the new fields -> g_out, and their column sums
        R po;
        int win[VEC] = {0, 0, 0, 0};
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            float mx = h[v];
#pragma unroll
            for (int k = 0; k < kStages; ++k) mx = fmax(mx, __shfl_sync(0xffffffffu, mx, partner[k]));
            const float e = fexp(h[v] - mx);
            float z = e;
#pragma unroll
            for (int k = 0; k < kStages; ++k) z += __shfl_sync(0xffffffffu, z, partner[k]);
            po.v[v] = fma(e, frcp(z), -inv_q);
            if (DISC) {  // centred one-hot of the new fields: lowest state among the maxima (rounding rule R3)
                int cand = h[v] == mx ? s : 1 << 30;
#pragma unroll
                for (int k = 0; k < kStages; ++k) cand = min(cand, __shfl_sync(0xffffffffu, cand, partner[k]));
                win[v] = cand;
                po.v[v] = (cand == s ? 1.0f : 0.0f) - inv_q;
            }
            colacc[v] += __float2ll_rn(po.v[v] * fx_scale_t);
        }
        if (DISC) {
            if (s == 0) st_bytes<VEC>(p.g8_out + blk + (int64_t)i * p.Rb + (unsigned)rl * VEC, win);
        } else {
            po.st(p.g_out + off);
        }
    }

    // column sums: exact integer adds -- lanes -> CTA (shared atomics) -> grid (global atomics)
    __syncthreads();
#pragma unroll
    for (int v = 0; v < VEC; ++v)
        if (colacc[v] != 0ll) atomicAdd(&cta_sum[lane * VEC + v], (unsigned long long)colacc[v]);
    __syncthreads();
    if (threadIdx.x < p.row_len) {
        const unsigned long long v = cta_sum[threadIdx.x];
        if (v != 0ull)
            atomicAdd(reinterpret_cast<unsigned long long *>(p.S_out) + (int64_t)blockIdx.y * p.row_len + threadIdx.x, v);
    }
}

// ---- host side ----
bool potts_tma_applicable(const Handle *hd) {
    const int q = hd->dp.q, Rb = hd->Rb, deg = hd->dp.max_deg;
    if (hd->dp.vw) return false;  // node-weighted balance term: register path / state-innermost kernel only
    if (hd->opt_potts_tma == 0) return false;
    if (hd->gather_disc && Rb % 16 != 0) return false;  // id rows travel as bulk copies of Rb bytes (q <= 8)
    if (q < 2 || (q & (q - 1)) != 0 || Rb % 4 != 0 || q * (Rb / 4) != 32) return false;  // one variable = one warp of float4 lanes
    return deg >= 1 && deg <= kTmaMaxDeg && hd->dp.nnz < ((int64_t)1 << 31);
}

template <int QPAD, bool UNITW, bool DISC>
static cudaError_t launch_tma_one(Handle *hd, const PottsTmaParams &p, int blk_count, size_t smem) {
    // CTAs resident at once, per ring size (the degree sets it), cached per handle (= per device and context)
    const void *fn = reinterpret_cast<const void *>(&potts_tma_kernel<QPAD, UNITW, DISC>);
    int &resident = hd->resident_ctas[{fn, smem}];
    if (resident == 0) {
        const size_t smem_max = (size_t)kTmaWarps * (3 + kTmaMaxDeg) * 128 * sizeof(float);
        cudaError_t e = cudaFuncSetAttribute(potts_tma_kernel<QPAD, UNITW, DISC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
        if (e != cudaSuccess) return e;
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, potts_tma_kernel<QPAD, UNITW, DISC>, kTmaWarps * 32, smem) != cudaSuccess ||
            occ < 1)
            occ = 1;
        resident = occ * hd->sm_count;
    }
    const unsigned gx = (unsigned)std::min<int64_t>(resident, ceil_div(p.n, kTmaWarps));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(gx, (unsigned)blk_count);
    cfg.blockDim = dim3(kTmaWarps * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = hd->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, potts_tma_kernel<QPAD, UNITW, DISC>, p);
}

// One fp32 exact-gradient Potts step of replica blocks [blk_begin, blk_begin + blk_count); false = not applicable.
bool launch_potts_tma(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count) {
    if (!potts_tma_applicable(hd)) return false;
    const int Rb = hd->Rb, q = hd->dp.q;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    PottsTmaParams p;
    p.h = hd->h + base;
    p.m1 = hd->m1 + base;
    p.m2 = hd->m2 + base;
    p.g_in = hd->g[hd->cur] + base;
    p.g_out = hd->g[hd->cur ^ 1] + base;
    p.blk_stride = hd->rows * Rb;
    p.col = hd->dp.col;
    p.w = hd->dp.w;
    p.sc = Sc<float>(sc);
    const int64_t so = (int64_t)blk_begin * q * Rb;
    const int t = sc.t;  // column-sum buffers rotate with the step number exactly as in launch_potts_typed
    p.S_in = hd->colsum[t % 3] + so;
    p.S_out = hd->colsum[(t + 1) % 3] + so;
    p.S_zero = hd->colsum[(t + 2) % 3] + so;
    p.fx_scale = hd->colsum_scale;
    p.fx_inv = 1.0 / hd->colsum_scale;
    p.n = hd->dp.n;
    p.q = q;
    p.Rb = Rb;
    p.deg = hd->dp.uniform_deg;
    p.max_deg = hd->dp.max_deg;
    p.row_ptr = hd->dp.row_ptr;
    p.row_len = 128;
    const size_t smem = (size_t)kTmaWarps * (3 + p.max_deg) * 128 * sizeof(float);
    p.g8_in = reinterpret_cast<const signed char *>(hd->g[hd->cur]) + base;
    p.g8_out = reinterpret_cast<signed char *>(hd->g[hd->cur ^ 1]) + base;
    p.rowsum = hd->rowsum;
    cudaError_t e;
    const bool unit = p.w == nullptr, disc = hd->gather_disc;
    auto go = [&](auto qtag) -> cudaError_t {
        constexpr int Q = decltype(qtag)::value;
        if (disc) return unit ? launch_tma_one<Q, true, true>(hd, p, blk_count, smem) : launch_tma_one<Q, false, true>(hd, p, blk_count, smem);
        return unit ? launch_tma_one<Q, true, false>(hd, p, blk_count, smem) : launch_tma_one<Q, false, false>(hd, p, blk_count, smem);
    };
    switch (q) {
        case 2: e = go(std::integral_constant<int, 2>{}); break;
        case 4: e = go(std::integral_constant<int, 4>{}); break;
        case 8: e = go(std::integral_constant<int, 8>{}); break;
        case 16: e = go(std::integral_constant<int, 16>{}); break;
        default: e = go(std::integral_constant<int, 32>{}); break;
    }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    hd->launches++;
    hd->tma_launches++;
    return true;
}

}  // namespace fem
