// Fused annealing step for the q-state Potts kind (balanced minimum cut).
//
// A TEAM of lanes owns one variable: the variable's row is q*Rb contiguous values [state][replica], lane l
// of the team holds VEC consecutive replicas of state s = l / (Rb/VEC), so every access of the team -- the
// streamed h / m1 / m2 rows and each CSR neighbour gather of the centred marginals D_j = P_j - 1/q -- is one
// contiguous, vectorised segment (north_star subsystem 1).  Sums over the states (softmax normaliser, the
// mean <g^p>_P of the chain rule S20) are butterfly shuffles across the team.  Per step and
// lane: softmax of the fields, f_i(s) = sum_j W_ij D_j(s) over the CSR row, g^p from S26
// (edge-once reading R1) with the balance term 2*lambda*[S_s - P_i(s)] (balance(),
// PAPER.md:536) and the entropy term h_i(s)/beta (ln P = h - lse; lse is constant in s and cancels in
// S20, like the "+1"), the chain rule, Adam, and the next marginals.  The column sums S_s of the NEXT step
// are a by-product: every lane adds its new D' in 64-bit fixed point, so the sum is exact, independent of
// the order and of the replica blocking, and integer atomics keep it deterministic (no float atomics).
#include <algorithm>
#include <map>

#include "device_math.cuh"

namespace fem {

template <typename T>
struct PottsParams {
    BlockArrays<T> a;
    DevProblem dp;
    Sc<T> sc;
    const double *rowsum;   // sum_j W_ij per node (manipulated gradients: c^f_i, c^a_i)
    const signed char *g8_in;  // manipulated gradients: the state id argmax_s h_j(s), one byte per (variable, replica)
    signed char *g8_out;       // (device_math.cuh); byte offsets of a replica block = its element offsets
    const long long *S_in;  // fixed-point column sums of D(t), [q*Rb] per replica block
    long long *S_out;       // accumulated by this launch: column sums of D(t+1)
    long long *S_zero;      // cleared by this launch (the buffer the launch after next accumulates into)
    double fx_scale, fx_inv;
    int disc_out;        // the gathered quantity is the centred one-hot vector (manipulated gradients)
    int lps;             // lanes per state = Rb / VEC
    int team;            // QPAD * lps lanes per variable (<= 32)
    int teams_per_warp;  // 32 / team
    unsigned row_len;    // q * Rb
};

__device__ __forceinline__ long long fixed_of(float x, float scale) { return __float2ll_rn(x * scale); }
__device__ __forceinline__ long long fixed_of(double x, double scale) { return __double2ll_rn(x * scale); }
__device__ __forceinline__ float shfl_any(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_any(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }

constexpr int kGatherChunk = 5;  // neighbour rows in flight per lane

constexpr int kTeamMinCtas = 4;  // CTAs per SM the exact-gradient kernel is compiled for (measured optimum)
template <typename T, int QPAD, int VEC, bool STEP, bool DISC, bool UNITW>
__global__ void __launch_bounds__(kThreads, DISC ? 3 : kTeamMinCtas) potts_team_kernel(const PottsParams<T> p) {
    using R = Row<T, VEC>;
    constexpr int kStages = QPAD == 32 ? 5 : QPAD == 16 ? 4 : QPAD == 8 ? 3 : QPAD == 4 ? 2 : 1;
    __shared__ unsigned long long cta_sum[32 * VEC];
    pdl_trigger();
    const int q = p.dp.q, n = p.dp.n;
    const int lane = threadIdx.x & 31;
    const int tw = lane / p.team;       // team within the warp
    const int l = lane - tw * p.team;   // lane within the team
    const int s = l / p.lps;            // state of this lane
    const int rl = l - s * p.lps;       // replica group of this lane
    const bool lane_ok = tw < p.teams_per_warp && s < q;
    int partner[kStages];               // butterfly partners across the states of the same replica group
#pragma unroll
    for (int k = 0; k < kStages; ++k)
        partner[k] = tw < p.teams_per_warp ? tw * p.team + ((s ^ (1 << k)) * p.lps + rl) : lane;

    // centred one-hot of the team's fields: 1 - 1/q on the lowest state among the maxima (rounding rule R3), -1/q
    // elsewhere (S27's e_j; constants in s cancel in S20 like for the centred marginals)
    auto winner = [&](T hv, T mx, bool okk) -> int {
        int cand = (okk && hv == mx) ? s : 1 << 30;
#pragma unroll
        for (int k = 0; k < kStages; ++k) cand = min(cand, __shfl_sync(0xffffffffu, cand, partner[k]));
        return cand;
    };
    const int64_t blk = (int64_t)blockIdx.y * p.a.blk_stride;
    const unsigned lo = (unsigned)(s * p.lps + rl) * VEC;  // offset inside a row
    const T *__restrict__ gin = p.a.g_in + blk + lo;
    const Sc<T> &sc = p.sc;
    const T inv_q = (T)1 / (T)q;
    const T fx_scale_t = (T)p.fx_scale;
    const T neg_big = (T)-3.0e38;
    const int warps_total = gridDim.x * (kThreads / 32);
    const int warp_id = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    const int stride = warps_total * p.teams_per_warp;

    if (threadIdx.x < 32 * VEC) cta_sum[threadIdx.x] = 0ull;
    pdl_wait();  // everything below reads or overwrites what the previous launch wrote

    T Ss[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) Ss[v] = (T)0;
    if (STEP && lane_ok) {
        const long long *Sp = p.S_in + (int64_t)blockIdx.y * p.row_len + lo;
#pragma unroll
        for (int v = 0; v < VEC; ++v) Ss[v] = (T)((double)Sp[v] * p.fx_inv);
    }
    if (blockIdx.x == 0)
        for (unsigned k = threadIdx.x; k < p.row_len; k += kThreads) p.S_zero[(int64_t)blockIdx.y * p.row_len + k] = 0ll;

    long long colacc[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) colacc[v] = 0ll;

    for (int base = warp_id * p.teams_per_warp; base < n; base += stride) {  // warp-uniform trip count
        const int i = base + tw;
        const bool ok = lane_ok && i < n;
        const int64_t off = blk + (int64_t)(ok ? i : 0) * p.row_len + lo;
        // node weight V_i of the balance term (S33-S35; integral, 1 without node weights): the term is
        // 2 lambda V_i [sum_j V_j P_j(s) - V_i P_i(s)], and the column sums are those of V_i D_i(s)
        const T Vi = (p.dp.vw && ok) ? (T)__ldg(p.dp.vw + i) : (T)1;
        T h[VEC];
        {
            R r;
            if (ok) r = R::ld_stream(p.a.h + off);
#pragma unroll
            for (int v = 0; v < VEC; ++v) h[v] = ok ? r.v[v] : neg_big;
        }
        if (STEP) {
            // coupling contraction f(s) = sum_j W_ij D_j(s): kGatherChunk neighbour rows in flight
            T f[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) f[v] = (T)0;
            if (ok) {
                int e0, e1;
                if (p.dp.uniform_deg > 0) {
                    e0 = i * p.dp.uniform_deg;
                    e1 = e0 + p.dp.uniform_deg;
                } else {
                    e0 = __ldg(p.dp.row_ptr + i);
                    e1 = __ldg(p.dp.row_ptr + i + 1);
                }
                if (DISC) {
                    // one-hot neighbours: f(s) = sum_j W_ij [state_j == s]; a neighbour is VEC bytes per lane.  Centred
                    // by sum_j W_ij / q (constant in s, cancels in S20) so that f stays as small as in the exact path.
                    constexpr int kIds = 10;
                    const signed char *__restrict__ gin8 = p.g8_in + blk + (unsigned)rl * VEC;
                    for (int e = e0; e < e1; e += kIds) {
                        unsigned jj[kIds];
                        T ww[kIds];
                        unsigned ids[kIds];  // VEC state ids per neighbour, packed
#pragma unroll
                        for (int k = 0; k < kIds; ++k) {
                            const bool in = e + k < e1;
                            jj[k] = in ? (unsigned)__ldg(p.dp.col + e + k) : (unsigned)i;
                            ww[k] = in ? (UNITW ? (T)1 : (T)__ldg(p.dp.w + e + k)) : (T)0;
                        }
#pragma unroll
                        for (int k = 0; k < kIds; ++k) ids[k] = ld_bytes_packed<VEC>(gin8 + jj[k] * (unsigned)p.a.Rb);
#pragma unroll
                        for (int k = 0; k < kIds; ++k)
#pragma unroll
                            for (int v = 0; v < VEC; ++v) f[v] += ((ids[k] >> (8 * v)) & 0xffu) == (unsigned)s ? ww[k] : (T)0;
                    }
                    const T shift = (T)(__ldg(p.rowsum + i) / (double)q);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) f[v] -= shift;
                } else {
                const unsigned row_bytes = p.row_len * (unsigned)sizeof(T);
                auto row_of = [&](unsigned j) -> const T * {  // one wide multiply-add per neighbour row
                    return reinterpret_cast<const T *>(reinterpret_cast<const char *>(gin) + (unsigned long long)j * row_bytes);
                };
                if (UNITW && (e1 - e0) % kGatherChunk == 0) {
                    // unit weights, whole chunks (10-regular graphs): indices, then kGatherChunk rows in flight, then adds
                    for (int e = e0; e < e1; e += kGatherChunk) {
                        unsigned jj[kGatherChunk];
                        R nb[kGatherChunk];
#pragma unroll
                        for (int k = 0; k < kGatherChunk; ++k) jj[k] = (unsigned)__ldg(p.dp.col + e + k);
#pragma unroll
                        for (int k = 0; k < kGatherChunk; ++k) nb[k] = R::ld(row_of(jj[k]));
#pragma unroll
                        for (int k = 0; k < kGatherChunk; ++k)
#pragma unroll
                            for (int v = 0; v < VEC; ++v) f[v] += nb[k].v[v];  // == fma(1, D_j, f)
                    }
                } else {
                for (int e = e0; e < e1; e += kGatherChunk) {
                    unsigned jj[kGatherChunk];
                    T ww[kGatherChunk];
                    R nb[kGatherChunk];
#pragma unroll
                    for (int k = 0; k < kGatherChunk; ++k) {
                        const bool in = e + k < e1;
                        jj[k] = in ? (unsigned)__ldg(p.dp.col + e + k) : (unsigned)i;
                        ww[k] = in ? (UNITW ? (T)1 : (T)__ldg(p.dp.w + e + k)) : (T)0;
                    }
#pragma unroll
                    for (int k = 0; k < kGatherChunk; ++k) nb[k] = R::ld(row_of(jj[k]));
#pragma unroll
                    for (int k = 0; k < kGatherChunk; ++k)
#pragma unroll
                        for (int v = 0; v < VEC; ++v) f[v] = fma(ww[k], nb[k].v[v], f[v]);
                }
                }
                }
            }
            unsigned own_ids = 0;
            if (DISC && ok) own_ids = ld_bytes_packed<VEC>(p.g8_in + blk + (int64_t)i * p.a.Rb + (unsigned)rl * VEC);
            // softmax of h(t) across the team's states
            T P[VEC], own[VEC];  // own: what the balance term subtracts (P_i, or the centred one-hot e_i when manipulated)
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                T mx = h[v];
#pragma unroll
                for (int k = 0; k < kStages; ++k) mx = fmax(mx, shfl_any(mx, partner[k]));
                const T e = ok ? fexp(h[v] - mx) : (T)0;
                T z = e;
#pragma unroll
                for (int k = 0; k < kStages; ++k) z += shfl_any(z, partner[k]);
                P[v] = e * frcp(z);
                own[v] = P[v];
                // manipulated: the variable's own one-hot vector is the state id the previous launch stored for it
                if (DISC) own[v] = ((((own_ids >> (8 * v)) & 0xffu) == (unsigned)s) ? (T)1 : (T)0) - inv_q;
            }
            // manipulated gradients (S27): c^f = q / sum_j W_ij on the cut term, lambda c^a with
            // c^a = q / sqrt(sum_j W_ij) on the balance term (S26's 2 lambda becomes lambda); no neighbours: 0
            T cf = (T)1, lam_c = sc.two_lambda;
            if (DISC) {
                const double rs = ok ? __ldg(p.rowsum + i) : 0.0;
                cf = rs > 0.0 ? (T)((double)q / rs) : (T)0;
                lam_c = rs > 0.0 ? (T)(0.5 * (double)sc.two_lambda * ((double)q / sqrt(rs))) : (T)0;
            }
            // g^p (S26), then g^h = P (g^p - <g^p>_P) (S20), Adam
            R m1 = {}, m2 = {}, hn;
            const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();
            if (ok) {
                if (use_m1) m1 = R::ld_stream(p.a.m1 + off);
                if (use_m2) m2 = R::ld_stream(p.a.m2 + off);
            }
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                T gp = (T)0;
                if (ok) {
                    // explicit fma: potts_tma_kernel must round exactly alike
                    // (V_i = 1: the products below are exact, so nothing changes without node weights)
                    if (DISC) gp = fma(h[v], sc.inv_beta, fma(lam_c * Vi, Ss[v] - Vi * own[v], -(cf * f[v])));
                    else gp = fma(h[v], sc.inv_beta, fma(sc.two_lambda * Vi, Ss[v] - Vi * P[v], -f[v]));
                }
                T gbar = P[v] * gp;
#pragma unroll
                for (int k = 0; k < kStages; ++k) gbar += shfl_any(gbar, partner[k]);
                if (ok) {
                    const T g = sc.gamma * (P[v] * (gp - gbar));
                    hn.v[v] = opt_update(h[v], g, m1.v[v], m2.v[v], sc);
                    h[v] = hn.v[v];
                }
            }
            if (ok) {
                hn.st_stream(p.a.h + off);
                if (use_m1) m1.st_stream(p.a.m1 + off);
                if (use_m2) m2.st_stream(p.a.m2 + off);
            }
        }
        // centred marginals D = P - 1/q of the (new) fields -> g_out, and their column sums.  Constants in s
        // cancel in S20, and near the uniform start the deviation from 1/q is all the signal there is, so it
        // is what gets stored and gathered.
        R po;
        int win[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            win[v] = 0;
            T mx = h[v];
#pragma unroll
            for (int k = 0; k < kStages; ++k) mx = fmax(mx, shfl_any(mx, partner[k]));
            const T e = ok ? fexp(h[v] - mx) : (T)0;
            T z = e;
#pragma unroll
            for (int k = 0; k < kStages; ++k) z += shfl_any(z, partner[k]);
            po.v[v] = fma(e, frcp(z), -inv_q);
            if (DISC) {
                win[v] = winner(h[v], mx, ok);
                po.v[v] = (win[v] == s ? (T)1 : (T)0) - inv_q;
            }
            // fixed point straight from the compute type: the scale is a power of two, so the product is exact
            if (ok) colacc[v] += (long long)Vi * fixed_of(po.v[v], fx_scale_t);
        }
        if (DISC) {  // the state-0 lane of each replica group stores the VEC winners as bytes
            if (ok && s == 0) st_bytes<VEC>(p.g8_out + blk + (int64_t)i * p.a.Rb + (unsigned)rl * VEC, win);
        } else if (ok) {
            po.st(p.a.g_out + off);
        }
    }

    // column sums: exact integer adds -- lanes -> CTA (shared atomics) -> grid (global atomics)
    __syncthreads();
    if (lane_ok) {
#pragma unroll
        for (int v = 0; v < VEC; ++v)
            if (colacc[v] != 0ll) atomicAdd(&cta_sum[l * VEC + v], (unsigned long long)colacc[v]);
    }
    __syncthreads();
    if (threadIdx.x < p.row_len) {  // row_len = q * Rb <= 32 * VEC; team lane l covers row offsets l*VEC ..
        const unsigned long long v = cta_sum[threadIdx.x];
        if (v != 0ull)
            atomicAdd(reinterpret_cast<unsigned long long *>(p.S_out) + (int64_t)blockIdx.y * p.row_len + threadIdx.x, v);
    }
}

// grid-stride kernel: never more CTAs than are resident at once (occupancy x SMs), so no second wave
template <typename T, int QPAD, int VEC, bool STEP, bool DISC, bool UNITW>
static void launch_potts_w(Handle *hd, const PottsParams<T> &p, dim3 grid) {
    // CTAs resident at once for THIS instantiation, cached per handle (= per device and context)
    int &r = hd->resident_ctas[{reinterpret_cast<const void *>(&potts_team_kernel<T, QPAD, VEC, STEP, DISC, UNITW>), 0}];
    if (r == 0) {
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, potts_team_kernel<T, QPAD, VEC, STEP, DISC, UNITW>, kThreads,
                                                          0) != cudaSuccess || occ < 1)
            occ = 1;
        r = occ * hd->sm_count;
    }
    grid.x = std::min<unsigned>(grid.x, (unsigned)r);
    launch_pdl(potts_team_kernel<T, QPAD, VEC, STEP, DISC, UNITW>, grid, dim3(kThreads), hd->stream, p);
}

template <typename T, int QPAD, int VEC, bool STEP, bool DISC>
static void launch_potts_one(Handle *hd, const PottsParams<T> &p, dim3 grid) {
    if (p.dp.w) launch_potts_w<T, QPAD, VEC, STEP, DISC, false>(hd, p, grid);
    else launch_potts_w<T, QPAD, VEC, STEP, DISC, true>(hd, p, grid);
}

template <typename T, int QPAD, int VEC>
static void launch_potts_t(Handle *hd, const PottsParams<T> &p, dim3 grid, bool step) {
    // DISC (manipulated gradients) is a template parameter so that the exact-gradient kernel carries none of it
    const bool disc = p.disc_out != 0;
    if (step && disc) launch_potts_one<T, QPAD, VEC, true, true>(hd, p, grid);
    else if (step) launch_potts_one<T, QPAD, VEC, true, false>(hd, p, grid);
    else if (disc) launch_potts_one<T, QPAD, VEC, false, true>(hd, p, grid);
    else launch_potts_one<T, QPAD, VEC, false, false>(hd, p, grid);
}

template <typename T, int QPAD>
static void launch_potts_v(Handle *hd, const PottsParams<T> &p, dim3 grid, bool step, int vec) {
    if (vec == 4) launch_potts_t<T, QPAD, 4>(hd, p, grid, step);
    else if (vec == 2) launch_potts_t<T, QPAD, 2>(hd, p, grid, step);
    else launch_potts_t<T, QPAD, 1>(hd, p, grid, step);
}

bool launch_potts_tma(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count);  // k_step_potts_tma.cu
bool launch_potts_si(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count);    // k_step_potts_si.cu

int potts_qpad(int q) {
    int qp = 2;
    while (qp < q) qp <<= 1;
    return qp;
}
int potts_vec(int Rb) { return Rb % 4 == 0 ? 4 : (Rb % 2 == 0 ? 2 : 1); }
// a replica block fits the team mapping when one variable's lanes fit a warp
bool potts_block_ok(int q, int Rb) { return potts_qpad(q) * (Rb / potts_vec(Rb)) <= 32; }

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
    // column-sum buffers rotate with the step number: step t reads [t%3], accumulates [(t+1)%3], clears [(t+2)%3];
    // the preparation at step t accumulates [t%3] (cleared by the caller) and clears [(t+1)%3]
    const int64_t so = (int64_t)blk_begin * q * Rb;
    const int t = sc.t;
    p.S_in = hd->colsum[t % 3] + so;
    p.S_out = hd->colsum[(step ? t + 1 : t) % 3] + so;
    p.S_zero = hd->colsum[(step ? t + 2 : t + 1) % 3] + so;
    p.rowsum = hd->rowsum;
    p.g8_in = reinterpret_cast<const signed char *>(hd->g[hd->cur]) + base;
    p.g8_out = reinterpret_cast<signed char *>(step ? hd->g[hd->cur ^ 1] : hd->g[hd->cur]) + base;
    p.disc_out = hd->gather_disc ? 1 : 0;
    p.fx_scale = hd->colsum_scale;
    p.fx_inv = 1.0 / hd->colsum_scale;
    const int vec = potts_vec(Rb);
    const int qpad = potts_qpad(q);
    p.lps = Rb / vec;
    p.team = qpad * p.lps;
    p.teams_per_warp = 32 / p.team;
    p.row_len = (unsigned)(q * Rb);
    const int64_t warps_needed = ceil_div(hd->dp.n, p.teams_per_warp);
    const int nblk = (int)std::min<int64_t>(kColBlocks, ceil_div(warps_needed, kThreads / 32));
    dim3 grid((unsigned)nblk, (unsigned)blk_count);
    switch (qpad) {
        case 2: launch_potts_v<T, 2>(hd, p, grid, step, vec); break;
        case 4: launch_potts_v<T, 4>(hd, p, grid, step, vec); break;
        case 8: launch_potts_v<T, 8>(hd, p, grid, step, vec); break;
        case 16: launch_potts_v<T, 16>(hd, p, grid, step, vec); break;
        default: launch_potts_v<T, 32>(hd, p, grid, step, vec); break;
    }
    hd->launches++;
}

// step == false: centred marginals + column sums of the current fields into g[cur] / colsum[t % 3].
void launch_potts(Handle *hd, const StepScalars &sc, bool wide, bool step, int blk_begin, int blk_count) {
    if (!step) {
        const size_t bytes = (size_t)hd->dp.q * hd->Rb * blk_count * sizeof(long long);
        cudaMemsetAsync(hd->colsum[sc.t % 3] + (int64_t)blk_begin * hd->dp.q * hd->Rb, 0, bytes, hd->stream);
    }
    if (hd->si_live) {  // the fp32 arrays are in the state-innermost layout: only this kernel reads it (fem_anneal)
        (void)launch_potts_si(hd, sc, blk_begin, blk_count);  // a failed launch surfaces through cudaGetLastError
        return;
    }
    if (!wide && step && launch_potts_tma(hd, sc, blk_begin, blk_count)) return;  // TMA-staged fast path where it applies
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
