// Potts (balanced minimum cut) step on a STATE-INNERMOST replica block: fp32, exact gradient, q = 4 or 8, replica blocks
// of Rb = 4, 8, 16 or 32 with n a multiple of 32 / Rb -- BASELINE.json configs[2] (q = 8, 10-regular, n = 100,000, R = 64).
//
// Why (profiles/r02_cfg2_step.md).  The team kernels spread the q states of a variable over lanes: every sum over
// states is a butterfly of shuffles and every lane repeats the scalar work of its 4 fields (634 warp instructions per
// 128 fields, issue-bound at 0.47 of the HBM roof on cfg 2).  A lane-per-replica kernel (round 2, first half; removed: profiles/r02_cfg2_step.md) does
// the arithmetic with a lane owning all q states of one (variable, replica) cell, but keeps the [state][replica] rows in
// HBM, so every row passes through shared memory twice (22% of its instructions are LDS / STS and it stalls on them:
// 9.1 ns per kilo-field against 7.4).  Here the LAYOUT follows the arithmetic instead.  For the fp32 steps of one
// fem_anneal call the block's arrays h, m1, m2 and the gather buffer are re-laid out in place (potts_si_relayout_kernel,
// a permutation inside each 32q-float chunk, once in and once out per call):
//
//   cell c = i * Rb + r  (variable i, replica r);  groups of 32 consecutive cells = G = 32 / Rb variables;
//   field (i, s, r)  ->  (c / 32) * 32q + (s / 4) * 128 + (c % 32) * 4 + (s % 4)          ["quad-major" inside a group]
//
// so lane l of the warp that works on group `it` owns cell it * 32 + l and reads / writes its q states as q / 4 float4
// pieces that sit 512 B apart: every global access is a 16-byte vector, a warp instruction covers 512 contiguous bytes,
// a neighbour's states arrive in the lane that needs them (no shuffles, no shared memory), and all sums over states
// are register adds.  A neighbour gather of one lane is q / 4 16-byte loads; the Rb lanes of a variable read Rb * 16
// contiguous bytes per piece.
//
// The arithmetic is potts_team_kernel's, operation for operation (same device functions, CSR-order neighbour sum, sums
// over states in the butterfly's tree order), so the kernels are bit-identical
// (tests/test_gpu_parity.py::test_potts_si_bit_identical_to_team_kernel) and results do not depend on the replica blocking.
// Rows a1-a4 of DESIGN.md section 2: softmax, S26 coupling + balance terms, chain rule S20
// (PAPER.md:599), optimiser update.
#include <algorithm>

#include "device_math.cuh"

namespace fem {

struct PottsSiParams {
    float *h, *m1, *m2;   // block base pointers (blockIdx.y walks replica blocks)
    const float *g_in;
    float *g_out;
    int64_t blk_stride;
    const int *col;
    const float *w;       // nullptr = unit weights
    const int *row_ptr;
    const float *vw;      // node weights V_i of the balance term (S33-S35), or nullptr
    Sc<float> sc;
    const long long *S_in;
    long long *S_out, *S_zero;
    double fx_scale, fx_inv;
    int n;
    int deg;              // uniform degree, or 0: rows from row_ptr
    int iters;            // groups of 32 cells: n * Rb / 32
};

constexpr int kSiWarps = 4;  // warps per CTA (every warp works on its own)

// sum / maximum over the states in the butterfly's order: ((z0+z1)+(z2+z3))+((z4+z5)+(z6+z7))
template <int Q>
__device__ __forceinline__ float si_tree_sum(const float (&z)[Q]) {
    float t[Q];
#pragma unroll
    for (int s = 0; s < Q; ++s) t[s] = z[s];
#pragma unroll
    for (int k = 1; k < Q; k <<= 1)
#pragma unroll
        for (int s = 0; s < Q; s += 2 * k) t[s] = t[s] + t[s + k];
    return t[0];
}
template <int Q>
__device__ __forceinline__ float si_tree_max(const float (&z)[Q]) {
    float t[Q];
#pragma unroll
    for (int s = 0; s < Q; ++s) t[s] = z[s];
#pragma unroll
    for (int k = 1; k < Q; k <<= 1)
#pragma unroll
        for (int s = 0; s < Q; s += 2 * k) t[s] = fmax(t[s], t[s + k]);
    return t[0];
}

// float offset of variable j's cells inside a block (before the lane's own r * 4 and the piece's x * 128)
template <int Q, int RB>
__device__ __forceinline__ unsigned si_var_offset(unsigned j) {
    constexpr unsigned G = 32 / RB;
    if (Q == 4) return j * (unsigned)(Q * RB);
    return j * (unsigned)(Q * RB) - (j & (G - 1)) * (unsigned)(RB * (Q - 4));
}

// DEG > 0: every row of the CSR has exactly DEG entries (regular graphs): column indices of the NEXT group are
// prefetched into registers and all loops over the neighbours are unrolled.  DEG = 0: rows of any length.
// BATCH: neighbour rows requested before the first of them is added (registers in flight: BATCH * Q per lane).
// STAGE (regular graphs only): the own rows and the neighbour rows of the NEXT group are copied by cp.async into a
// per-warp slot of shared memory ((3 + DEG) * Q / 4 pieces of 512 B, every lane reads back only what it copied: no warp
// synchronisation) while the current group is computed, so no warp waits for a memory round trip; BATCH is then unused.
template <int Q, int RB, bool UNITW, int DEG, int BATCH, bool STAGE, int MINB>
__global__ void __launch_bounds__(kSiWarps * 32, MINB) potts_si_kernel(const __grid_constant__ PottsSiParams p) {
    constexpr int G = 32 / RB, NQ = Q / 4, GROUP = 32 * Q, ROW = Q * RB;
    constexpr int ND = DEG > 0 ? DEG : 1;
    constexpr int PIECES = (3 + ND) * NQ;  // STAGE: 512-byte pieces of a warp's slot: h, m1, m2, then the neighbours
    static_assert(!STAGE || DEG > 0, "staging needs a regular degree");
    extern __shared__ __align__(16) float4 si_slots[];  // STAGE: [warp][PIECES][32 lanes]
    __shared__ unsigned long long cta_sum[ROW];
    pdl_trigger();
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int g = lane / RB, r = lane - g * RB;
    const int64_t blk = (int64_t)blockIdx.y * p.blk_stride;
    const Sc<float> &sc = p.sc;
    const float inv_q = 1.0f / (float)Q;
    const float fx_scale_t = (float)p.fx_scale;
    const int warps_total = gridDim.x * kSiWarps;
    const int warp_gid = blockIdx.x * kSiWarps + wib;
    const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();
    const float *gsrc = p.g_in + blk + r * 4;

    // raw column indices (and weights) of a group's variables: static problem structure, legal before pdl_wait.  They
    // stay raw until they are used one iteration later, so the load has a whole iteration to land.
    int cr[ND];
    float wj[ND];
    auto load_cols = [&](int it_) {
        if (DEG > 0) {
            const int i = it_ * G + g;
#pragma unroll
            for (int k = 0; k < ND; ++k) {
                cr[k] = 0;
                wj[k] = 0.0f;
                if (it_ < p.iters) {
                    cr[k] = __ldg(p.col + (int64_t)i * DEG + k);
                    if (!UNITW) wj[k] = __ldg(p.w + (int64_t)i * DEG + k);
                }
            }
        }
    };
    auto cp16 = [](float4 *dst, const float *src) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
    };
    float4 *slot = si_slots + (size_t)wib * (PIECES * 32) + lane;
    // STAGE: own rows of group it_ and the neighbour rows named by cr -> the warp's slot (each lane copies, and later
    // reads back, only its own 16-byte pieces: no warp synchronisation)
    auto issue_stage = [&](int it_) {
        const int64_t off = blk + (int64_t)it_ * GROUP + lane * 4;
#pragma unroll
        for (int x = 0; x < NQ; ++x) {
            cp16(slot + x * 32, p.h + off + x * 128);
            if (use_m1) cp16(slot + (NQ + x) * 32, p.m1 + off + x * 128);
            if (use_m2) cp16(slot + (2 * NQ + x) * 32, p.m2 + off + x * 128);
        }
#pragma unroll
        for (int k = 0; k < ND; ++k) {
            const float *src = gsrc + si_var_offset<Q, RB>((unsigned)cr[k]);
#pragma unroll
            for (int x = 0; x < NQ; ++x) cp16(slot + ((3 + k) * NQ + x) * 32, src + x * 128);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    if (threadIdx.x < ROW) cta_sum[threadIdx.x] = 0ull;
    int it = warp_gid;
    load_cols(it);
    __syncthreads();
    pdl_wait();  // everything below reads or overwrites what the previous launch wrote
    float wst[ND];  // STAGE: weights of the rows that are in the slot (wj already belongs to the group after)
#pragma unroll
    for (int k = 0; k < ND; ++k) wst[k] = wj[k];
    if (STAGE) {
        if (it < p.iters) issue_stage(it);
        load_cols(it + warps_total);
    }

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

    // not STAGE: own rows travel in registers, requested one iteration ahead
    float4 own[3][NQ];
    auto load_own = [&](int it_) {
        const int64_t off = blk + (int64_t)it_ * GROUP + lane * 4;
#pragma unroll
        for (int x = 0; x < NQ; ++x) {
            own[0][x] = own[1][x] = own[2][x] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (it_ < p.iters) {
                own[0][x] = __ldcs(reinterpret_cast<const float4 *>(p.h + off + x * 128));
                if (use_m1) own[1][x] = __ldcs(reinterpret_cast<const float4 *>(p.m1 + off + x * 128));
                if (use_m2) own[2][x] = __ldcs(reinterpret_cast<const float4 *>(p.m2 + off + x * 128));
            }
        }
    };
    if (!STAGE) load_own(it);

    for (; it < p.iters; it += warps_total) {
        const int64_t off = blk + (int64_t)it * GROUP + lane * 4;
        // ---- coupling contraction f(s) = sum_j W_ij D_j(s) in CSR order
        float f[Q];
#pragma unroll
        for (int s = 0; s < Q; ++s) f[s] = 0.0f;
        auto add = [&](const float4 (&nb)[NQ], float ww) {
#pragma unroll
            for (int x = 0; x < NQ; ++x) {
                if (UNITW) {  // == fma(1, D_j, f)
                    f[4 * x] += nb[x].x; f[4 * x + 1] += nb[x].y; f[4 * x + 2] += nb[x].z; f[4 * x + 3] += nb[x].w;
                } else {
                    f[4 * x] = fma(ww, nb[x].x, f[4 * x]); f[4 * x + 1] = fma(ww, nb[x].y, f[4 * x + 1]);
                    f[4 * x + 2] = fma(ww, nb[x].z, f[4 * x + 2]); f[4 * x + 3] = fma(ww, nb[x].w, f[4 * x + 3]);
                }
            }
        };
        if (STAGE) {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
            for (int k = 0; k < ND; ++k) {
                float4 nb[NQ];
#pragma unroll
                for (int x = 0; x < NQ; ++x) nb[x] = slot[((3 + k) * NQ + x) * 32];
                add(nb, wst[k]);
            }
#pragma unroll
            for (int x = 0; x < NQ; ++x) {
                own[0][x] = slot[x * 32];
                own[1][x] = use_m1 ? slot[(NQ + x) * 32] : make_float4(0.f, 0.f, 0.f, 0.f);
                own[2][x] = use_m2 ? slot[(2 * NQ + x) * 32] : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        } else if (DEG > 0) {
#pragma unroll
            for (int k0 = 0; k0 < DEG; k0 += BATCH) {
                float4 nb[BATCH][NQ];
#pragma unroll
                for (int b = 0; b < BATCH; ++b)
                    if (k0 + b < DEG) {
                        const float *src = gsrc + si_var_offset<Q, RB>((unsigned)cr[k0 + b]);
#pragma unroll
                        for (int x = 0; x < NQ; ++x) nb[b][x] = __ldg(reinterpret_cast<const float4 *>(src + x * 128));
                    }
#pragma unroll
                for (int b = 0; b < BATCH; ++b)
                    if (k0 + b < DEG) add(nb[b], wj[k0 + b]);
            }
        } else {
            const int i = it * G + g;
            const int e0 = __ldg(p.row_ptr + i);
            const int d = __ldg(p.row_ptr + i + 1) - e0;
            int dmax = d;
#pragma unroll
            for (int o = RB; o < 32; o <<= 1) dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
            for (int k0 = 0; k0 < dmax; k0 += 4) {
                unsigned c4[4];
                float w4[4];
                float4 nb[4][NQ];
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const bool on = k0 + b < d;
                    c4[b] = on ? si_var_offset<Q, RB>((unsigned)__ldg(p.col + e0 + k0 + b)) : 0u;
                    w4[b] = on ? (UNITW ? 1.0f : __ldg(p.w + e0 + k0 + b)) : 0.0f;
                }
#pragma unroll
                for (int b = 0; b < 4; ++b)
#pragma unroll
                    for (int x = 0; x < NQ; ++x) {
                        nb[b][x] = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (k0 + b < d) nb[b][x] = __ldg(reinterpret_cast<const float4 *>(gsrc + c4[b] + x * 128));
                    }
#pragma unroll
                for (int b = 0; b < 4; ++b)
                    if (k0 + b < d) add(nb[b], w4[b]);
            }
        }
        // ---- this group's own rows into the working registers
        float h[Q], m1[Q], m2[Q];
#pragma unroll
        for (int x = 0; x < NQ; ++x) {
            h[4 * x] = own[0][x].x; h[4 * x + 1] = own[0][x].y; h[4 * x + 2] = own[0][x].z; h[4 * x + 3] = own[0][x].w;
            m1[4 * x] = own[1][x].x; m1[4 * x + 1] = own[1][x].y; m1[4 * x + 2] = own[1][x].z; m1[4 * x + 3] = own[1][x].w;
            m2[4 * x] = own[2][x].x; m2[4 * x + 1] = own[2][x].y; m2[4 * x + 2] = own[2][x].z; m2[4 * x + 3] = own[2][x].w;
        }
        // ---- next group: its rows travel while this one is computed
        if (STAGE) {
            // the slot is in registers: refill it with the next group's rows (cr holds its columns), then fetch the
            // columns of the group after that
            if (!UNITW) {
#pragma unroll
                for (int k = 0; k < ND; ++k) wst[k] = wj[k];
            }
            if (it + warps_total < p.iters) issue_stage(it + warps_total);
            load_cols(it + 2 * warps_total);
        } else {
            load_cols(it + warps_total);
            load_own(it + warps_total);
        }

        // ---- softmax of h(t) over the states
        float P[Q];
        {
            const float mx = si_tree_max<Q>(h);
            float e[Q];
#pragma unroll
            for (int s = 0; s < Q; ++s) e[s] = fexp(h[s] - mx);
            const float rz = frcp(si_tree_sum<Q>(e));
#pragma unroll
            for (int s = 0; s < Q; ++s) P[s] = e[s] * rz;
        }
        // ---- g^p (S26; with node weights S33-S35: 2 lambda V_i [sum_j V_j P_j - V_i P_i]), g^h = P (g^p - <g^p>_P) (S20), optimiser
        const float Vi = p.vw ? __ldg(p.vw + it * G + g) : 1.0f;  // (V_i = 1: the products are exact, nothing changes)
        {
            float gp[Q], t[Q];
            const float lamV = sc.two_lambda * Vi;
#pragma unroll
            for (int s = 0; s < Q; ++s) gp[s] = fma(h[s], sc.inv_beta, fma(lamV, Ss[s] - Vi * P[s], -f[s]));
#pragma unroll
            for (int s = 0; s < Q; ++s) t[s] = __fmul_rn(P[s], gp[s]);  // (never contracted into the adds)
            const float gbar = si_tree_sum<Q>(t);
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                const float gh = sc.gamma * (P[s] * (gp[s] - gbar));
                h[s] = opt_update(h[s], gh, m1[s], m2[s], sc);
            }
        }
        // ---- centred marginals of the new fields and their column sums (exact fixed point)
        float po[Q];
        {
            const float mx = si_tree_max<Q>(h);
            float e[Q];
#pragma unroll
            for (int s = 0; s < Q; ++s) e[s] = fexp(h[s] - mx);
            const float rz = frcp(si_tree_sum<Q>(e));
#pragma unroll
            for (int s = 0; s < Q; ++s) {
                po[s] = fma(e[s], rz, -inv_q);
                colacc[s] += (long long)Vi * __float2ll_rn(po[s] * fx_scale_t);
            }
        }
#pragma unroll
        for (int x = 0; x < NQ; ++x) {
            __stcs(reinterpret_cast<float4 *>(p.h + off + x * 128), make_float4(h[4 * x], h[4 * x + 1], h[4 * x + 2], h[4 * x + 3]));
            if (use_m1) __stcs(reinterpret_cast<float4 *>(p.m1 + off + x * 128), make_float4(m1[4 * x], m1[4 * x + 1], m1[4 * x + 2], m1[4 * x + 3]));
            if (use_m2) __stcs(reinterpret_cast<float4 *>(p.m2 + off + x * 128), make_float4(m2[4 * x], m2[4 * x + 1], m2[4 * x + 2], m2[4 * x + 3]));
            *reinterpret_cast<float4 *>(p.g_out + off + x * 128) = make_float4(po[4 * x], po[4 * x + 1], po[4 * x + 2], po[4 * x + 3]);
        }
    }

    // column sums: exact integer adds -- variables of the group (shuffles) -> CTA (shared atomics) -> grid (global atomics)
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

// In-place change of layout of one array of a replica block: [variable][state][replica] <-> quad-major groups (header).
// One warp per 32-cell group (32 q floats, the same address range in both layouts): all reads, then all writes.
template <int Q, int RB>
__global__ void __launch_bounds__(256) potts_si_relayout_kernel(float *a0, float *a1, float *a2, float *a3, int64_t blk_stride,
                                                                int groups, int to_si) {
    constexpr int NQ = Q / 4, GROUP = 32 * Q;
    const int lane = threadIdx.x & 31;
    const int grp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (grp >= groups) return;
    float *arr[4] = {a0, a1, a2, a3};
    const int il = lane / RB, r = lane - il * RB;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        if (!arr[a]) continue;
        float *base = arr[a] + (int64_t)blockIdx.y * blk_stride + (int64_t)grp * GROUP;
        float v[Q];
        if (to_si) {
#pragma unroll
            for (int s = 0; s < Q; ++s) v[s] = base[(il * Q + s) * RB + r];
        } else {
#pragma unroll
            for (int x = 0; x < NQ; ++x) {
                const float4 t = *reinterpret_cast<const float4 *>(base + x * 128 + lane * 4);
                v[4 * x] = t.x; v[4 * x + 1] = t.y; v[4 * x + 2] = t.z; v[4 * x + 3] = t.w;
            }
        }
        __syncwarp();
        if (to_si) {
#pragma unroll
            for (int x = 0; x < NQ; ++x)
                *reinterpret_cast<float4 *>(base + x * 128 + lane * 4) = make_float4(v[4 * x], v[4 * x + 1], v[4 * x + 2], v[4 * x + 3]);
        } else {
#pragma unroll
            for (int s = 0; s < Q; ++s) base[(il * Q + s) * RB + r] = v[s];
        }
        __syncwarp();
    }
}

// ---- host side ----
bool potts_si_applicable(const Handle *hd) {
    const int q = hd->dp.q, Rb = hd->Rb;
    if (hd->opt_potts_si == 0 || hd->gather_disc || hd->dp.kind != FEM_BMINCUT) return false;
    if ((q != 4 && q != 8) || (Rb != 4 && Rb != 8 && Rb != 16 && Rb != 32)) return false;
    if (hd->dp.n % (32 / Rb) != 0 || hd->dp.max_deg < 1) return false;
    return hd->dp.nnz < ((int64_t)1 << 31);
}

template <int Q, int RB>
static void relayout_one(Handle *hd, bool to_si) {
    const int groups = (int)((int64_t)hd->dp.n * RB / 32);
    const int nb = hd->R / hd->Rb;
    dim3 grid((unsigned)ceil_div(groups, 8), (unsigned)nb);
    potts_si_relayout_kernel<Q, RB><<<grid, 256, 0, hd->stream>>>(hd->h, hd->m1, hd->m2, hd->g[hd->cur], hd->rows * (int64_t)hd->Rb,
                                                                   groups, to_si ? 1 : 0);
    hd->launches++;
}

// h, m1, m2 and the live gather buffer of every replica block, in place
void launch_potts_si_relayout(Handle *hd, bool to_si) {
    auto go = [&](auto qtag) {
        constexpr int Q = decltype(qtag)::value;
        switch (hd->Rb) {
            case 4: relayout_one<Q, 4>(hd, to_si); break;
            case 8: relayout_one<Q, 8>(hd, to_si); break;
            case 16: relayout_one<Q, 16>(hd, to_si); break;
            default: relayout_one<Q, 32>(hd, to_si); break;
        }
    };
    if (hd->dp.q == 4) go(std::integral_constant<int, 4>{});
    else go(std::integral_constant<int, 8>{});
}

template <int Q, int RB, bool UNITW, int DEG, int BATCH, bool STAGE, int MINB>
static cudaError_t launch_si_deg(Handle *hd, PottsSiParams &p, int blk_count) {
    p.iters = (int)((int64_t)p.n * RB / 32);
    auto kernel = potts_si_kernel<Q, RB, UNITW, DEG, BATCH, STAGE, MINB>;
    const void *fn = reinterpret_cast<const void *>(kernel);
    const size_t smem = STAGE ? (size_t)kSiWarps * (3 + DEG) * (Q / 4) * 32 * sizeof(float4) : 0;
    int &resident = hd->resident_ctas[{fn, smem}];
    if (resident == 0) {
        if (smem > 48 * 1024) {
            const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, kSiWarps * 32, smem) != cudaSuccess || occ < 1) occ = 1;
        resident = occ * hd->sm_count;
    }
    const unsigned gx = (unsigned)std::min<int64_t>(resident, ceil_div(p.iters, kSiWarps));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(gx, (unsigned)blk_count);
    cfg.blockDim = dim3(kSiWarps * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = hd->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (hd->l2_persist_on) {
        // the gather buffer this step WRITES goes to the persisting set-aside (fem_api.cu: l2_persist_begin); it is the one
        // the next step gathers from, and the set-aside holds both, so the gathers hit whatever h, m1, m2 stream through
        attr[1].id = cudaLaunchAttributeAccessPolicyWindow;
        attr[1].val.accessPolicyWindow.base_ptr = (void *)p.g_out;
        attr[1].val.accessPolicyWindow.num_bytes = (size_t)blk_count * (size_t)p.blk_stride * sizeof(float);
        attr[1].val.accessPolicyWindow.hitRatio = 1.0f;
        attr[1].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
        attr[1].val.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, kernel, p);
}

// regular graphs of the common degrees: staged, unrolled instantiation; everything else: rows from row_ptr, direct loads
template <int Q, int RB, bool UNITW>
static cudaError_t launch_si_one(Handle *hd, PottsSiParams &p, int blk_count) {
    switch (p.deg) {
        case 3: return launch_si_deg<Q, RB, UNITW, 3, 3, true, 4>(hd, p, blk_count);
        case 4: return launch_si_deg<Q, RB, UNITW, 4, 4, true, 4>(hd, p, blk_count);
        case 6: return launch_si_deg<Q, RB, UNITW, 6, 6, true, 4>(hd, p, blk_count);
        case 10: return launch_si_deg<Q, RB, UNITW, 10, 5, true, 4>(hd, p, blk_count);
        default: return launch_si_deg<Q, RB, UNITW, 0, 4, false, 4>(hd, p, blk_count);
    }
}

template <int Q>
static cudaError_t launch_si_q(Handle *hd, PottsSiParams &p, int blk_count) {
    const bool unit = p.w == nullptr;
    switch (hd->Rb) {
        case 4: return unit ? launch_si_one<Q, 4, true>(hd, p, blk_count) : launch_si_one<Q, 4, false>(hd, p, blk_count);
        case 8: return unit ? launch_si_one<Q, 8, true>(hd, p, blk_count) : launch_si_one<Q, 8, false>(hd, p, blk_count);
        case 16: return unit ? launch_si_one<Q, 16, true>(hd, p, blk_count) : launch_si_one<Q, 16, false>(hd, p, blk_count);
        default: return unit ? launch_si_one<Q, 32, true>(hd, p, blk_count) : launch_si_one<Q, 32, false>(hd, p, blk_count);
    }
}

// One fp32 exact-gradient Potts step of replica blocks [blk_begin, blk_begin + blk_count) whose arrays are in the
// state-innermost layout (hd->si_live); false = launch failed.
bool launch_potts_si(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count) {
    const int Rb = hd->Rb, q = hd->dp.q;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    PottsSiParams p;
    p.h = hd->h + base;
    p.m1 = hd->m1 + base;
    p.m2 = hd->m2 + base;
    p.g_in = hd->g[hd->cur] + base;
    p.g_out = hd->g[hd->cur ^ 1] + base;
    p.blk_stride = hd->rows * Rb;
    p.col = hd->dp.col;
    p.w = hd->dp.w;
    p.row_ptr = hd->dp.row_ptr;
    p.vw = hd->dp.vw;
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
    const cudaError_t e = q == 4 ? launch_si_q<4>(hd, p, blk_count) : launch_si_q<8>(hd, p, blk_count);
    if (e != cudaSuccess) return false;
    hd->launches++;
    hd->si_launches++;
    return true;
}

}  // namespace fem
