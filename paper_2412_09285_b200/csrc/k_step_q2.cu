// Fused annealing step for the two-state kinds (MaxCut, sparse/dense Ising, Max-SAT).
//
// One thread owns VEC consecutive replicas of one variable and does, in registers, rows a1-a4 of
// the coupling contraction over the variable's CSR row (a coalesced VEC-wide
// gather of m_j = tanh(h_j/2) per neighbour, S30 PAPER.md:671) or the clause leave-one-out products
// (S28 PAPER.md:650, from the same m_j: the literal-false probabilities are (1 -+ m_j)/2), the entropy
// gradient h/beta and chain rule (S29 PAPER.md:667), Adam, and the next step's gathered
// quantity.  No gradient ever reaches HBM.  The step is synchronous (Jacobi): gathers read g_in (from
// h(t)), results go to g_out.  T is both the arithmetic and the storage type: float for the bulk of the
// anneal, double for the wide phase of the first precise_steps steps.
#include "device_math.cuh"

namespace fem {

template <typename T>
struct Q2Params {
    BlockArrays<T> a;
    DevProblem dp;
    Sc<T> sc;
    const T *field;     // dense Ising: precomputed J*m, same layout as h
    T *h_out;           // gather-the-fields mode (GH): the new fields go to the other field array
    const double *rowsum;  // sum_j |W_ij| per node (manipulated gradients), or nullptr
    const signed char *g8_in;  // manipulated gradients: sgn(m) as bytes (device_math.cuh), same offsets as g_in
    signed char *g8_out;
    unsigned rv;        // Rb / VEC lanes per variable
    int rv_shift;       // log2(rv) when rv is a power of two, else -1
    unsigned total;     // n * rv threads per replica block
    unsigned long_blocks;  // the first long_blocks CTAs take one long row each (they start first: the longest work of the launch);
                           // the CTAs after them map one thread to (variable, VEC replicas)
    int long_on;        // rows longer than kLongRow are left to those CTAs (dp.long_rows)
    unsigned long_chunks;  // CTAs per long row: ceil(rv / kLongLanes)
};

constexpr int kLongSlices = 32;  // interleaved slices a long row is cut into (fixed: the summation order depends on the row only)
constexpr int kLongLanes = 32;   // lanes (VEC replicas each) one long-row CTA serves; a wider replica block takes several CTAs per row

enum { MODE_MAXCUT = 0, MODE_ISING = 1, MODE_SAT = 3, MODE_FIELD = 4 };

// Threads per CTA and the register cap (as CTAs per SM) of each instantiation.  Max-SAT fp32 steps use CTAs of 64 threads:
// at R = 128 a warp is one variable's replicas, the time of a CTA is that of its slowest variable, and the finer the CTAs the
// shorter the tail of a launch (cfg 3: 85.9 -> 82.4 us); 16 of them per SM = 64 registers, four resident CTAs' worth of warps
// more than the 68 registers the compiler would take (93.9 -> 85.9 us).  CSR graphs without a uniform degree: 64 registers too
// (skew workload 31.0 -> 28.3 us).  Gather-the-fields: 32 registers, eight CTAs of 256 (six: 193 us against 184 at cfg 4a).
constexpr int kSatThreads = 64;
template <typename T, int MODE, int DEG, bool GH>
struct Q2Block {
    static constexpr bool kSat32 = MODE == MODE_SAT && sizeof(T) == 4;
    static constexpr bool kCsr32 = (MODE == MODE_MAXCUT || MODE == MODE_ISING) && DEG == 0 && !GH && sizeof(T) == 4;
    static constexpr int kTpb = kSat32 ? kSatThreads : kThreads;
    static constexpr int kMinBlocks = GH ? 8 : (kSat32 ? 1024 / kSatThreads : (kCsr32 ? 4 : 1));
};

// GH ("gather the fields", fp32 MaxCut / sparse Ising, regular degree 3 or 4): neighbours are gathered from the FIELD
// array (p.a.g_in == p.a.h) and m_j = tanh(h_j / 2) is recomputed per neighbour with the very function the owner
// would have used, so the results are bit-identical while no gather array is written: 24 B of HBM traffic per field
// and step instead of 28, for DEG more exp / rcp per field (cfg 4a is DRAM-bound: profiles/r02_cfg4a_step.md).
template <typename T, int VEC, int MODE, int DEG, bool GH = false, int KB = 4>
__global__ void __launch_bounds__(Q2Block<T, MODE, DEG, GH>::kTpb, Q2Block<T, MODE, DEG, GH>::kMinBlocks) step_q2_kernel(const Q2Params<T> p) {
    constexpr unsigned TPB = Q2Block<T, MODE, DEG, GH>::kTpb;
    using R = Row<T, VEC>;
    pdl_trigger();
    // Degree-skewed rows (north_star subsystem 2; the paper's scale-free MaxCut instances, and the reason c_i
    // exists).  One thread walking a hub's row alone is the tail of the whole launch, so a row with more
    // than kLongRow entries gets a CTA of its own: the row is cut into kLongSlices interleaved slices (slice s = entries
    // e0 + s, e0 + s + kLongSlices, ... in ascending order), a thread sums one slice for its VEC replicas, the partial
    // sums meet in shared memory and are added in ascending s -- a FIXED order that depends on the row only, so results
    // are deterministic and independent of the replica blocking -- and the first rv threads finish the update like any
    // other thread.  The hub's own row of the gather array is read by all its neighbours and stays in L1 / L2.
    constexpr bool LONG = (MODE == MODE_MAXCUT || MODE == MODE_ISING) && DEG == 0 && !GH;
    bool long_cta = false;
    if constexpr (LONG) long_cta = blockIdx.x < p.long_blocks;
    const unsigned idx = (blockIdx.x - (LONG && !long_cta ? p.long_blocks : 0u)) * TPB + threadIdx.x;
    if (!long_cta && idx >= p.total) return;
    unsigned i = p.rv_shift >= 0 ? idx >> p.rv_shift : idx / p.rv;
    unsigned c = (idx - i * p.rv) * VEC;
    if constexpr (LONG) {  // rows of different lengths: threads take the variables in degree-sorted order (fem_create)
        // (longest rows first: the order is ascending in degree, and the last CTAs of a launch are its tail)
        if (!long_cta && p.dp.order) i = (unsigned)__ldg(p.dp.order + (p.dp.n - 1 - i));
    }
    if constexpr (MODE == MODE_SAT) {  // variables with the most occurrences first (fem_create)
        if (p.dp.order) i = (unsigned)__ldg(p.dp.order + (p.dp.n - 1 - i));
    }
    unsigned lane0 = 0, lanes = 1;  // long-row CTA: the lanes of the replica block it serves
    if constexpr (LONG) {
        if (long_cta) {
            const unsigned L = blockIdx.x;
            i = (unsigned)__ldg(p.dp.long_rows + L / p.long_chunks);
            lane0 = (L % p.long_chunks) * kLongLanes;
            lanes = min((unsigned)kLongLanes, p.rv - lane0);
            c = (lane0 + threadIdx.x % lanes) * VEC;  // (the first `lanes` threads finish the row; the others only sum slices)
        }
    }
    const int64_t blk = (int64_t)blockIdx.y * p.a.blk_stride;
    const unsigned Rb = p.a.Rb;
    const int64_t off = blk + (i * Rb + c);  // a replica block holds < 2^32 elements (checked at fem_anneal)
    const T *__restrict__ gin = p.a.g_in + blk + c;
    const signed char *__restrict__ gin8 = p.g8_in + blk + c;
    const bool disc = p.sc.disc != 0;  // uniform; only ever set for the sparse graph kinds
    // one neighbour row: VEC floats (exact gradient) or VEC bytes holding sgn(m_j) (manipulated gradients)
    // row j of the gather array: one IMAD.WIDE (32 x 32 -> 64-bit product added to the base) instead of a 32-bit
    // multiply plus a two-instruction 64-bit scale-and-add
    const unsigned row_bytes = Rb * (unsigned)sizeof(T);
    auto row_of = [&](unsigned j) -> const T * {
        return reinterpret_cast<const T *>(reinterpret_cast<const char *>(gin) + (unsigned long long)j * row_bytes);
    };
    auto gather = [&](unsigned j) -> R {
        if ((MODE == MODE_MAXCUT || MODE == MODE_ISING) && disc) {
            int b[VEC];
            ld_bytes<VEC>(gin8 + j * Rb, b);
            R r;
#pragma unroll
            for (int v = 0; v < VEC; ++v) r.v[v] = (T)b[v];
            return r;
        }
        R r = R::ld(row_of(j));
        if (GH) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) r.v[v] = mag_of(r.v[v]);
        }
        return r;
    };

    // static structure first (legal before pdl_wait), then everything the previous step wrote
    int jj[DEG > 0 ? DEG : 1];
    float wj[DEG > 0 ? DEG : 1];
    if ((MODE == MODE_MAXCUT || MODE == MODE_ISING) && DEG > 0) {
#pragma unroll
        for (int k = 0; k < DEG; ++k) {
            jj[k] = __ldg(p.dp.col + i * DEG + k);
            wj[k] = p.dp.w ? __ldg(p.dp.w + i * DEG + k) : 1.0f;
        }
    }
    pdl_wait();
    const Sc<T> &sc = p.sc;
    const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();  // uniform: SGD keeps no second moment (8 B per field less)
    // (GH: the own row is one of the rows the neighbours gather -- keep it in L2 like them)
    const R h4 = GH ? R::ld(p.a.h + off) : R::ld_stream(p.a.h + off);
    R m1 = {}, m2 = {};
    if (use_m1) m1 = R::ld_stream(p.a.m1 + off);
    if (use_m2) m2 = R::ld_stream(p.a.m2 + off);

    T dU[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) dU[v] = (T)0;

    if (MODE == MODE_MAXCUT || MODE == MODE_ISING) {
        const int *__restrict__ col = p.dp.col;
        const float *__restrict__ w = p.dp.w;
        if (DEG > 0) {
            R nb[DEG > 0 ? DEG : 1];
#pragma unroll
            for (int k = 0; k < DEG; ++k) nb[k] = gather((unsigned)jj[k]);
#pragma unroll
            for (int k = 0; k < DEG; ++k)
#pragma unroll
                for (int v = 0; v < VEC; ++v) dU[v] = fma((T)wj[k], nb[k].v[v], dU[v]);
        } else {
            const int e0 = __ldg(p.dp.row_ptr + i), e1 = __ldg(p.dp.row_ptr + i + 1);
            if constexpr (LONG) {
                if (!long_cta && p.long_on && is_long_row(e1 - e0, p.dp.nnz, p.dp.n)) return;  // a CTA of its own does this row
            }
            if (LONG && long_cta) {
                if constexpr (LONG) {
                    __shared__ T red[kLongSlices * kLongLanes * VEC];
                    const unsigned units = kLongSlices * lanes;  // (slice, lane) pairs; at most 4 per thread
                    for (unsigned u = threadIdx.x; u < units; u += kThreads) {
                        const unsigned sl = u / lanes, cl = u - sl * lanes;
                        const T *__restrict__ gsl = p.a.g_in + blk + (lane0 + cl) * VEC;
                        const signed char *__restrict__ gsl8 = p.g8_in + blk + (lane0 + cl) * VEC;
                        T part[VEC];
#pragma unroll
                        for (int v = 0; v < VEC; ++v) part[v] = (T)0;
                        // batches of 4 entries of the slice, all loads of a batch in flight (entries past the end: the
                        // slice's first entry again with weight 0), added in ascending order
                        for (int e = e0 + (int)sl; e < e1; e += 4 * kLongSlices) {
                            unsigned jb[4];
                            float wb[4];
                            R nb[4];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const bool on = e + k * kLongSlices < e1;
                                const int ee = on ? e + k * kLongSlices : e;
                                jb[k] = (unsigned)__ldg(col + ee);
                                wb[k] = on ? (w ? __ldg(w + ee) : 1.0f) : 0.0f;
                            }
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                if (disc) {
                                    int b[VEC];
                                    ld_bytes<VEC>(gsl8 + jb[k] * Rb, b);
#pragma unroll
                                    for (int v = 0; v < VEC; ++v) nb[k].v[v] = (T)b[v];
                                } else {
                                    nb[k] = R::ld(reinterpret_cast<const T *>(reinterpret_cast<const char *>(gsl) + (unsigned long long)jb[k] * row_bytes));
                                }
                            }
#pragma unroll
                            for (int k = 0; k < 4; ++k)
#pragma unroll
                                for (int v = 0; v < VEC; ++v) part[v] = fma((T)wb[k], nb[k].v[v], part[v]);
                        }
#pragma unroll
                        for (int v = 0; v < VEC; ++v) red[u * VEC + v] = part[v];
                    }
                    __syncthreads();
                    if (threadIdx.x >= lanes) return;
                    for (unsigned s2 = 0; s2 < kLongSlices; ++s2)
#pragma unroll
                        for (int v = 0; v < VEC; ++v) dU[v] += red[(s2 * lanes + threadIdx.x) * VEC + v];
                }
            } else {
                // batches of kB entries: the column indices of a batch, then its neighbour rows, all in flight at once (a
                // remainder loop would pay two dependent round trips per entry).  No branches inside a batch: entries past
                // the end of the row re-read the row's last entry with weight 0 (fma(0, m, dU) = dU); added in CSR order
                auto batched = [&](auto tag) {
                    constexpr int kB = decltype(tag)::value;
                    for (int e = e0; e < e1; e += kB) {
                        unsigned jb[kB];
                        float wb[kB];
                        R nb[kB];
#pragma unroll
                        for (int k = 0; k < kB; ++k) {
                            const int ee = min(e + k, e1 - 1);
                            jb[k] = (unsigned)__ldg(col + ee);
                            wb[k] = e + k < e1 ? (w ? __ldg(w + ee) : 1.0f) : 0.0f;
                        }
#pragma unroll
                        for (int k = 0; k < kB; ++k) nb[k] = gather(jb[k]);
#pragma unroll
                        for (int k = 0; k < kB; ++k)
#pragma unroll
                            for (int v = 0; v < VEC; ++v) dU[v] = fma((T)wb[k], nb[k].v[v], dU[v]);
                    }
                };
                // batch size KB by the mean degree (chosen at launch): 4 where most rows are short (measured on the scale-free
                // workload: 19.3 us per launch against 21.6 with a remainder loop and 25+ with batches of 8), 8 for denser
                // graphs (cfg 0 stepwise: 7.5 us against 9.4 with batches of 4)
                batched(std::integral_constant<int, KB>{});
            }
        }
        if (MODE == MODE_ISING) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) dU[v] = (T)-2 * dU[v];  // dU/dp = 2 dU/dm = -2 sum_j J_ij m_j
        }
    } else if (MODE == MODE_FIELD) {
        const R f = R::ld_stream(p.field + off);
#pragma unroll
        for (int v = 0; v < VEC; ++v) dU[v] = (T)-2 * f.v[v];
    } else {  // MODE_SAT: dU/dp_i = sum_{m ni i} s_mi prod_{k != i} u_mk; DEG = entries per occurrence (k_max - 1)
        constexpr int KS = DEG > 0 ? DEG : 1;
        constexpr int B = KS == 1 ? 8 : (KS == 2 ? 4 : 2);  // occurrences in flight per thread (measured at KS = 3: 2 -> 86 us, 3 -> 87, 4 -> 98, 6 -> 93 on cfg 3)
        const int o0 = __ldg(p.dp.occ_ptr + i), o1 = __ldg(p.dp.occ_ptr + i + 1);
        const unsigned pad = ((unsigned)p.dp.n << 1) | 1u;  // the constant-1 row, "negated": factor 0.5 + 0.5*1 = 1
        for (int o = o0; o < o1; o += B) {
            // one occurrence = KST entries (KS padded to a power of two): one aligned 4-, 8- or 16-byte load
            constexpr int KST = KS <= 1 ? 1 : (KS <= 2 ? 2 : (KS <= 4 ? 4 : 8));
            unsigned pk[B][KST];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int *__restrict__ ent = p.dp.occ + (unsigned)(o + b) * (unsigned)KST;
                if (o + b < o1) {
                    if constexpr (KST == 1) {
                        pk[b][0] = (unsigned)__ldg(ent);
                    } else if constexpr (KST == 2) {
                        const int2 t = __ldg(reinterpret_cast<const int2 *>(ent));
                        pk[b][0] = (unsigned)t.x; pk[b][1] = (unsigned)t.y;
                    } else {
#pragma unroll
                        for (int x4 = 0; x4 < KST / 4; ++x4) {
                            const int4 t = __ldg(reinterpret_cast<const int4 *>(ent) + x4);
                            pk[b][4 * x4] = (unsigned)t.x; pk[b][4 * x4 + 1] = (unsigned)t.y;
                            pk[b][4 * x4 + 2] = (unsigned)t.z; pk[b][4 * x4 + 3] = (unsigned)t.w;
                        }
                    }
                } else {
#pragma unroll
                    for (int x = 0; x < KST; ++x) pk[b][x] = pad;
                }
            }
            R mr[B][KS];
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int x = 0; x < KS; ++x) mr[b][x] = R::ld(row_of((pk[b][x] & 0x7fffffffu) >> 1));
#pragma unroll
            for (int b = 0; b < B; ++b) {
                T prod[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) prod[v] = (T)1;
#pragma unroll
                for (int x = 0; x < KS; ++x) {
                    // probability the literal is false: 1-p = (1-m)/2 (positive literal), p = (1+m)/2 (negated)
                    const T sg = (pk[b][x] & 1u) ? (T)0.5 : (T)-0.5;
#pragma unroll
                    for (int v = 0; v < VEC; ++v) prod[v] *= fma(sg, mr[b][x].v[v], (T)0.5);  // as in persist_q2_kernel
                }
                const bool positive = (pk[b][0] >> 31) != 0u;  // bit 31 of entry 0: own literal is positive
                if (o + b < o1) {
#pragma unroll
                    for (int v = 0; v < VEC; ++v) dU[v] += positive ? -prod[v] : prod[v];
                }
            }
        }
    }

    // manipulated gradients (S29/S30): the gathered values are sgn(m_j) and the coupling term is
    // normalised by c_i = 1 / sum_j |W_ij| (Ising: |2 J_ij|; nodes without neighbours: 0); all kinds: times gamma_grad
    T ci = (T)1;
    if (sc.disc) {  // only set for the sparse graph kinds (fem_anneal)
        const double rs = __ldg(p.rowsum + i) * (MODE == MODE_ISING ? 2.0 : 1.0);
        ci = rs > 0.0 ? (T)(1.0 / rs) : (T)0;
    }
    R hn, gn;
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
        const T h = h4.v[v];
        const T g = q2_grad(dU[v], ci, h, sc);  // S29 with ln(p/(1-p)) = h
        hn.v[v] = opt_update(h, g, m1.v[v], m2.v[v], sc);
        gn.v[v] = disc ? sign_of(hn.v[v]) : mag_of(hn.v[v]);
    }
    if (GH) hn.st(p.h_out + off);
    else hn.st_stream(p.a.h + off);
    if (use_m1) m1.st_stream(p.a.m1 + off);
    if (use_m2) m2.st_stream(p.a.m2 + off);
    if (GH) return;
    if (disc) {
        int b[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) b[v] = (int)gn.v[v];
        st_bytes<VEC>(p.g8_out + off, b);
    } else {
        gn.st(p.a.g_out + off);
    }
}

// Gathered quantity m = tanh(h/2) from the fields (used at t = 0 and after fem_set_fields); also writes
// the constant-1 row that pads short clauses, in both gather buffers.
template <typename T>
__global__ void __launch_bounds__(kThreads) q2_prepare_kernel(const T *h, T *g, T *g_other, int64_t blk_stride, int Rb,
                                                              int n, int nblocks, int disc, signed char *g8) {
    const int64_t per = (int64_t)n * Rb;
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx >= per * nblocks) return;
    const int64_t b = idx / per, r = idx - b * per;
    const int64_t off = b * blk_stride + r;
    if (disc) {
        g8[off] = (signed char)(int)sign_of(h[off]);
        return;
    }
    g[off] = (T)mag_of((double)h[off]);
    if (r < Rb) {
        g[b * blk_stride + per + r] = (T)1;
        g_other[b * blk_stride + per + r] = (T)1;
    }
}

// ---- dense Ising: field = J * m on CUDA cores (placeholder GEMM; the tcgen05 path replaces it) ----
// C[n x Rb] = J[n x n] * M[n x Rb], all row-major.  64x64 tile, 16x16 threads, 4x4 micro-tile.
template <typename T>
__global__ void __launch_bounds__(256) dense_field_kernel(const float *__restrict__ J, const T *__restrict__ M,
                                                          T *__restrict__ C, int n, int Rb) {
    __shared__ T As[16][64 + 1];
    __shared__ T Bs[16][64];
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    const int row0 = blockIdx.y * 64, col0 = blockIdx.x * 64;
    T acc[4][4] = {};
    for (int k0 = 0; k0 < n; k0 += 16) {
        for (int t = threadIdx.x; t < 64 * 16; t += 256) {
            const int r = t / 16, k = t % 16;
            const int gr = row0 + r, gk = k0 + k;
            As[k][r] = (gr < n && gk < n) ? (T)J[(int64_t)gr * n + gk] : (T)0;
        }
        for (int t = threadIdx.x; t < 16 * 64; t += 256) {
            const int k = t / 64, cc = t % 64;
            const int gk = k0 + k, gc = col0 + cc;
            Bs[k][cc] = (gk < n && gc < Rb) ? M[(int64_t)gk * Rb + gc] : (T)0;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            T a[4], b[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) a[x] = As[k][ty * 4 + x];
#pragma unroll
            for (int x = 0; x < 4; ++x) b[x] = Bs[k][tx * 4 + x];
#pragma unroll
            for (int x = 0; x < 4; ++x)
#pragma unroll
                for (int y = 0; y < 4; ++y) acc[x][y] += a[x] * b[y];
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < 4; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            const int gr = row0 + ty * 4 + x, gc = col0 + tx * 4 + y;
            if (gr < n && gc < Rb) C[(int64_t)gr * Rb + gc] = acc[x][y];
        }
}

// The same product for the fp64 wide phase and the CUDA-core fallback, as a register-tiled GEMM: 128 x 128 tile per
// CTA, k step 8, 16 x 16 threads with an 8 x 8 micro-tile each (64 accumulators), J converted on load.  The generic
// 64 x 64 / 4 x 4 kernel above reached 8.5 TFLOP/s in fp64 on cfg 4b (4 ms per wide step, 12% of the whole pass).
// Sums run over k in ascending order per output, as in dense_field_kernel (the order inside a k step is the same).
template <typename T>
__global__ void __launch_bounds__(256) dense_field_big_kernel(const float *__restrict__ J, const T *__restrict__ M,
                                                              T *__restrict__ C, int n, int Rb) {
    constexpr int BM = 128, BN = 128, BK = 8;
    __shared__ __align__(16) T As[BK][BM];
    __shared__ __align__(16) T Bs[BK][BN];
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    const int row0 = blockIdx.y * BM, col0 = blockIdx.x * BN;
    T acc[8][8];
#pragma unroll
    for (int x = 0; x < 8; ++x)
#pragma unroll
        for (int y = 0; y < 8; ++y) acc[x][y] = (T)0;
    const int ar = threadIdx.x / 2, ak = (threadIdx.x % 2) * 4;   // A tile: row ar, k = ak .. ak+3
    const int bk = threadIdx.x / 32, bc = (threadIdx.x % 32) * 4;  // B tile: row bk, columns bc .. bc+3
    for (int k0 = 0; k0 < n; k0 += BK) {
#pragma unroll
        for (int z = 0; z < 4; ++z) {
            const int gr = row0 + ar, gk = k0 + ak + z;
            As[ak + z][ar] = (gr < n && gk < n) ? (T)J[(int64_t)gr * n + gk] : (T)0;
            const int gkb = k0 + bk, gc = col0 + bc + z;
            Bs[bk][bc + z] = (gkb < n && gc < Rb) ? M[(int64_t)gkb * Rb + gc] : (T)0;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            T a[8], b[8];
#pragma unroll
            for (int x = 0; x < 8; ++x) a[x] = As[k][ty * 8 + x];
#pragma unroll
            for (int y = 0; y < 8; ++y) b[y] = Bs[k][tx * 8 + y];
#pragma unroll
            for (int x = 0; x < 8; ++x)
#pragma unroll
                for (int y = 0; y < 8; ++y) acc[x][y] = fma(a[x], b[y], acc[x][y]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < 8; ++x)
#pragma unroll
        for (int y = 0; y < 8; ++y) {
            const int gr = row0 + ty * 8 + x, gc = col0 + tx * 8 + y;
            if (gr < n && gc < Rb) C[(int64_t)gr * Rb + gc] = acc[x][y];
        }
}

// fp64 on the tensor cores: the vector FP64 pipe of this part tops out near 9 TFLOP/s (both CUDA-core kernels above
// run the cfg 4b wide step in 3.9 ms), the DMMA path (mma.sync m8n8k4 f64) is the one rated ~37 TFLOP/s.
// CTA tile 64 x 64, k step 16, 8 warps as 4 x 2, each warp 16 x 32 = 2 x 4 mma tiles; fragments straight from padded
// shared memory (conflict-free per half-warp).  Used for the fp64 wide phase of dense couplings.
__device__ __forceinline__ void dmma_8x8x4(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) dense_field_dmma_kernel(const float *__restrict__ J, const double *__restrict__ M,
                                                               double *__restrict__ C, int n, int Rb) {
    constexpr int BM = 64, BN = 64, BK = 16;
    __shared__ double As[BM][BK + 4];
    __shared__ double Bs[BK][BN + 4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wm = (warp >> 1) * 16, wn = (warp & 1) * 32;
    const int row0 = blockIdx.y * BM, col0 = blockIdx.x * BN;
    double acc[2][4][2];
#pragma unroll
    for (int x = 0; x < 2; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y) acc[x][y][0] = acc[x][y][1] = 0.0;
    const int ar = threadIdx.x / 4, ak = (threadIdx.x % 4) * 4;    // A tile: row ar, k = ak .. ak+3
    const int bk = threadIdx.x / 16, bc = (threadIdx.x % 16) * 4;  // B tile: row bk, columns bc .. bc+3
    for (int k0 = 0; k0 < n; k0 += BK) {
#pragma unroll
        for (int z = 0; z < 4; ++z) {
            const int gr = row0 + ar, gk = k0 + ak + z;
            As[ar][ak + z] = (gr < n && gk < n) ? (double)J[(int64_t)gr * n + gk] : 0.0;
            const int gkb = k0 + bk, gc = col0 + bc + z;
            Bs[bk][bc + z] = (gkb < n && gc < Rb) ? M[(int64_t)gkb * Rb + gc] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[2], b[4];
#pragma unroll
            for (int x = 0; x < 2; ++x) a[x] = As[wm + x * 8 + (lane >> 2)][kk + (lane & 3)];
#pragma unroll
            for (int y = 0; y < 4; ++y) b[y] = Bs[kk + (lane & 3)][wn + y * 8 + (lane >> 2)];
#pragma unroll
            for (int x = 0; x < 2; ++x)
#pragma unroll
                for (int y = 0; y < 4; ++y) dmma_8x8x4(acc[x][y][0], acc[x][y][1], a[x], b[y]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < 2; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            const int gr = row0 + wm + x * 8 + (lane >> 2), gc = col0 + wn + y * 8 + 2 * (lane & 3);
            if (gr < n) {
                if (gc < Rb) C[(int64_t)gr * Rb + gc] = acc[x][y][0];
                if (gc + 1 < Rb) C[(int64_t)gr * Rb + gc + 1] = acc[x][y][1];
            }
        }
}

template <typename T>
static void launch_dense_field(Handle *hd, const T *M, T *C, int n, int Rb) {
    if (n >= 256 && Rb >= 64) {
        if constexpr (std::is_same<T, double>::value) {
            dim3 gb((unsigned)ceil_div(Rb, 64), (unsigned)ceil_div(n, 64));
            dense_field_dmma_kernel<<<gb, 256, 0, hd->stream>>>(hd->dp.J, M, C, n, Rb);
        } else {
            dim3 gb((unsigned)ceil_div(Rb, 128), (unsigned)ceil_div(n, 128));
            dense_field_big_kernel<T><<<gb, 256, 0, hd->stream>>>(hd->dp.J, M, C, n, Rb);
        }
    } else {
        dim3 g((unsigned)ceil_div(Rb, 64), (unsigned)ceil_div(n, 64));
        dense_field_kernel<T><<<g, 256, 0, hd->stream>>>(hd->dp.J, M, C, n, Rb);
    }
}

// C = J * M in fp64 for the dense readout (k_readout.cu): the DMMA kernel where the shape allows
void launch_dense_field_f64(Handle *hd, const double *M, double *C, int n, int R) { launch_dense_field<double>(hd, M, C, n, R); }

template <typename T, int VEC, int MODE>
static void launch_q2_deg(Handle *hd, const Q2Params<T> &p, dim3 grid) {
    if constexpr (MODE == MODE_SAT) {
        switch (hd->dp.kstride) {
            case 1: launch_pdl(step_q2_kernel<T, VEC, MODE, 1>, grid, dim3(Q2Block<T, MODE, 1, false>::kTpb), hd->stream, p); break;
            case 2: launch_pdl(step_q2_kernel<T, VEC, MODE, 2>, grid, dim3(Q2Block<T, MODE, 2, false>::kTpb), hd->stream, p); break;
            case 3: launch_pdl(step_q2_kernel<T, VEC, MODE, 3>, grid, dim3(Q2Block<T, MODE, 3, false>::kTpb), hd->stream, p); break;
            case 4: launch_pdl(step_q2_kernel<T, VEC, MODE, 4>, grid, dim3(Q2Block<T, MODE, 4, false>::kTpb), hd->stream, p); break;
            case 5: launch_pdl(step_q2_kernel<T, VEC, MODE, 5>, grid, dim3(Q2Block<T, MODE, 5, false>::kTpb), hd->stream, p); break;
            case 6: launch_pdl(step_q2_kernel<T, VEC, MODE, 6>, grid, dim3(Q2Block<T, MODE, 6, false>::kTpb), hd->stream, p); break;
            default: launch_pdl(step_q2_kernel<T, VEC, MODE, 7>, grid, dim3(Q2Block<T, MODE, 7, false>::kTpb), hd->stream, p); break;
        }
    } else {
        const int d = (MODE == MODE_MAXCUT || MODE == MODE_ISING) ? hd->dp.uniform_deg : 0;
        if constexpr (std::is_same<T, float>::value && VEC == 4 && (MODE == MODE_MAXCUT || MODE == MODE_ISING)) {
            if (hd->gather_h && p.h_out) {
                if (d == 3) launch_pdl(step_q2_kernel<T, VEC, MODE, 3, true>, grid, dim3(kThreads), hd->stream, p);
                else launch_pdl(step_q2_kernel<T, VEC, MODE, 4, true>, grid, dim3(kThreads), hd->stream, p);
                return;
            }
        }
        if (d == 3)
            launch_pdl(step_q2_kernel<T, VEC, MODE, 3>, grid, dim3(kThreads), hd->stream, p);
        else if (d == 4)
            launch_pdl(step_q2_kernel<T, VEC, MODE, 4>, grid, dim3(kThreads), hd->stream, p);
        else if (std::is_same<T, float>::value && (MODE == MODE_MAXCUT || MODE == MODE_ISING) && hd->dp.nnz > 8 * (int64_t)hd->dp.n)
            launch_pdl(step_q2_kernel<T, VEC, MODE, 0, false, 8>, grid, dim3(kThreads), hd->stream, p);
        else
            launch_pdl(step_q2_kernel<T, VEC, MODE, 0>, grid, dim3(kThreads), hd->stream, p);
    }
}

template <typename T, int VEC>
static void launch_q2_mode(Handle *hd, const Q2Params<T> &p, dim3 grid, int mode) {
    switch (mode) {
        case MODE_MAXCUT: launch_q2_deg<T, VEC, MODE_MAXCUT>(hd, p, grid); break;
        case MODE_ISING: launch_q2_deg<T, VEC, MODE_ISING>(hd, p, grid); break;
        case MODE_SAT: launch_q2_deg<T, VEC, MODE_SAT>(hd, p, grid); break;
        default: launch_q2_deg<T, VEC, MODE_FIELD>(hd, p, grid); break;
    }
}

bool launch_step_dense_tc(Handle *hd, const StepScalars &sc);  // k_dense_tc.cu
bool launch_step_dense_i8(Handle *hd, const StepScalars &sc);  // k_dense_i8.cu
void launch_prepare_q2(Handle *hd, bool wide);

template <typename T>
static void launch_step_q2_t(Handle *hd, const StepScalars &sc, int blk_begin, int blk_count) {
    using S = StateOf<T>;
    if (std::is_same<T, float>::value && hd->dp.kind == FEM_ISING && hd->dp.J && blk_begin == 0 && blk_count == 1 && hd->plain_adam) {
        // dense couplings: tcgen05 GEMM with the update fused in its epilogue -- the int8 digit path (k_dense_i8.cu) where it
        // applies, else 3xTF32 (k_dense_tc.cu).  A trajectory stays on the path its first tensor-core step took.
        if (!hd->tc_ready && launch_step_dense_i8(hd, sc)) return;
        if (!hd->tc8_ready && launch_step_dense_tc(hd, sc)) return;
    }
    if (std::is_same<T, float>::value && hd->tc8_ready) {  // the fp32 gather array was not maintained by the int8 steps
        hd->tc8_ready = false;
        launch_prepare_q2(hd, false);
    }
    if (std::is_same<T, float>::value && hd->tc_ready) {
        // a tensor-core step (or its preparation) left g[cur] in the TRANSPOSED layout GT[a][i]; this path reads
        // g[cur] as [i][Rb].  Rebuild it from the fields before gathering from it.
        hd->tc_ready = false;
        launch_prepare_q2(hd, false);
    }
    const int Rb = hd->Rb;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    Q2Params<T> p;
    p.a.h = S::h(hd) + base;
    p.a.m1 = S::m1(hd) + base;
    p.a.m2 = S::m2(hd) + base;
    p.a.g_in = S::g(hd, hd->cur) + base;
    p.a.g_out = S::g(hd, hd->cur ^ 1) + base;
    p.a.blk_stride = hd->rows * Rb;
    p.a.Rb = Rb;
    p.dp = hd->dp;
    p.sc = Sc<T>(sc);
    p.field = nullptr;
    p.h_out = nullptr;
    if (std::is_same<T, float>::value && hd->gather_h) {  // fields ping-pong between h and g[0]; gathers read the input fields
        p.a.g_in = reinterpret_cast<const T *>(hd->fields()) + base;
        p.h_out = reinterpret_cast<T *>(hd->fields_other()) + base;
    }
    p.rowsum = hd->rowsum;
    p.g8_in = reinterpret_cast<const signed char *>(hd->g[hd->cur]) + base;   // byte offsets = element offsets
    p.g8_out = reinterpret_cast<signed char *>(hd->g[hd->cur ^ 1]) + base;
    int mode = hd->dp.kind == FEM_MAXCUT ? MODE_MAXCUT : hd->dp.kind == FEM_MAXSAT ? MODE_SAT : MODE_ISING;
    if (hd->dp.kind == FEM_ISING && hd->dp.J) {
        mode = MODE_FIELD;
        p.field = S::field(hd) + base;
        const int n = hd->dp.n;
        dim3 g((unsigned)ceil_div(Rb, 64), (unsigned)ceil_div(n, 64));
        for (int b = 0; b < blk_count; ++b) {
            const int64_t o = (int64_t)b * p.a.blk_stride;
            launch_dense_field<T>(hd, p.a.g_in + o, S::field(hd) + base + o, n, Rb);
            hd->launches++;
        }
    }
    const int VEC = (Rb % 4 == 0) ? 4 : 1;
    p.rv = (unsigned)(Rb / VEC);
    p.rv_shift = (p.rv & (p.rv - 1)) == 0 ? __builtin_ctz(p.rv) : -1;
    p.total = (unsigned)hd->dp.n * p.rv;
    const unsigned main_blocks = (unsigned)ceil_div(p.total, mode == MODE_SAT ? Q2Block<T, MODE_SAT, 1, false>::kTpb : kThreads);
    // long rows (CSR kinds without a uniform degree): one extra CTA each, when a row's lanes fit a CTA
    p.long_on = (mode == MODE_MAXCUT || mode == MODE_ISING) && hd->opt_long_rows && hd->dp.n_long > 0 && hd->dp.uniform_deg == 0;
    p.long_chunks = (unsigned)ceil_div(p.rv, kLongLanes);
    p.long_blocks = p.long_on ? (unsigned)hd->dp.n_long * p.long_chunks : 0u;
    dim3 grid(main_blocks + p.long_blocks, (unsigned)blk_count);
    if (VEC == 4) launch_q2_mode<T, 4>(hd, p, grid, mode);
    else launch_q2_mode<T, 1>(hd, p, grid, mode);
    hd->launches++;
}

void launch_step_q2(Handle *hd, const StepScalars &sc, bool wide, int blk_begin, int blk_count) {
    if (wide) launch_step_q2_t<double>(hd, sc, blk_begin, blk_count);
    else launch_step_q2_t<float>(hd, sc, blk_begin, blk_count);
}

void launch_prepare_q2(Handle *hd, bool wide) {
    const int nb = hd->R / hd->Rb;
    const int64_t total = (int64_t)hd->dp.n * hd->Rb * nb;
    const unsigned grid = (unsigned)ceil_div(total, kThreads);
    if (wide)
        q2_prepare_kernel<double><<<grid, kThreads, 0, hd->stream>>>(hd->hW, hd->gW[hd->cur], hd->gW[hd->cur ^ 1],
                                                                     hd->rows * hd->Rb, hd->Rb, hd->dp.n, nb, hd->gather_disc ? 1 : 0,
                                                                     reinterpret_cast<signed char *>(hd->g[hd->cur]));
    else
        q2_prepare_kernel<float><<<grid, kThreads, 0, hd->stream>>>(hd->h, hd->g[hd->cur], hd->g[hd->cur ^ 1],
                                                                    hd->rows * hd->Rb, hd->Rb, hd->dp.n, nb, hd->gather_disc ? 1 : 0,
                                                                     reinterpret_cast<signed char *>(hd->g[hd->cur]));
    hd->launches++;
}

}  // namespace fem
