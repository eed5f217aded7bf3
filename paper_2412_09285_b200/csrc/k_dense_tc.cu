// Dense-coupling Ising step on the 5th-generation tensor cores (cfg 4b: SK, n = 4096, R = 1024).
//
// J*M really is a dense GEMM here (north_star subsystem 5):  F[i][a] = sum_j J_ij m_j^a, 2 n^2 R flop per step.
// One CTA computes a 128 x BN tile of F with tcgen05.mma (kind::tf32, fp32 accumulation in TMEM), fed by TMA
// (cp.async.bulk.tensor, 128-byte swizzle) through an mbarrier ring, and applies the whole FEM update
// (S29 PAPER.md:667 + Adam PAPER.md:88) in the epilogue straight out of TMEM -- the field never reaches HBM.
//
// Accuracy: plain TF32 (10-bit mantissa) would put ~5e-4 absolute error on the local field, which fails the
// marginal tolerance.  3xTF32 split: x = hi + lo with hi = the top 19 bits (what the tensor core reads from a
// 32-bit container) and lo = x - hi (exact in fp32); F ~= Jhi*Mhi + Jhi*Mlo + Jlo*Mhi, three MMAs per k-step,
// error ~2^-21 relative per product.  J_lo is made once at fem_create; M_lo is made by the previous step's epilogue.
//
// Operands are K-major: A = J[i][j] (row-major as given), B = GT[a][j], the gathered magnetisations stored
// TRANSPOSED for this kind (the epilogue's lanes are rows i, so for a fixed replica a the 32 lanes of a warp
// write 32 consecutive GT[a][i] -- coalesced).
//
// Warp roles (192 threads): warp 0 = TMA producer (one elected lane), warp 1 = TMEM allocator + MMA issuer
// (one elected lane), warps 2..5 = epilogue (warp w reads TMEM lanes 32*(w%4) .. +31).
#include <cuda.h>

#include "device_math.cuh"

namespace fem {

constexpr int TC_BM = 128;      // rows of F (variables i) per CTA = TMEM lanes
constexpr int TC_BK = 32;       // floats per k-block = one 128-byte swizzle atom
constexpr int TC_UMMA_K = 8;    // tf32 elements per tcgen05.mma
constexpr int TC_THREADS = 192;

// The tensor core adds each MMA's result into the fp32 accumulator with truncation, so a long accumulation
// chain carries a bias towards zero that grows with the number of adds and the size of the running sum
// (measured: one 1536-add chain per output leaves 1.6e-4 on the marginals at step 50 of cfg 4b).  The k range
// is therefore cut into chunks that accumulate in SEPARATE TMEM accumulators, and the two small 3xTF32 terms
// get an accumulator of their own; the epilogue adds the kAcc partial sums in fp32, round to nearest.
template <int BN>
struct TcShape {
    static constexpr int kStageBytes = 2 * TC_BM * 128 + 2 * BN * 128;  // A_hi, A_lo, B_hi, B_lo
    static constexpr int kStages = BN >= 256 ? 2 : (BN >= 128 ? 3 : 4);
    static constexpr int kSmem = kStages * kStageBytes + 1024;  // + alignment slack
    static constexpr int kAcc = 512 / BN > 8 ? 8 : 512 / BN;    // accumulators: [0] small terms, [1..] chunks of k
    static constexpr int kTmemCols = kAcc * BN;                 // 256 or 512 columns (a power of two >= 32)
};

struct TcParams {
    float *h, *m1, *m2;       // [i][a], row pitch Rb
    float *gt_out, *gtlo_out;  // [a][i], row pitch n
    Sc<float> sc;
    int n, Rb;
};

// ---- PTX wrappers -------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *smem_dst, const CUtensorMap *tm, int c0, int c1, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_u32(smem_dst)),
        "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
// K-major operand tile, 128-byte swizzle: rows of 128 B, 8-row groups 1024 B apart (SBO), descriptor version 1.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFF) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) |
           (2ull << 61);
}
// kind::tf32, fp32 accumulator, both operands K-major, M = 128
__host__ __device__ constexpr uint32_t umma_idesc_tf32(int M, int N) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float *v) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(r[k]);
}

__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }

// ---- the fused step ----------------------------------------------------------------------------------
template <int BN>
__global__ void __launch_bounds__(TC_THREADS, 1)
dense_tc_step_kernel(const __grid_constant__ CUtensorMap tmJ, const __grid_constant__ CUtensorMap tmJlo,
                     const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmGlo,
                     const TcParams p) {
    using S = TcShape<BN>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[S::kStages], empty_bar[S::kStages], tmem_full_bar;
    __shared__ uint32_t tmem_base_slot;

    pdl_trigger();
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m0 = blockIdx.x * TC_BM, n0 = blockIdx.y * BN;
    const int nkb = (p.n + TC_BK - 1) / TC_BK;
    const int nchunks = nkb < S::kAcc - 1 ? nkb : S::kAcc - 1;  // chunks of k the main term is cut into

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJ));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJlo));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmGlo));
        for (int s = 0; s < S::kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
        }
        mbar_init(&tmem_full_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {  // whole warp: allocate the accumulator columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_slot)),
                     "r"((uint32_t)S::kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = tmem_base_slot;

    pdl_wait();  // everything below reads what the previous step wrote (GT, GT_lo, h, m1, m2)

    if (warp == 0 && lane == 0) {
        // ===== TMA producer =====
        for (int kb = 0; kb < nkb; ++kb) {
            const int s = kb % S::kStages;
            const uint32_t ph = (kb / S::kStages) & 1;
            mbar_wait(&empty_bar[s], ph ^ 1);
            uint8_t *st = smem + (size_t)s * S::kStageBytes;
            mbar_expect_tx(&full_bar[s], S::kStageBytes);
            tma_load_2d(st, &tmJ, kb * TC_BK, m0, &full_bar[s]);
            tma_load_2d(st + TC_BM * 128, &tmJlo, kb * TC_BK, m0, &full_bar[s]);
            tma_load_2d(st + 2 * TC_BM * 128, &tmG, kb * TC_BK, n0, &full_bar[s]);
            tma_load_2d(st + 2 * TC_BM * 128 + BN * 128, &tmGlo, kb * TC_BK, n0, &full_bar[s]);
        }
    } else if (warp == 1 && lane == 0) {
        // ===== MMA issuer =====
        constexpr uint32_t idesc = umma_idesc_tf32(TC_BM, BN);
        uint32_t started = 0;  // bit c: accumulator c holds something
        for (int kb = 0; kb < nkb; ++kb) {
            const int c = 1 + (kb * nchunks) / nkb;  // accumulator of this k-block's main term
            const uint32_t d_main = tmem_d + (uint32_t)(c * BN);
            const int s = kb % S::kStages;
            const uint32_t ph = (kb / S::kStages) & 1;
            mbar_wait(&full_bar[s], ph);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t a_hi = smem_u32(smem + (size_t)s * S::kStageBytes);
            const uint32_t a_lo = a_hi + TC_BM * 128;
            const uint32_t b_hi = a_hi + 2 * TC_BM * 128;
            const uint32_t b_lo = b_hi + BN * 128;
#pragma unroll
            for (int k = 0; k < TC_BK / TC_UMMA_K; ++k) {
                const uint32_t ko = k * TC_UMMA_K * 4;  // bytes inside the 128-byte swizzle atom
                const uint64_t dAh = umma_desc_sw128(a_hi + ko), dAl = umma_desc_sw128(a_lo + ko);
                const uint64_t dBh = umma_desc_sw128(b_hi + ko), dBl = umma_desc_sw128(b_lo + ko);
                umma_tf32(tmem_d, dAl, dBh, idesc, started & 1u);
                umma_tf32(tmem_d, dAh, dBl, idesc, 1);
                umma_tf32(d_main, dAh, dBh, idesc, (started >> c) & 1u);
                started |= 1u | (1u << c);
            }
            umma_commit(&empty_bar[s]);  // frees the smem stage when these MMAs have read it
        }
        umma_commit(&tmem_full_bar);  // accumulator complete
    } else if (warp >= 2) {
        // ===== epilogue: TMEM -> registers -> FEM update -> HBM =====
        mbar_wait(&tmem_full_bar, 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int quad = warp & 3;
        const int i = m0 + quad * 32 + lane;
        const bool row_ok = i < p.n;
        const Sc<float> &sc = p.sc;
        const size_t rowoff = (size_t)(row_ok ? i : 0) * p.Rb + n0;
#pragma unroll 1
        for (int c0 = 0; c0 < BN; c0 += 16) {
            float f[16];
            const uint32_t lane_base = tmem_d + ((uint32_t)(quad * 32) << 16) + (uint32_t)c0;
            tmem_ld16(lane_base + (uint32_t)BN, f);  // warp-collective: no divergence here
#pragma unroll
            for (int c = 2; c <= S::kAcc; ++c) {    // chunks of the main term in k order, the small terms last
                if (c < S::kAcc && c > nchunks) continue;  // (warp-uniform)
                float part[16];
                tmem_ld16(lane_base + (uint32_t)((c % S::kAcc) * BN), part);
#pragma unroll
                for (int k = 0; k < 16; ++k) f[k] += part[k];
            }
            if (row_ok) {
                float hv[16], a1[16], a2[16];
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    const float4 x = __ldcs(reinterpret_cast<const float4 *>(p.h + rowoff + c0) + v);
                    const float4 y = __ldcs(reinterpret_cast<const float4 *>(p.m1 + rowoff + c0) + v);
                    const float4 z = __ldcs(reinterpret_cast<const float4 *>(p.m2 + rowoff + c0) + v);
                    hv[4 * v] = x.x, hv[4 * v + 1] = x.y, hv[4 * v + 2] = x.z, hv[4 * v + 3] = x.w;
                    a1[4 * v] = y.x, a1[4 * v + 1] = y.y, a1[4 * v + 2] = y.z, a1[4 * v + 3] = y.w;
                    a2[4 * v] = z.x, a2[4 * v + 1] = z.y, a2[4 * v + 2] = z.z, a2[4 * v + 3] = z.w;
                }
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    const float hk = hv[k];
                    const float g = (-2.0f * f[k] + hk * sc.inv_beta) * p1mp_of(hk);  // dU/dp = -2 sum_j J_ij m_j
                    hv[k] = opt_update(hk, g, a1[k], a2[k], sc);
                    const float mg = mag_of(hv[k]);
                    const size_t go = (size_t)(n0 + c0 + k) * p.n + i;  // GT[a][i]: lanes = consecutive i
                    p.gt_out[go] = mg;
                    p.gtlo_out[go] = mg - tf32_hi(mg);
                }
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    __stcs(reinterpret_cast<float4 *>(p.h + rowoff + c0) + v,
                           make_float4(hv[4 * v], hv[4 * v + 1], hv[4 * v + 2], hv[4 * v + 3]));
                    __stcs(reinterpret_cast<float4 *>(p.m1 + rowoff + c0) + v,
                           make_float4(a1[4 * v], a1[4 * v + 1], a1[4 * v + 2], a1[4 * v + 3]));
                    __stcs(reinterpret_cast<float4 *>(p.m2 + rowoff + c0) + v,
                           make_float4(a2[4 * v], a2[4 * v + 1], a2[4 * v + 2], a2[4 * v + 3]));
                }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"((uint32_t)S::kTmemCols));
    }
}

// J_lo = J - hi(J), once at fem_create
__global__ void __launch_bounds__(kThreads) tc_split_kernel(const float *x, float *lo, int64_t count) {
    const int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (idx < count) lo[idx] = x[idx] - tf32_hi(x[idx]);
}

// GT[a][i] = tanh(h[i][a] / 2) and its low part, from the fp32 fields (entry to the tensor-core phase)
__global__ void __launch_bounds__(kThreads) tc_prepare_kernel(const float *h, float *gt, float *gtlo, int n, int Rb) {
    __shared__ float tile[32][33];
    const int i0 = blockIdx.x * 32, a0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int k = ty; k < 32; k += 8) {
        const int i = i0 + k, a = a0 + tx;
        if (i < n && a < Rb) tile[k][tx] = (float)mag_of((double)h[(size_t)i * Rb + a]);
    }
    __syncthreads();
    for (int k = ty; k < 32; k += 8) {
        const int a = a0 + k, i = i0 + tx;
        if (i < n && a < Rb) {
            const float mg = tile[tx][k];
            gt[(size_t)a * n + i] = mg;
            gtlo[(size_t)a * n + i] = mg - tf32_hi(mg);
        }
    }
}

// ---- host side ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
    }
    return fn;
}

// row-major fp32 matrix [rows][cols] (pitch = cols), box = 32 columns x box_rows, 128-byte swizzle
static bool make_map(CUtensorMap *tm, const float *base, int rows, int cols, int box_rows) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)cols * 4};
    cuuint32_t box[2] = {(cuuint32_t)TC_BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int tc_tile_n(int n, int Rb, int forced) {  // 0 = tensor-core path not applicable
    if (n % 4 != 0) return 0;   // TMA needs a 16-byte row pitch
    // default 128: four accumulators (small terms + three chunks of k); 256 is ~7% faster per step but has room
    // for two accumulators only (5e-5 instead of 2e-5 on the marginals at step 50 of cfg 4b)
    for (int bn : {128, 64, 32})
        if (Rb % bn == 0 && (forced == 0 || forced == bn)) return bn;
    if (forced == 256 && Rb % 256 == 0) return 256;
    return 0;
}

template <int BN>
static bool launch_tc(Handle *hd, const TcParams &p, const CUtensorMap *maps) {
    using S = TcShape<BN>;
    const void *fn = reinterpret_cast<const void *>(&dense_tc_step_kernel<BN>);
    if (!hd->attr_done.count(fn)) {  // per handle, i.e. per device and context
        if (cudaFuncSetAttribute(dense_tc_step_kernel<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::kSmem) !=
            cudaSuccess)
            return false;
        hd->attr_done.insert(fn);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ceil_div(p.n, TC_BM), (unsigned)(p.Rb / BN));
    cfg.blockDim = dim3(TC_THREADS);
    cfg.dynamicSmemBytes = S::kSmem;
    cfg.stream = hd->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, dense_tc_step_kernel<BN>, maps[0], maps[1], maps[2], maps[3], p) == cudaSuccess;
}

void launch_tc_split(Handle *hd) {
    const int64_t count = (int64_t)hd->dp.n * hd->dp.n;
    tc_split_kernel<<<(unsigned)ceil_div(count, kThreads), kThreads, 0, hd->stream>>>(hd->dp.J, hd->Jlo, count);
    hd->launches++;
}

// One fp32 step of the dense kind on the tensor cores.  Returns false when the path does not apply (caller falls
// back to the CUDA-core GEMM).
bool launch_step_dense_tc(Handle *hd, const StepScalars &sc) {
    const int n = hd->dp.n, Rb = hd->Rb;
    const int bn = tc_tile_n(n, Rb, (int)hd->opt_tc_tile_n);
    if (bn == 0 || hd->R != Rb || !hd->Jlo || !hd->opt_tensor_cores) return false;  // (tensor_cores = 2 forces this path)
    if (hd->tc_maps_R != hd->R || hd->tc_maps_bn != bn) {  // the maps bake in R (rows of GT) and the box height bn
        CUtensorMap *m = reinterpret_cast<CUtensorMap *>(hd->tc_maps);
        bool ok = make_map(&m[0], hd->dp.J, n, n, TC_BM) && make_map(&m[1], hd->Jlo, n, n, TC_BM);
        for (int k = 0; k < 2 && ok; ++k)
            ok = make_map(&m[2 + 2 * k], hd->g[k], hd->R, n, bn) && make_map(&m[3 + 2 * k], hd->glo[k], hd->R, n, bn);
        if (!ok) return false;
        hd->tc_maps_R = hd->R;
        hd->tc_maps_bn = bn;
    }
    if (!hd->tc_ready) {
        dim3 grid((unsigned)ceil_div(n, 32), (unsigned)ceil_div(Rb, 32));
        tc_prepare_kernel<<<grid, kThreads, 0, hd->stream>>>(hd->h, hd->g[hd->cur], hd->glo[hd->cur], n, Rb);
        hd->launches++;
        hd->tc_ready = true;
    }
    TcParams p;
    p.h = hd->h;
    p.m1 = hd->m1;
    p.m2 = hd->m2;
    p.gt_out = hd->g[hd->cur ^ 1];
    p.gtlo_out = hd->glo[hd->cur ^ 1];
    p.sc = Sc<float>(sc);
    p.n = n;
    p.Rb = Rb;
    const CUtensorMap *all = reinterpret_cast<const CUtensorMap *>(hd->tc_maps);
    CUtensorMap maps[4] = {all[0], all[1], all[2 + 2 * hd->cur], all[3 + 2 * hd->cur]};
    bool ok = false;
    switch (bn) {
        case 256: ok = launch_tc<256>(hd, p, maps); break;
        case 128: ok = launch_tc<128>(hd, p, maps); break;
        case 64: ok = launch_tc<64>(hd, p, maps); break;
        default: ok = launch_tc<32>(hd, p, maps); break;
    }
    if (ok) {
        hd->launches++;
        hd->tc_launches++;
    } else {
        (void)cudaGetLastError();
        // g[cur] was overwritten with the TRANSPOSED layout above: the CUDA-core path must rebuild it from h
        // (launch_step_q2_t does so when it sees tc_ready)
    }
    return ok;
}

}  // namespace fem
