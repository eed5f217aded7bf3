// Dense-coupling Ising step on the INT8 path of the 5th-generation tensor cores (cfg 4b: SK, n = 4096, R = 1024).
//
// Why: the 3xTF32 kernel (k_dense_tc.cu) issues three tf32 MMAs per product and moves 8 bytes of operands per matrix
// element (hi + lo fp32 containers); it is bound by 1.73 waves of tensor time plus the operand feed out of L2
// (DESIGN.md section 6).  Here both operands are FIXED-POINT numbers cut into three signed 8-bit digits (the Ozaki
// scheme): J_ij = sJ_i * Jx_ij / 2^22 with Jx an integer of 23 bits (sJ_i = the row's largest |J_ij|, once at the first
// step), m_j = Mx_j / 2^22 likewise (|m| < 1), Jx = d0 2^16 + d1 2^8 + d2 with d in [-128, 127].  The product sum
//     sum_j Jx_ij Mx_j = 2^32 S00 + 2^24 (S01 + S10) + 2^16 (S02 + S11 + S20) + [2^8 (S12 + S21) + S22],   S_ab = sum_j d_a(J) d_b(M)
// is formed by SIX kind::i8 MMAs per k-step into three int32 TMEM accumulators (one per weight); the bracket is dropped
// (2^-24 of the leading term, the level of fp32 rounding).  Integer accumulation is EXACT: no accumulator truncation bias,
// hence no need to cut k into separate accumulators as the tf32 kernel must.  Per matrix element the step moves 3 bytes per
// operand instead of 8, and the int8 MMA rate is 4x the tf32 rate (6 MMAs = 1.5 tf32-equivalents instead of 3).
// Error of the local field: both operands carry an absolute error of 2^-23 of their scale, random in sign: ~5e-7 on
// F = O(1) at n = 4096, the level of the 3xTF32 kernel.
//
// Everything else follows k_dense_tc.cu: one CTA computes a 128 x BN tile of F, operands K-major through TMA (128-byte
// swizzle, a k-block is 128 int8 = one swizzle atom) and an mbarrier ring, accumulators in TMEM, and the whole FEM update
// (S29 PAPER.md:667 + Adam PAPER.md:88) fused in the epilogue, which also cuts the new magnetisations into digits for the
// next step (GT8[digit][a][j], transposed: the epilogue's lanes are rows i).
#include <cuda.h>

#include "device_math.cuh"

namespace fem {

constexpr int I8_BM = 128;       // rows of F per CTA = TMEM lanes
constexpr int I8_BK = 128;       // int8 elements per k-block = one 128-byte swizzle atom
constexpr int I8_UMMA_K = 32;    // int8 elements per tcgen05.mma
constexpr int I8_EPI_GROUPS = 4;  // epilogue warps per TMEM lane quadrant (each takes BN / groups columns)
constexpr int I8_THREADS = 64 + 128 * I8_EPI_GROUPS;
constexpr int I8_FRAC_BITS = 22; // fixed point: |x| <= 2^22 - 1, digits d0 in [-64, 64], d1, d2 in [-128, 127]

template <int BN>
struct I8Shape {
    static constexpr int kStageBytes = 3 * I8_BM * 128 + 3 * BN * 128;  // three digits of A and of B
    static constexpr int kStages = BN >= 128 ? 2 : 3;
    static constexpr int kColsWarp = BN / I8_EPI_GROUPS >= 8 ? BN / I8_EPI_GROUPS : 8;
    static constexpr int kEpiBytes = 4 * I8_EPI_GROUPS * 3 * 32 * (kColsWarp + 4) * 4;  // epilogue staging (reuses the stages)
    static constexpr int kSmem = (kStages * kStageBytes > kEpiBytes ? kStages * kStageBytes : kEpiBytes) + 1024;
    static constexpr int kTmemCols = 3 * BN <= 128 ? 128 : (3 * BN <= 256 ? 256 : 512);
};

struct I8Params {
    float *h, *m1, *m2;        // [i][a], row pitch Rb
    signed char *gt8_out;      // [3][R][np] digits of the new magnetisations, transposed
    const double *jscale;      // [n] sJ_i / 2^6: F = jscale_i * (2^16 acc0 + 2^8 acc1 + acc2)
    Sc<float> sc;
    int n, np, Rb;
};

// ---- PTX wrappers (as in k_dense_tc.cu) ----
__device__ __forceinline__ uint32_t i8_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void i8_mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(i8_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void i8_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(i8_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void i8_mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(i8_smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void i8_tma_load_2d(void *smem_dst, const CUtensorMap *tm, int c0, int c1, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            i8_smem_u32(smem_dst)),
        "l"(tm), "r"(c0), "r"(c1), "r"(i8_smem_u32(bar))
        : "memory");
}
// the same tile delivered to the same shared-memory offset (and mbarrier) of every CTA of the cluster named in cta_mask
__device__ __forceinline__ void i8_tma_load_2d_mc(void *smem_dst, const CUtensorMap *tm, int c0, int c1, uint64_t *bar, uint16_t cta_mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
            i8_smem_u32(smem_dst)),
        "l"(tm), "r"(c0), "r"(c1), "r"(i8_smem_u32(bar)), "h"(cta_mask)
        : "memory");
}
__device__ __forceinline__ void i8_commit_mc(uint64_t *bar, uint16_t cta_mask) {  // arrive on the barrier at this offset in every CTA of the mask
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(i8_smem_u32(bar)),
                 "h"(cta_mask)
                 : "memory");
}
__device__ __forceinline__ void i8_cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint64_t i8_desc_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFF) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// kind::i8: int32 accumulator (c_format 2), signed 8-bit A and B (format 1), both K-major
__host__ __device__ constexpr uint32_t i8_idesc(int M, int N) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void i8_umma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void i8_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(i8_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void i8_tmem_ld16(uint32_t taddr, int *v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void i8_tmem_ld8(uint32_t taddr, int *v) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void i8_tmem_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// x in [-(2^22 - 1), 2^22 - 1] -> three balanced digits, x = d0 2^16 + d1 2^8 + d2
__host__ __device__ __forceinline__ void i8_digits(int x, int &d0, int &d1, int &d2) {
    d2 = ((x + 128) & 255) - 128;
    const int x1 = (x - d2) >> 8;
    d1 = ((x1 + 128) & 255) - 128;
    d0 = (x1 - d1) >> 8;
}
__device__ __forceinline__ int i8_fixed_of(float m) {  // |m| <= 1
    const int x = __float2int_rn(m * (float)(1 << I8_FRAC_BITS));
    return max(-((1 << I8_FRAC_BITS) - 1), min((1 << I8_FRAC_BITS) - 1, x));
}

// ---- the fused step ----
// Warp roles: warp 0 = TMA producer (one elected lane), warp 1 = TMEM allocator + MMA issuer (one elected lane), warps 2..17 =
// epilogue (warp w reads TMEM lanes 32*(w%4) .. +31; the two warps of a lane quadrant split the BN columns).  With one warp per
// scheduler the epilogue was bound by its own dependency chains and by DRAM round trips (2 x 44 us of a 147 us step): two warps
// per scheduler, and the h / m1 / m2 rows of a 16-column block are requested one block ahead (the first before the main loop ends).
// CL: 2 x 2 thread-block clusters with operand multicast.  The four CTAs of a cluster compute a 256 x 2 BN block of F; the two
// CTAs with the same rows share the J digits, the two with the same replica columns share the GT8 digits: every CTA fetches
// HALF of each of its operand tiles and multicasts it to the CTA that needs it too, so the L2 -> SMEM traffic per CTA is
// halved (the int8 main loop is bound by that feed: 96 KB per 24 MMAs).  A stage may be refilled when the CTA itself and
// both CTAs it multicasts to have consumed it: the MMA issuer's commit arrives on the empty barrier of all three.
template <int BN, bool CL>
__global__ void __launch_bounds__(I8_THREADS, 1)
dense_i8_step_kernel(const __grid_constant__ CUtensorMap tmJ0, const __grid_constant__ CUtensorMap tmJ1,
                     const __grid_constant__ CUtensorMap tmJ2, const __grid_constant__ CUtensorMap tmG0,
                     const __grid_constant__ CUtensorMap tmG1, const __grid_constant__ CUtensorMap tmG2, const I8Params p) {
    using S = I8Shape<BN>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[S::kStages], empty_bar[S::kStages], tmem_full_bar;
    __shared__ uint32_t tmem_base_slot;

    pdl_trigger();
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m0 = blockIdx.x * I8_BM, n0 = blockIdx.y * BN;
    const int nkb = (p.n + I8_BK - 1) / I8_BK;
    uint32_t cx = 0, cy = 0;  // position inside the 2 x 2 cluster (rank = cx + 2 cy)
    if (CL) {
        asm volatile("mov.u32 %0, %%cluster_ctaid.x;" : "=r"(cx));
        asm volatile("mov.u32 %0, %%cluster_ctaid.y;" : "=r"(cy));
    }

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJ0));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJ1));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJ2));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG0));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG1));
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG2));
        for (int s = 0; s < S::kStages; ++s) {
            i8_mbar_init(&full_bar[s], 1);
            i8_mbar_init(&empty_bar[s], CL ? 3 : 1);  // CL: this CTA and the two it multicasts to
        }
        i8_mbar_init(&tmem_full_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {  // whole warp: allocate the accumulator columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(i8_smem_u32(&tmem_base_slot)),
                     "r"((uint32_t)S::kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CL) i8_cluster_sync();  // every CTA's barriers are initialised before a peer multicasts into it or arrives on them
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = tmem_base_slot;

    pdl_wait();  // everything below reads what the previous step wrote (GT8, h, m1, m2)

    if (warp == 0 && lane == 0) {
        // ===== TMA producer: three digit tiles of J rows m0.., three of GT rows n0.. per k-block =====
        for (int kb = 0; kb < nkb; ++kb) {
            const int s = kb % S::kStages;
            const uint32_t ph = (kb / S::kStages) & 1;
            i8_mbar_wait(&empty_bar[s], ph ^ 1);
            uint8_t *st = smem + (size_t)s * S::kStageBytes;
            i8_mbar_expect_tx(&full_bar[s], S::kStageBytes);
            uint8_t *sb = st + 3 * I8_BM * 128;
            if (CL) {
                // my half of the J rows (the other CTA of my row pair loads the other half), to both of us
                const uint16_t maskA = (uint16_t)((1u << cx) | (1u << (cx + 2)));
                uint8_t *da = st + cy * (I8_BM / 2) * 128;
                const int ra = m0 + (int)cy * (I8_BM / 2);
                i8_tma_load_2d_mc(da, &tmJ0, kb * I8_BK, ra, &full_bar[s], maskA);
                i8_tma_load_2d_mc(da + I8_BM * 128, &tmJ1, kb * I8_BK, ra, &full_bar[s], maskA);
                i8_tma_load_2d_mc(da + 2 * I8_BM * 128, &tmJ2, kb * I8_BK, ra, &full_bar[s], maskA);
                // my half of the GT8 rows, to both CTAs of my column pair
                const uint16_t maskB = (uint16_t)(3u << (2 * cy));
                uint8_t *db = sb + cx * (BN / 2) * 128;
                const int rb = n0 + (int)cx * (BN / 2);
                i8_tma_load_2d_mc(db, &tmG0, kb * I8_BK, rb, &full_bar[s], maskB);
                i8_tma_load_2d_mc(db + BN * 128, &tmG1, kb * I8_BK, rb, &full_bar[s], maskB);
                i8_tma_load_2d_mc(db + 2 * BN * 128, &tmG2, kb * I8_BK, rb, &full_bar[s], maskB);
            } else {
                i8_tma_load_2d(st, &tmJ0, kb * I8_BK, m0, &full_bar[s]);
                i8_tma_load_2d(st + I8_BM * 128, &tmJ1, kb * I8_BK, m0, &full_bar[s]);
                i8_tma_load_2d(st + 2 * I8_BM * 128, &tmJ2, kb * I8_BK, m0, &full_bar[s]);
                i8_tma_load_2d(sb, &tmG0, kb * I8_BK, n0, &full_bar[s]);
                i8_tma_load_2d(sb + BN * 128, &tmG1, kb * I8_BK, n0, &full_bar[s]);
                i8_tma_load_2d(sb + 2 * BN * 128, &tmG2, kb * I8_BK, n0, &full_bar[s]);
            }
        }
    } else if (warp == 1 && lane == 0) {
        // ===== MMA issuer: acc0 = S00, acc1 = S01 + S10, acc2 = S02 + S11 + S20 =====
        constexpr uint32_t idesc = i8_idesc(I8_BM, BN);
        const uint32_t acc0 = tmem_d, acc1 = tmem_d + BN, acc2 = tmem_d + 2 * BN;
        uint32_t started = 0;
        for (int kb = 0; kb < nkb; ++kb) {
            const int s = kb % S::kStages;
            const uint32_t ph = (kb / S::kStages) & 1;
            i8_mbar_wait(&full_bar[s], ph);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t a0 = i8_smem_u32(smem + (size_t)s * S::kStageBytes);
            const uint32_t a1 = a0 + I8_BM * 128, a2 = a0 + 2 * I8_BM * 128;
            const uint32_t b0 = a0 + 3 * I8_BM * 128, b1 = b0 + BN * 128, b2 = b0 + 2 * BN * 128;
#pragma unroll
            for (int k = 0; k < I8_BK / I8_UMMA_K; ++k) {
                const uint32_t ko = k * I8_UMMA_K;  // bytes inside the 128-byte swizzle atom
                const uint64_t dA0 = i8_desc_sw128(a0 + ko), dA1 = i8_desc_sw128(a1 + ko), dA2 = i8_desc_sw128(a2 + ko);
                const uint64_t dB0 = i8_desc_sw128(b0 + ko), dB1 = i8_desc_sw128(b1 + ko), dB2 = i8_desc_sw128(b2 + ko);
                i8_umma(acc0, dA0, dB0, idesc, started);
                i8_umma(acc1, dA0, dB1, idesc, started);
                i8_umma(acc1, dA1, dB0, idesc, 1);
                i8_umma(acc2, dA0, dB2, idesc, started);
                i8_umma(acc2, dA1, dB1, idesc, 1);
                i8_umma(acc2, dA2, dB0, idesc, 1);
                started = 1;
            }
            // frees the smem stage when these MMAs have read it -- here and, with clusters, in the two CTAs that multicast into it
            if (CL) i8_commit_mc(&empty_bar[s], (uint16_t)((1u << (cx + 2 * cy)) | (1u << (cx + 2 * (1 - cy))) | (1u << ((1 - cx) + 2 * cy))));
            else i8_commit(&empty_bar[s]);
        }
        i8_commit(&tmem_full_bar);  // accumulators complete
    } else if (warp >= 2) {
        // ===== epilogue: TMEM -> registers -> FEM update -> HBM =====
        const int quad = warp & 3;
        const int i = m0 + quad * 32 + lane;
        const bool row_ok = i < p.n;
        const Sc<float> &sc = p.sc;
        constexpr int kCols = BN / I8_EPI_GROUPS >= 8 ? BN / I8_EPI_GROUPS : 8;  // columns of this warp
        const int cbeg = ((warp - 2) >> 2) * kCols;
        const bool has_cols = cbeg < BN;
        const float js = row_ok ? (float)p.jscale[i] : 0.0f;
        const size_t plane = (size_t)p.Rb * p.np;  // one digit plane of GT8
        // TMEM lanes are rows i, so a lane's h / m1 / m2 values sit a whole row pitch apart in HBM: read straight from there,
        // every load instruction touched 32 different lines and the epilogue was bound by L1 tag lookups and exposed DRAM round
        // trips (2 x 31 us of a 137 us step).  When the accumulators are complete the operand stages are free: each warp stages its
        // 32 x kCols sub-tile of the three arrays there with cp.async -- 16 lanes per row, coalesced, the whole sub-tile in flight
        // at once --, works out of shared memory (rows padded to kPitch floats: conflict-free 16-byte accesses), and writes the
        // results back through the same slots.
        constexpr int kPitch = kCols + 4;                    // floats per staged row
        constexpr int kArr = 32 * kPitch;                    // floats per staged array
        float *stg = reinterpret_cast<float *>(smem) + (size_t)(warp - 2) * (3 * kArr);
        constexpr int kChunks = kCols / 4;                   // 16-byte pieces per row
        i8_mbar_wait(&tmem_full_bar, 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (has_cols) {
            const int rows_ok = min(32, p.n - (m0 + quad * 32));  // rows of this warp inside the matrix (<= 0: none)
            const float *src[3] = {p.h, p.m1, p.m2};
#pragma unroll
            for (int arr = 0; arr < 3; ++arr)
                for (int x = lane; x < 32 * kChunks; x += 32) {
                    const int r = x / kChunks, ch = x - r * kChunks;
                    if (r < rows_ok) {
                        const float *g = src[arr] + (size_t)(m0 + quad * 32 + r) * p.Rb + n0 + cbeg + ch * 4;
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(i8_smem_u32(stg + arr * kArr + r * kPitch + ch * 4)), "l"(g)
                                     : "memory");
                    }
                }
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
            float *my = stg + lane * kPitch;
#pragma unroll 1
            for (int c0 = 0; c0 < kCols; c0 += 8) {  // 8 columns at a time: few live registers, four warps per scheduler
                int s0[8], s1[8], s2[8];
                const uint32_t lane_base = tmem_d + ((uint32_t)(quad * 32) << 16) + (uint32_t)(cbeg + c0);
                i8_tmem_ld8(lane_base, s0);  // warp-collective: no divergence here
                i8_tmem_ld8(lane_base + (uint32_t)BN, s1);
                i8_tmem_ld8(lane_base + (uint32_t)(2 * BN), s2);
                i8_tmem_wait();
                if (row_ok) {
                    float hv[8], a1[8], a2[8];
#pragma unroll
                    for (int v = 0; v < 2; ++v) {
                        const float4 x = *reinterpret_cast<const float4 *>(my + c0 + 4 * v);
                        const float4 y = *reinterpret_cast<const float4 *>(my + kArr + c0 + 4 * v);
                        const float4 z = *reinterpret_cast<const float4 *>(my + 2 * kArr + c0 + 4 * v);
                        hv[4 * v] = x.x, hv[4 * v + 1] = x.y, hv[4 * v + 2] = x.z, hv[4 * v + 3] = x.w;
                        a1[4 * v] = y.x, a1[4 * v + 1] = y.y, a1[4 * v + 2] = y.z, a1[4 * v + 3] = y.w;
                        a2[4 * v] = z.x, a2[4 * v + 1] = z.y, a2[4 * v + 2] = z.z, a2[4 * v + 3] = z.w;
                    }
                    signed char *gp = p.gt8_out + (size_t)(n0 + cbeg + c0) * p.np + i;  // GT8[digit][a][i]: lanes = consecutive i
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        // 2^16 acc0 + 2^8 acc1 + acc2 in fp32: |acc0| <= 2^24 converts exactly, the other two round at 2^-24 of
                        // themselves, the sums at 2^-24 of the total -- the level of the digits that were dropped
                        const float t = fmaf((float)s0[k], 65536.0f, fmaf((float)s1[k], 256.0f, (float)s2[k]));
                        const float f = js * t;  // F_i = sum_j J_ij m_j
                        const float hk = hv[k];
                        const float g = (-2.0f * f + hk * sc.inv_beta) * p1mp_of(hk);  // dU/dp = -2 sum_j J_ij m_j
                        hv[k] = opt_update(hk, g, a1[k], a2[k], sc);
                        int d0, d1, d2;
                        i8_digits(i8_fixed_of(mag_of(hv[k])), d0, d1, d2);
                        gp[0] = (signed char)d0;
                        gp[plane] = (signed char)d1;
                        gp[2 * plane] = (signed char)d2;
                        gp += p.np;
                    }
#pragma unroll
                    for (int v = 0; v < 2; ++v) {
                        *reinterpret_cast<float4 *>(my + c0 + 4 * v) = make_float4(hv[4 * v], hv[4 * v + 1], hv[4 * v + 2], hv[4 * v + 3]);
                        *reinterpret_cast<float4 *>(my + kArr + c0 + 4 * v) = make_float4(a1[4 * v], a1[4 * v + 1], a1[4 * v + 2], a1[4 * v + 3]);
                        *reinterpret_cast<float4 *>(my + 2 * kArr + c0 + 4 * v) = make_float4(a2[4 * v], a2[4 * v + 1], a2[4 * v + 2], a2[4 * v + 3]);
                    }
                }
            }
            __syncwarp();
            float *dst[3] = {p.h, p.m1, p.m2};
#pragma unroll
            for (int arr = 0; arr < 3; ++arr)
                for (int x = lane; x < 32 * kChunks; x += 32) {
                    const int r = x / kChunks, ch = x - r * kChunks;
                    if (r < rows_ok)
                        __stcs(reinterpret_cast<float4 *>(dst[arr] + (size_t)(m0 + quad * 32 + r) * p.Rb + n0 + cbeg + ch * 4),
                               *reinterpret_cast<const float4 *>(stg + arr * kArr + r * kPitch + ch * 4));
                }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();
    if (CL) i8_cluster_sync();  // no CTA leaves while a peer may still arrive on its barriers
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"((uint32_t)S::kTmemCols));
    }
}

// J -> row scales and three digit planes, once per handle.  One CTA per row i; columns n .. np-1 of the planes are zero.
__global__ void __launch_bounds__(256) i8_split_J_kernel(const float *J, signed char *J8, double *jscale, int n, int np) {
    __shared__ float red[256];
    const int i = blockIdx.x;
    const float *row = J + (size_t)i * n;
    float mx = 0.0f;
    for (int j = threadIdx.x; j < n; j += 256) mx = fmaxf(mx, fabsf(row[j]));
    red[threadIdx.x] = mx;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] = fmaxf(red[threadIdx.x], red[threadIdx.x + s]);
        __syncthreads();
    }
    mx = red[0];
    const double lim = (double)((1 << I8_FRAC_BITS) - 1);
    const double sJ = mx > 0.0f ? (double)mx / lim : 1.0;  // J_ij ~= sJ * Jx_ij
    if (threadIdx.x == 0) jscale[i] = sJ / 64.0;           // F = sJ 2^-22 2^16 (2^16 acc0 + 2^8 acc1 + acc2)
    const size_t plane = (size_t)n * np;
    for (int j = threadIdx.x; j < np; j += 256) {
        int d0 = 0, d1 = 0, d2 = 0;
        if (j < n) {
            const long long x = llrint((double)row[j] / sJ);
            i8_digits((int)max(-(long long)lim, min((long long)lim, x)), d0, d1, d2);
        }
        const size_t o = (size_t)i * np + j;
        J8[o] = (signed char)d0;
        J8[plane + o] = (signed char)d1;
        J8[2 * plane + o] = (signed char)d2;
    }
}

// GT8[digit][a][i] of m = tanh(h[i][a] / 2) from the fp32 fields (entry to the tensor-core phase)
__global__ void __launch_bounds__(kThreads) i8_prepare_kernel(const float *h, signed char *gt8, int n, int np, int Rb) {
    __shared__ float tile[32][33];
    const int i0 = blockIdx.x * 32, a0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int k = ty; k < 32; k += 8) {
        const int i = i0 + k, a = a0 + tx;
        if (i < n && a < Rb) tile[k][tx] = mag_of(h[(size_t)i * Rb + a]);  // the fp32 function the epilogue uses
    }
    __syncthreads();
    const size_t plane = (size_t)Rb * np;
    for (int k = ty; k < 32; k += 8) {
        const int a = a0 + k, i = i0 + tx;
        if (i < n && a < Rb) {
            int d0, d1, d2;
            i8_digits(i8_fixed_of(tile[tx][k]), d0, d1, d2);
            const size_t o = (size_t)a * np + i;
            gt8[o] = (signed char)d0;
            gt8[plane + o] = (signed char)d1;
            gt8[2 * plane + o] = (signed char)d2;
        }
    }
}

// ---- host side ----
typedef CUresult (*I8EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static I8EncodeTiledFn i8_encode_fn() {
    static I8EncodeTiledFn fn = nullptr;  // a driver entry point: process-wide by nature
    if (!fn) {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<I8EncodeTiledFn>(ptr);
    }
    return fn;
}

// int8 matrix [rows][cols] with a row pitch of `pitch` bytes, box = 128 columns x box_rows, 128-byte swizzle; columns past
// `cols` read as zero
static bool i8_make_map(CUtensorMap *tm, const signed char *base, int rows, int cols, int pitch, int box_rows) {
    I8EncodeTiledFn fn = i8_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)pitch};
    cuuint32_t box[2] = {(cuuint32_t)I8_BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<signed char *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static int i8_tile_n(int Rb, int forced) {  // 0 = not applicable (three accumulators of BN columns must fit 512 TMEM columns)
    for (int bn : {128, 64, 32})
        if (Rb % bn == 0 && (forced == 0 || forced == bn)) return bn;
    return 0;
}

template <int BN, bool CL>
static bool i8_launch(Handle *hd, const I8Params &p, const CUtensorMap *maps) {
    using S = I8Shape<BN>;
    const void *fn = reinterpret_cast<const void *>(&dense_i8_step_kernel<BN, CL>);
    if (!hd->attr_done.count(fn)) {
        if (cudaFuncSetAttribute(dense_i8_step_kernel<BN, CL>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::kSmem) != cudaSuccess) return false;
        hd->attr_done.insert(fn);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ceil_div(p.n, I8_BM), (unsigned)(p.Rb / BN));
    cfg.blockDim = dim3(I8_THREADS);
    cfg.dynamicSmemBytes = S::kSmem;
    cfg.stream = hd->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.numAttrs = 1;
    if (CL) {
        attr[1].id = cudaLaunchAttributeClusterDimension;
        attr[1].val.clusterDim.x = 2;
        attr[1].val.clusterDim.y = 2;
        attr[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    cfg.attrs = attr;
    return cudaLaunchKernelEx(&cfg, dense_i8_step_kernel<BN, CL>, maps[0], maps[1], maps[2], maps[3], maps[4], maps[5], p) == cudaSuccess;
}

// One fp32 step of the dense kind on the int8 tensor-core path.  Returns false when the path does not apply (the caller
// tries the 3xTF32 kernel, then the CUDA-core GEMM).
bool launch_step_dense_i8(Handle *hd, const StepScalars &sc) {
    const int n = hd->dp.n, Rb = hd->Rb, np = hd->i8_np;
    const int bn = i8_tile_n(Rb, (int)hd->opt_tc_tile_n);
    if (bn == 0 || hd->R != Rb || !hd->J8 || hd->opt_tensor_cores != 1) return false;
    // 2 x 2 clusters with operand multicast where the grid allows it ("tc_cluster" option: 1 = automatic, 0 = off)
    const bool cl = hd->opt_tc_cluster != 0 && bn >= 64 && ceil_div(n, I8_BM) % 2 == 0 && (Rb / bn) % 2 == 0;
    CUtensorMap *m = reinterpret_cast<CUtensorMap *>(hd->tc8_maps);
    const int key_bn = cl ? -bn : bn;  // the maps bake in R (rows of GT8) and the box heights (halved with multicast)
    if (hd->tc8_maps_R != hd->R || hd->tc8_maps_bn != key_bn) {
        bool ok = true;
        for (int d = 0; d < 3 && ok; ++d) ok = i8_make_map(&m[d], hd->J8 + (size_t)d * n * np, n, n, np, cl ? I8_BM / 2 : I8_BM);
        for (int k = 0; k < 2 && ok; ++k)
            for (int d = 0; d < 3 && ok; ++d)
                ok = i8_make_map(&m[3 + 3 * k + d], hd->gt8[k] + (size_t)d * hd->R * np, hd->R, n, np, cl ? bn / 2 : bn);
        if (!ok) return false;
        hd->tc8_maps_R = hd->R;
        hd->tc8_maps_bn = key_bn;
    }
    if (!hd->tc8_split_done) {
        i8_split_J_kernel<<<(unsigned)n, 256, 0, hd->stream>>>(hd->dp.J, hd->J8, hd->jscale, n, np);
        hd->launches++;
        hd->tc8_split_done = true;
    }
    if (!hd->tc8_ready) {
        dim3 grid((unsigned)ceil_div(n, 32), (unsigned)ceil_div(Rb, 32));
        i8_prepare_kernel<<<grid, kThreads, 0, hd->stream>>>(hd->h, hd->gt8[hd->cur], n, np, Rb);
        hd->launches++;
        hd->tc8_ready = true;
    }
    I8Params p;
    p.h = hd->h;
    p.m1 = hd->m1;
    p.m2 = hd->m2;
    p.gt8_out = hd->gt8[hd->cur ^ 1];
    p.jscale = hd->jscale;
    p.sc = Sc<float>(sc);
    p.n = n;
    p.np = np;
    p.Rb = Rb;
    CUtensorMap maps[6] = {m[0], m[1], m[2], m[3 + 3 * hd->cur], m[4 + 3 * hd->cur], m[5 + 3 * hd->cur]};
    bool ok = false;
    switch (bn) {
        case 128: ok = cl ? i8_launch<128, true>(hd, p, maps) : i8_launch<128, false>(hd, p, maps); break;
        case 64: ok = cl ? i8_launch<64, true>(hd, p, maps) : i8_launch<64, false>(hd, p, maps); break;
        default: ok = i8_launch<32, false>(hd, p, maps); break;
    }
    if (ok) {
        hd->launches++;
        hd->tc_launches++;
        hd->tc8_launches++;
    } else {
        (void)cudaGetLastError();
        hd->tc8_ready = false;
    }
    return ok;
}

}  // namespace fem
