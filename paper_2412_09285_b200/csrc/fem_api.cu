// C ABI of libfem_b200 (include/fem.h): validation, workspace carve-up, step scheduling, result copies.
// All arithmetic of the method runs in the kernels (k_*.cu); the host only computes the per-step
// scalars (1/beta_t and Adam's bias corrections) in double, as DESIGN.md section 6 states.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <thread>

#include "fem_internal.cuh"

namespace fem {

// launchers defined in the kernel files
void launch_step_q2(Handle *hd, const StepScalars &sc, bool wide, int blk_begin, int blk_count);
void launch_prepare_q2(Handle *hd, bool wide);
void launch_potts(Handle *hd, const StepScalars &sc, bool wide, bool step, int blk_begin, int blk_count);
void launch_sigmoid(Handle *hd, float *out);
bool potts_block_ok(int q, int Rb);
bool potts_si_applicable(const Handle *hd);                  // k_step_potts_si.cu
void launch_potts_si_relayout(Handle *hd, bool to_si);
void launch_potts_softmax(Handle *hd, float *out);
void launch_qsat(Handle *hd, const StepScalars &sc, bool wide, bool step, int blk_begin, int blk_count);  // k_step_qsat.cu
void launch_tc_split(Handle *hd);
bool persist_eligible(const Handle *hd);
void persist_prepare(Handle *hd, const int64_t *row_ptr, const int *order);
cudaError_t persist_run(Handle *hd, bool wide, int t_begin, int t_end, StepScalars (*scalars)(void *, int), void *ctx);

static std::string g_create_error;

struct Layout {
    size_t row_ptr, col, w, rowsum, long_rows, vw, lit_state, order, rank, J, Jlo, glo0, glo1, J8, gt8_0, gt8_1, jscale, field, occ_ptr, occ, clause_ptr, lits;
    size_t h, m1, m2, g0, g1, stage, hW, m1W, m2W, gW0, gW1, colsum0, colsum1, colsum2, cfg, e_part_i, e_part_d, part_part, e_int, e_real, part,
        best, total;
};

static size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

// entries per Max-SAT occurrence are padded to a power of two so that one occurrence is one aligned vector load
static int occ_stride(int kmax) {
    const int ks = std::max(1, kmax - 1);
    int st = 1;
    while (st < ks) st <<= 1;
    return st;
}

struct ProblemShape {
    int64_t nnz = 0, nlits = 0, nocc = 0;
    int kmax = 0;
    int64_t n_long = 0;  // rows with more than kLongRow entries (two-state graph kinds)
    bool weighted = false, dense = false;
};

static bool shape_of(const fem_problem *pb, ProblemShape *s, std::string *err) {
    if (!pb) return *err = "problem is NULL", false;
    if (pb->n < 1) return *err = "n must be >= 1", false;
    if (pb->kind < FEM_MAXCUT || pb->kind > FEM_MAXSAT) return *err = "unknown kind", false;
    if (pb->kind == FEM_BMINCUT) {
        if (pb->q < 2 || pb->q > kMaxQ) return *err = "q must be in 2..32 for BMINCUT", false;
    } else if (pb->kind == FEM_MAXSAT && pb->lit_state) {
        if (pb->q < 2 || pb->q > 8) return *err = "q must be in 2..8 for non-Boolean MAXSAT", false;
    } else if (pb->q != 2) {
        return *err = "q must be 2 for MAXCUT / ISING / Boolean MAXSAT", false;
    }
    if (pb->lit_state && pb->kind != FEM_MAXSAT) return *err = "lit_state is for MAXSAT only", false;
    if (pb->node_weight && pb->kind != FEM_BMINCUT) return *err = "node_weight is for BMINCUT only", false;
    if (pb->kind == FEM_MAXSAT) {
        if (pb->m < 1 || !pb->clause_ptr || !pb->lits) return *err = "MAXSAT needs m >= 1, clause_ptr and lits", false;
        if (pb->clause_ptr[0] != 0) return *err = "clause_ptr[0] must be 0", false;
        for (int c = 0; c < pb->m; ++c) {
            const int64_t len = pb->clause_ptr[c + 1] - pb->clause_ptr[c];
            if (len < 1 || len > kMaxClauseLen) return *err = "clause length must be in 1..8", false;
            s->kmax = std::max<int>(s->kmax, (int)len);
        }
        s->nlits = s->nocc = pb->clause_ptr[pb->m];
        if (s->nlits >= (int64_t)1 << 30) return *err = "too many literals", false;
        if (pb->n >= (1 << 29)) return *err = "too many variables", false;
        return true;
    }
    if (pb->kind == FEM_ISING && pb->dense_J) {
        if (pb->row_ptr || pb->col_idx) return *err = "give either dense_J or a CSR, not both", false;
        if (pb->n > 32768) return *err = "dense n too large", false;
        s->dense = true;
        return true;
    }
    if (!pb->row_ptr || (!pb->col_idx && pb->row_ptr[pb->n] != 0)) return *err = "graph kinds need row_ptr and col_idx", false;
    if (pb->row_ptr[0] != 0) return *err = "row_ptr[0] must be 0", false;
    s->nnz = pb->row_ptr[pb->n];
    if (s->nnz < 0 || s->nnz >= (int64_t)1 << 31) return *err = "nnz out of range", false;
    s->weighted = pb->weight != nullptr;
    if (pb->node_weight) {
        if (pb->kind != FEM_BMINCUT) return *err = "node_weight is for BMINCUT only", false;
        for (int i = 0; i < pb->n; ++i) {
            const float v = pb->node_weight[i];
            if (!(v >= 1.f) || v > 1048576.f || v != std::nearbyint(v)) return *err = "node_weight must be integral, in 1 .. 2^20", false;
        }
    }
    if (pb->kind != FEM_BMINCUT)
        for (int i = 0; i < pb->n; ++i)
            if (is_long_row(pb->row_ptr[i + 1] - pb->row_ptr[i], s->nnz, pb->n)) ++s->n_long;
    return true;
}

static Layout make_layout(const fem_problem *pb, const ProblemShape &s, int R_cap) {
    Layout L{};
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t at = o;
        o = align_up(o + bytes);
        return at;
    };
    const int F = (pb->kind == FEM_BMINCUT || (pb->kind == FEM_MAXSAT && pb->lit_state)) ? pb->q : 1;
    const size_t rows = (size_t)pb->n * F + 1;
    const size_t state = rows * (size_t)R_cap * sizeof(float);
    L.row_ptr = take(((size_t)pb->n + 1) * 4);
    L.col = take((size_t)s.nnz * 4);
    L.w = take(s.weighted ? (size_t)s.nnz * 4 : 0);
    L.rowsum = take(s.nnz > 0 || pb->row_ptr ? (size_t)pb->n * 8 : 0);
    L.long_rows = take((size_t)s.n_long * 4);
    L.vw = take(pb->node_weight ? (size_t)pb->n * 4 : 0);
    L.order = take((pb->kind != FEM_BMINCUT && pb->row_ptr) || (pb->kind == FEM_MAXSAT && !pb->lit_state) ? (size_t)pb->n * 4 : 0);
    L.rank = take(pb->kind != FEM_BMINCUT && pb->row_ptr ? (size_t)pb->n * 4 : 0);
    L.J = take(s.dense ? (size_t)pb->n * pb->n * 4 : 0);
    L.Jlo = take(s.dense ? (size_t)pb->n * pb->n * 4 : 0);
    L.glo0 = take(s.dense ? state : 0);
    L.glo1 = take(s.dense ? state : 0);
    const size_t np8 = ((size_t)pb->n + 15) & ~(size_t)15;  // int8 digit planes (k_dense_i8.cu): rows padded to 16 bytes
    L.J8 = take(s.dense ? 3 * (size_t)pb->n * np8 : 0);
    L.gt8_0 = take(s.dense ? 3 * (size_t)R_cap * np8 : 0);
    L.gt8_1 = take(s.dense ? 3 * (size_t)R_cap * np8 : 0);
    L.jscale = take(s.dense ? (size_t)pb->n * 8 : 0);
    L.field = take(s.dense ? 2 * state : 0);  // fp64 in the wide phase
    L.occ_ptr = take(pb->kind == FEM_MAXSAT ? ((size_t)pb->n * F + 1) * 4 : 0);
    L.lit_state = take(pb->lit_state ? (size_t)s.nlits * 4 : 0);
    L.occ = take((size_t)s.nocc * occ_stride(s.kmax) * 4);
    L.clause_ptr = take(pb->kind == FEM_MAXSAT ? ((size_t)pb->m + 1) * 4 : 0);
    L.lits = take((size_t)s.nlits * 4);
    L.h = take(state);
    L.m1 = take(state);
    L.m2 = take(state);
    L.g0 = take(state);
    L.g1 = take(state);
    L.stage = take(state);
    L.hW = take(2 * state);  // wide phase: the same five arrays in fp64
    L.m1W = take(2 * state);
    L.m2W = take(2 * state);
    L.gW0 = take(2 * state);
    L.gW1 = take(2 * state);
    const size_t qR = (size_t)pb->q * R_cap;
    const bool potts = pb->kind == FEM_BMINCUT;
    L.colsum0 = take(potts ? qR * 8 : 0);
    L.colsum1 = take(potts ? qR * 8 : 0);
    L.colsum2 = take(potts ? qR * 8 : 0);
    L.cfg = take((size_t)pb->n * R_cap);
    L.e_part_i = take((size_t)kEnergyChunks * R_cap * 8);
    L.e_part_d = take((size_t)kEnergyChunks * R_cap * 8);
    L.part_part = take(potts ? (size_t)kEnergyChunks * qR * 4 : 0);
    L.e_int = take((size_t)R_cap * 8);
    L.e_real = take((size_t)R_cap * 8);
    L.part = take(qR * 4);
    L.best = take(((size_t)pb->n + 1) * 4);
    L.total = o;
    return L;
}

static bool cuda_ok(Handle *hd, cudaError_t e, const char *what) {
    if (e == cudaSuccess) return true;
    hd->err = std::string(what) + ": " + cudaGetErrorString(e);
    return false;
}

// Persisting L2 set-aside for the state-innermost Potts steps (k_step_potts_si.cu).  The two gather buffers of the replica
// block(s) a launch works on are written / gathered under an access-policy window with the persisting property, so that the
// streamed arrays (h, m1, m2) do not evict them: cfg 2, Rb = 8: 46.3 -> 43.3 us per launch, 0.51 -> 0.55 of the HBM model
// (DESIGN.md section 6).  The set-aside is a DEVICE-wide limit: it is raised when the fp32 steps of a call begin and put
// back (after a synchronize) by fem_result, fem_reset and fem_destroy; while it is raised, other work on the device has
// that much less L2 for ordinary accesses.  Sizes beyond 47% of the L2 are not asked for (measured: 58 MB of 126 fine,
// 66 MB slower than none, 75 MB 1.5x slower).
static void l2_persist_begin(Handle *hd, int blocks_per_launch) {
    if (hd->l2_persist_on || !hd->opt_l2_persist) return;
    const size_t need = 2 * (size_t)blocks_per_launch * (size_t)hd->rows * hd->Rb * sizeof(float);
    if ((double)need > 0.47 * (double)hd->l2_bytes) return;
    size_t prev = 0;
    if (cudaDeviceGetLimit(&prev, cudaLimitPersistingL2CacheSize) != cudaSuccess ||
        cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, std::max(need, prev)) != cudaSuccess) {
        (void)cudaGetLastError();  // not supported here: run without
        return;
    }
    size_t got = 0;
    (void)cudaDeviceGetLimit(&got, cudaLimitPersistingL2CacheSize);
    hd->l2_persist_prev = prev;
    hd->l2_persist_bytes = (int64_t)got;
    hd->l2_persist_on = got >= need;
    if (!hd->l2_persist_on) (void)cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, prev);
}

static void l2_persist_end(Handle *hd, bool synchronize) {
    if (!hd->l2_persist_on) return;
    if (synchronize) (void)cudaStreamSynchronize(hd->stream);
    (void)cudaCtxResetPersistingL2Cache();
    (void)cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, hd->l2_persist_prev);
    (void)cudaGetLastError();
    hd->l2_persist_on = false;
    hd->l2_persist_bytes = 0;
}

static fem_status fail(Handle *hd, fem_status st, const char *msg) {
    if (hd) hd->err = msg;
    else g_create_error = msg;
    return st;
}

// Validate the symmetric CSR and report whether all weights are integral.
static bool validate_graph(const fem_problem *pb, int64_t nnz, bool *integral, int *uniform_deg, int *max_deg, std::string *err) {
    const int n = pb->n;
    *integral = true;
    int64_t d0 = pb->row_ptr[1] - pb->row_ptr[0];
    bool uniform = true;
    for (int i = 0; i < n; ++i) {
        const int64_t a = pb->row_ptr[i], b = pb->row_ptr[i + 1];
        if (b < a || b > nnz) return *err = "row_ptr must be non-decreasing and end at nnz", false;
        if (b - a != d0) uniform = false;
        for (int64_t e = a; e < b; ++e) {
            const int j = pb->col_idx[e];
            if (j < 0 || j >= n) return *err = "column index out of range", false;
            if (j == i) return *err = "self loop", false;
            if (e > a && pb->col_idx[e - 1] >= j) return *err = "columns must be strictly ascending in each row", false;
            const float w = pb->weight ? pb->weight[e] : 1.0f;
            if (!std::isfinite(w)) return *err = "non-finite weight", false;
            if (pb->kind == FEM_BMINCUT && !(w > 0.f)) return *err = "BMINCUT weights must be > 0", false;
            if (w != std::nearbyint(w) || std::fabs(w) > 1e6f) *integral = false;
        }
    }
    // symmetry: every entry (i, j) has its mirror (j, i) with the same weight.  Small graphs (the CSR stays in the host
    // caches): one cursor per row, rows in ascending order -- the mirror of (i, j) is the next unread entry of row j.
    // Large graphs: a binary search in row j (columns are strictly ascending), rows shared out over the host threads (the
    // cursor sweep took 42 ms at cfg 4a, the search 0.75 ms at cfg 0: both inside every end-to-end pass)
    if (nnz <= (int64_t)1 << 20) {
        std::vector<int64_t> cur(pb->row_ptr, pb->row_ptr + n);
        for (int i = 0; i < n; ++i)
            for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                const int j = pb->col_idx[e];
                const int64_t c = cur[j]++;
                if (c >= pb->row_ptr[j + 1] || pb->col_idx[c] != i) return *err = "CSR is not symmetric", false;
                if (pb->weight && pb->weight[c] != pb->weight[e]) return *err = "weights are not symmetric", false;
            }
    } else {
        const unsigned hw = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
        const unsigned nt = hw;
        std::vector<int> bad(nt, 0);  // 0 ok, 1 not symmetric, 2 weights not symmetric
        auto work = [&](unsigned t) {
            const int a = (int)((int64_t)n * t / nt), b = (int)((int64_t)n * (t + 1) / nt);
            for (int i = a; i < b && !bad[t]; ++i)
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                    const int j = pb->col_idx[e];
                    const int32_t *lo = pb->col_idx + pb->row_ptr[j], *hi = pb->col_idx + pb->row_ptr[j + 1];
                    const int32_t *it = std::lower_bound(lo, hi, i);
                    if (it == hi || *it != i) {
                        bad[t] = 1;
                        break;
                    }
                    if (pb->weight && pb->weight[it - pb->col_idx] != pb->weight[e]) {
                        bad[t] = 2;
                        break;
                    }
                }
        };
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < nt; ++t) pool.emplace_back(work, t);
        work(0);
        for (auto &th : pool) th.join();
        for (unsigned t = 0; t < nt; ++t) {
            if (bad[t] == 1) return *err = "CSR is not symmetric", false;
            if (bad[t] == 2) return *err = "weights are not symmetric", false;
        }
    }
    *uniform_deg = (uniform && d0 > 0 && d0 <= 64) ? (int)d0 : 0;
    int64_t mx = 0;
    for (int i = 0; i < n; ++i) mx = std::max<int64_t>(mx, pb->row_ptr[i + 1] - pb->row_ptr[i]);
    *max_deg = (int)std::min<int64_t>(mx, 1 << 30);
    return true;
}

// Replica block size.  Replicas are independent, so a block whose five fp32 state arrays (h, m1, m2 and the
// two gather buffers: 20 B per field) fit in L2 can run its whole anneal out of L2 before the next block
// starts.  opt_replica_block: 0 = choose automatically, >= R = off, else that size.
static void configure_R(Handle *hd, int R) {
    hd->R = R;
    int Rb = R;
    const double per_replica = 20.0 * (double)hd->dp.n * hd->dp.F;
    // (one die's half of the L2, 63 MB of 126: working sets beyond it are served at 9 - 11 TB/s instead of 13 - 17, DESIGN.md
    // section 6; 0.52 rather than 0.5 keeps the 64 MB block of the scale-free workload, measured faster than its 32 MB one)
    const double budget = 0.52 * (double)hd->l2_bytes;
    if (hd->dp.kind == FEM_BMINCUT) {
        // a block must fit the team mapping of the Potts kernel (one variable's lanes inside a warp); among the
        // divisors of R that do, take the requested one, else the largest that is L2-resident, else the smallest
        const int q = hd->dp.q;
        // gathers_fit: the two gather buffers (8 B per field) of the block fit in 45% of L2 even though the streamed
        // arrays do not -- neighbour rows are then served from L2 while h, m1, m2 stream through (evict-first).  The L2
        // of this part is two halves of 63 MB, one per die: measured (profiles/r02_cfg2_step.md),
        // blocks whose gather buffers take more than about one half lose their gather hits (cfg 2: Rb = 16 moves 530 MB
        // of DRAM traffic per launch for 307 MB algorithmic, Rb = 8 moves 204 MB for 154 MB)
        int largest = 1, resident = 0, gathers_fit = 0, smallest_vec = 0;
        for (int d = 1; d <= R; ++d) {
            if (R % d || !potts_block_ok(q, d)) continue;
            largest = d;
            // (Potts: 45%, not the 52% of the two-state kinds -- a 64 MB block of cfg 2 (Rb = 4) does not stay resident in steady
            // state and runs at 0.41 against 0.49 for Rb = 8 with only its gather buffers in L2: profiles/r02_cfg2_step.md)
            if (per_replica * d <= 0.45 * (double)hd->l2_bytes && d % 4 == 0 && (double)hd->dp.n * hd->dp.F * d >= 1.0e6) resident = d;
            if (8.0 * (double)hd->dp.n * hd->dp.F * d <= 0.45 * (double)hd->l2_bytes) gathers_fit = d;
            if (!smallest_vec && d % 2 == 0) smallest_vec = d;
        }
        if (hd->opt_replica_block > 0 && hd->opt_replica_block <= R && R % hd->opt_replica_block == 0 &&
            potts_block_ok(q, (int)hd->opt_replica_block))
            Rb = (int)hd->opt_replica_block;
        else if (per_replica * R <= budget || hd->l2_bytes == 0)
            Rb = largest;
        else
            Rb = resident > 1 ? resident : (gathers_fit > 1 ? gathers_fit : (smallest_vec ? smallest_vec : largest));
    } else if (hd->opt_replica_block > 0) {
        if (hd->opt_replica_block < R && R % hd->opt_replica_block == 0) Rb = (int)hd->opt_replica_block;
    } else if (!hd->dp.J) {  // (the dense kind runs as one block: its tensor maps cover all R replicas)
        if (per_replica * R > budget) {
            const int vec = (R % 4 == 0) ? 4 : 1;
            int best = 0;
            for (int d = vec; d < R; d += vec)
                if (R % d == 0 && per_replica * d <= budget && (double)hd->dp.n * hd->dp.F * d >= 1.0e6) best = d;
            if (best > 0) Rb = best;
        }
    }
    hd->Rb = Rb;
    while ((uint64_t)hd->rows * (uint64_t)hd->Rb >= (1ull << 32)) {  // kernels index a replica block with 32 bits
        int nb = R / hd->Rb + 1;
        while (R % nb || (hd->dp.kind == FEM_BMINCUT && !potts_block_ok(hd->dp.q, R / nb))) ++nb;
        hd->Rb = R / nb;
    }
}

}  // namespace fem

using namespace fem;

extern "C" {

int32_t fem_abi_version(void) { return 4; }

// a5: the two schedules, in double on the host.  beta(0) = beta_min, beta(N-1) = beta_max.
fem_status fem_schedule_inverse_proportional(double T_max, double T_min, int32_t N, double *beta_out) {
    if (N < 1 || !beta_out || !(T_max > 0) || !(T_min > 0) || !std::isfinite(T_max) || !std::isfinite(T_min)) return FEM_EINVAL;
    for (int32_t t = 0; t < N; ++t) {
        const double T = N > 1 ? T_max + (T_min - T_max) * (double)t / (double)(N - 1) : T_max;  // linear in temperature
        beta_out[t] = 1.0 / T;
    }
    return FEM_OK;
}

fem_status fem_schedule_exponential(double beta_min, double beta_max, int32_t N, double *beta_out) {
    if (N < 1 || !beta_out || !(beta_min > 0) || !(beta_max > 0) || !std::isfinite(beta_min) || !std::isfinite(beta_max))
        return FEM_EINVAL;
    const double l0 = std::log(beta_min), l1 = std::log(beta_max);
    for (int32_t t = 0; t < N; ++t) {
        const double x = N > 1 ? (double)t / (double)(N - 1) : 0.0;
        beta_out[t] = std::exp((l1 - l0) * x + l0);
    }
    return FEM_OK;
}

const char *fem_last_error(const fem_handle *h) {
    return h ? reinterpret_cast<const Handle *>(h)->err.c_str() : g_create_error.c_str();
}

size_t fem_workspace_bytes(const fem_problem *problem, int32_t R_cap) {
    ProblemShape s;
    std::string err;
    if (R_cap < 1 || !shape_of(problem, &s, &err)) return 0;
    return make_layout(problem, s, R_cap).total;
}

fem_status fem_create(const fem_problem *pb, int32_t R_cap, void *workspace, size_t workspace_bytes, void *cuda_stream,
                      fem_handle **out) {
    if (!out) return fail(nullptr, FEM_EINVAL, "out is NULL");
    *out = nullptr;
    ProblemShape s;
    std::string err;
    if (R_cap < 1) return fail(nullptr, FEM_EINVAL, "R_cap must be >= 1");
    if (!shape_of(pb, &s, &err)) return fail(nullptr, FEM_EINVAL, err.c_str());
    const Layout L = make_layout(pb, s, R_cap);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255)) return fail(nullptr, FEM_EINVAL, "workspace must be a 256-byte aligned device pointer");
    if (workspace_bytes < L.total) return fail(nullptr, FEM_EINVAL, "workspace too small (see fem_workspace_bytes)");

    Handle *hd = new (std::nothrow) Handle();
    if (!hd) return fail(nullptr, FEM_ENOMEM, "out of host memory");
    hd->pb = *pb;
    hd->pb.row_ptr = nullptr;
    hd->pb.col_idx = nullptr;
    hd->pb.weight = nullptr;
    hd->pb.dense_J = nullptr;
    hd->pb.clause_ptr = nullptr;
    hd->pb.lits = nullptr;
    hd->pb.node_weight = nullptr;
    hd->pb.lit_state = nullptr;
    hd->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    hd->R_cap = R_cap;
    DevProblem &dp = hd->dp;
    dp.kind = pb->kind;
    dp.n = pb->n;
    dp.q = pb->q;
    dp.F = (pb->kind == FEM_BMINCUT || (pb->kind == FEM_MAXSAT && pb->lit_state)) ? pb->q : 1;
    dp.nnz = s.nnz;
    hd->rows = (int64_t)dp.n * dp.F + 1;
    char *base = static_cast<char *>(workspace);
    auto at = [&](size_t off) { return base + off; };

    // host staging vectors must outlive the async copies: they die after the synchronise below
    std::vector<int> h_row, h_occ_ptr, h_occ, h_cptr, h_long, h_ord, h_rank;  // staging of the uploads: alive until the synchronize below
    std::vector<double> h_rowsum;
    bool ok = true;
    bool device_checked = false;
    auto up = [&](void *dst, const void *src, size_t bytes, const char *what) {
        if (!device_checked) {  // argument errors are reported before the device is touched
            device_checked = true;
            int ndev = 0;
            if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
                hd->err = "no CUDA device: libfem_b200 has no CPU fallback";
                ok = false;
            }
        }
        if (ok && bytes) ok = cuda_ok(hd, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, hd->stream), what);
    };

    if (pb->kind == FEM_MAXSAT) {
        const int n = pb->n, m = pb->m;
        const int ks = std::max(1, s.kmax - 1);
        dp.m = m;
        dp.kstride = ks;
        const int kst = occ_stride(s.kmax);
        const int32_t *qs = pb->lit_state;  // non-Boolean SAT: rows are (variable, clause value) pairs
        const int F = dp.F;
        h_occ_ptr.assign((size_t)n * F + 1, 0);
        for (int c = 0; c < m; ++c) {
            for (int64_t x = pb->clause_ptr[c]; x < pb->clause_ptr[c + 1]; ++x) {
                const int lit = pb->lits[x];
                const int v = (lit > 0 ? lit : -lit) - 1;
                if (lit == 0 || v >= n || (qs && lit < 0)) {
                    delete hd;
                    return fail(nullptr, FEM_EINVAL, "literal out of range");
                }
                if (qs && (qs[x] < 0 || qs[x] >= pb->q)) {
                    delete hd;
                    return fail(nullptr, FEM_EINVAL, "lit_state out of range");
                }
                for (int64_t y = pb->clause_ptr[c]; y < x; ++y) {
                    const int l2 = pb->lits[y];
                    if ((l2 > 0 ? l2 : -l2) - 1 == v) {
                        delete hd;
                        return fail(nullptr, FEM_EINVAL, "a clause repeats a variable");
                    }
                }
                h_occ_ptr[(size_t)(qs ? v * F + qs[x] : v) + 1]++;
            }
        }
        for (int64_t i = 0; i < (int64_t)n * F; ++i) h_occ_ptr[(size_t)i + 1] += h_occ_ptr[i];
        // padding: Boolean -- the constant-1 row, read as "p"; non-Boolean -- the row n*q, which holds -1/q so that
        // its factor (1 - 1/q) - D is 1
        h_occ.assign((size_t)s.nocc * kst, qs ? n * F : ((n << 1) | 1));
        std::vector<int> fill(h_occ_ptr.begin(), h_occ_ptr.end() - 1);
        // clause order inside each variable's list == the oracle's summation order.  Large tables: the variables are shared out
        // over host threads, each scanning all clauses for its own range (the scattered 16-byte writes are what costs:
        // 14 ms of every end-to-end pass at cfg 3 with one thread)
        auto fill_range = [&](int vlo, int vhi) {
            for (int c = 0; c < m; ++c) {
                const int64_t a = pb->clause_ptr[c], b = pb->clause_ptr[c + 1];
                for (int64_t x = a; x < b; ++x) {
                    const int lit = pb->lits[x];
                    const int v = (lit > 0 ? lit : -lit) - 1;
                    if (v < vlo || v >= vhi) continue;
                    int *ent = h_occ.data() + (size_t)fill[qs ? v * F + qs[x] : v]++ * kst;
                    int k = 0;
                    for (int64_t y = a; y < b; ++y) {
                        if (y == x) continue;
                        const int l2 = pb->lits[y];
                        if (qs) ent[k++] = (l2 - 1) * F + qs[y];
                        else ent[k++] = (((l2 > 0 ? l2 : -l2) - 1) << 1) | (l2 < 0 ? 1 : 0);
                    }
                    if (!qs && lit > 0) ent[0] |= 0x80000000;
                }
            }
        };
        {
            const unsigned hw = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
            const unsigned nt = s.nlits < 200000 ? 1u : hw;
            std::vector<std::thread> pool;
            for (unsigned t = 1; t < nt; ++t) pool.emplace_back(fill_range, (int)((int64_t)n * t / nt), (int)((int64_t)n * (t + 1) / nt));
            fill_range(0, (int)((int64_t)n / nt));
            for (auto &th : pool) th.join();
        }
        h_cptr.resize((size_t)m + 1);
        for (int c = 0; c <= m; ++c) h_cptr[c] = (int)pb->clause_ptr[c];
        up(at(L.occ_ptr), h_occ_ptr.data(), h_occ_ptr.size() * 4, "upload occ_ptr");
        up(at(L.occ), h_occ.data(), h_occ.size() * 4, "upload occ");
        up(at(L.clause_ptr), h_cptr.data(), h_cptr.size() * 4, "upload clause_ptr");
        up(at(L.lits), pb->lits, (size_t)s.nlits * 4, "upload lits");
        dp.occ_ptr = reinterpret_cast<int *>(at(L.occ_ptr));
        dp.occ = reinterpret_cast<int *>(at(L.occ));
        dp.clause_ptr = reinterpret_cast<int *>(at(L.clause_ptr));
        dp.lits = reinterpret_cast<int *>(at(L.lits));
        if (qs) {
            up(at(L.lit_state), qs, (size_t)s.nlits * 4, "upload lit_state");
            dp.lit_state = reinterpret_cast<int *>(at(L.lit_state));
        }
        hd->integral_weights = true;
        hd->structure_bytes = 4 * ((int64_t)n * F + 1) + 4 * (int64_t)s.nocc * kst;
        if (!qs && n > 1) {
            // processing order of the stepwise kernel: the variables by ascending number of occurrences (counting sort, stable);
            // its threads take them from the end, so the last CTAs of a launch -- its tail -- hold the variables with the
            // fewest occurrences.  Which thread takes which variable changes no arithmetic.
            int mx = 0;
            for (int v = 0; v < n; ++v) mx = std::max(mx, h_occ_ptr[(size_t)v + 1] - h_occ_ptr[v]);
            std::vector<int> cnt((size_t)mx + 2, 0);
            h_ord.resize((size_t)n);
            for (int v = 0; v < n; ++v) cnt[(size_t)(h_occ_ptr[(size_t)v + 1] - h_occ_ptr[v]) + 1]++;
            for (size_t d = 1; d < cnt.size(); ++d) cnt[d] += cnt[d - 1];
            for (int v = 0; v < n; ++v) h_ord[(size_t)cnt[(size_t)(h_occ_ptr[(size_t)v + 1] - h_occ_ptr[v])]++] = v;
            up(at(L.order), h_ord.data(), h_ord.size() * 4, "upload order");
            dp.order = reinterpret_cast<int *>(at(L.order));
        }
        if (!qs) {   // sliced-ELL sizes of the replica-persistent kernel, from the occurrence counts
            hd->dp = dp;
            std::vector<int64_t> optr(h_occ_ptr.begin(), h_occ_ptr.end());
            persist_prepare(hd, optr.data(), nullptr);
        }
    } else if (s.dense) {
        const int n = pb->n;
        for (int i = 0; i < n; ++i)
            if (pb->dense_J[(size_t)i * n + i] != 0.f) {
                delete hd;
                return fail(nullptr, FEM_EINVAL, "dense_J must have a zero diagonal");
            }
        // symmetry and finiteness in 64 x 64 blocks (the transposed element of a block stays in cache: 16.7 M elements at
        // cfg 4b took 60 ms row by column, inside every end-to-end pass)
        constexpr int kBlk = 64;
        for (int i0 = 0; i0 < n; i0 += kBlk)
            for (int j0 = i0; j0 < n; j0 += kBlk)
                for (int i = i0; i < std::min(n, i0 + kBlk); ++i)
                    for (int j = std::max(j0, i + 1); j < std::min(n, j0 + kBlk); ++j)
                        if (pb->dense_J[(size_t)i * n + j] != pb->dense_J[(size_t)j * n + i] || !std::isfinite(pb->dense_J[(size_t)i * n + j])) {
                            delete hd;
                            return fail(nullptr, FEM_EINVAL, "dense_J must be symmetric and finite");
                        }
        up(at(L.J), pb->dense_J, (size_t)n * n * 4, "upload J");
        dp.J = reinterpret_cast<float *>(at(L.J));
        hd->field = reinterpret_cast<float *>(at(L.field));
        hd->Jlo = reinterpret_cast<float *>(at(L.Jlo));
        hd->glo[0] = reinterpret_cast<float *>(at(L.glo0));
        hd->glo[1] = reinterpret_cast<float *>(at(L.glo1));
        hd->J8 = reinterpret_cast<signed char *>(at(L.J8));
        hd->gt8[0] = reinterpret_cast<signed char *>(at(L.gt8_0));
        hd->gt8[1] = reinterpret_cast<signed char *>(at(L.gt8_1));
        hd->jscale = reinterpret_cast<double *>(at(L.jscale));
        hd->i8_np = (n + 15) & ~15;
        if (ok) launch_tc_split(hd);  // J_lo = J - tf32(J) for the 3xTF32 tensor-core path
        hd->integral_weights = false;
        hd->structure_bytes = 4 * (int64_t)n * n;
    } else {
        if (!validate_graph(pb, s.nnz, &hd->integral_weights, &dp.uniform_deg, &dp.max_deg, &err)) {
            delete hd;
            return fail(nullptr, FEM_EINVAL, err.c_str());
        }
        h_row.resize((size_t)pb->n + 1);
        for (int i = 0; i <= pb->n; ++i) h_row[i] = (int)pb->row_ptr[i];
        up(at(L.row_ptr), h_row.data(), h_row.size() * 4, "upload row_ptr");
        up(at(L.col), pb->col_idx, (size_t)s.nnz * 4, "upload col_idx");
        if (s.weighted) up(at(L.w), pb->weight, (size_t)s.nnz * 4, "upload weight");
        dp.row_ptr = reinterpret_cast<int *>(at(L.row_ptr));
        dp.col = reinterpret_cast<int *>(at(L.col));
        dp.w = s.weighted ? reinterpret_cast<float *>(at(L.w)) : nullptr;
        if (pb->kind == FEM_ISING) hd->integral_weights = false;
        hd->structure_bytes = (dp.uniform_deg > 0 ? 0 : 4 * ((int64_t)pb->n + 1)) + (s.weighted ? 8 : 4) * s.nnz;
        // long rows get a CTA each in the stepwise kernel (k_step_q2.cu)
        if (pb->kind != FEM_BMINCUT)
            for (int i = 0; i < pb->n; ++i)
                if (is_long_row(pb->row_ptr[i + 1] - pb->row_ptr[i], s.nnz, pb->n)) h_long.push_back(i);
        if (!h_long.empty()) {
            up(at(L.long_rows), h_long.data(), h_long.size() * 4, "upload long rows");
            dp.long_rows = reinterpret_cast<int *>(at(L.long_rows));
            dp.n_long = (int)h_long.size();
        }
        if (pb->kind != FEM_BMINCUT && dp.uniform_deg == 0 && pb->n > 1) {
            // degree-sorted processing order of the stepwise kernel (counting sort, ascending, stable): a warp's variables
            // then have rows of nearly the same length, so its batched gather loop does no idle iterations on a
            // degree-skewed graph.  Which thread takes which variable changes no arithmetic.
            std::vector<int> cnt((size_t)dp.max_deg + 2, 0);
            std::vector<int> &ord = h_ord;
            ord.resize((size_t)pb->n);
            for (int i = 0; i < pb->n; ++i) cnt[(size_t)(pb->row_ptr[i + 1] - pb->row_ptr[i]) + 1]++;
            for (size_t d = 1; d < cnt.size(); ++d) cnt[d] += cnt[d - 1];
            for (int i = 0; i < pb->n; ++i) ord[(size_t)cnt[(size_t)(pb->row_ptr[i + 1] - pb->row_ptr[i])]++] = i;
            up(at(L.order), ord.data(), ord.size() * 4, "upload order");
            dp.order = reinterpret_cast<int *>(at(L.order));
            h_rank.resize((size_t)pb->n);  // the inverse: the replica-persistent kernel turns columns into positions
            for (int pos = 0; pos < pb->n; ++pos) h_rank[(size_t)ord[(size_t)pos]] = pos;
            up(at(L.rank), h_rank.data(), h_rank.size() * 4, "upload rank");
            dp.rank = reinterpret_cast<int *>(at(L.rank));
        }
        if (pb->kind != FEM_BMINCUT) persist_prepare(hd, pb->row_ptr, dp.order ? h_ord.data() : nullptr);
        dp.vtotal = (double)pb->n;
        if (pb->node_weight) {  // balance-term node weights (S33-S35); pb->node_weight outlives the upload (synchronised below)
            up(at(L.vw), pb->node_weight, (size_t)pb->n * 4, "upload node weights");
            dp.vw = reinterpret_cast<float *>(at(L.vw));
            double tot = 0.0;
            for (int i = 0; i < pb->n; ++i) tot += (double)pb->node_weight[i];
            dp.vtotal = tot;
            hd->structure_bytes += 4 * (int64_t)pb->n;
        }
        {   // sum_j |W_ij| per node, in double in CSR order (the normalisation factors of the manipulated gradients)
            std::vector<double> &rs = h_rowsum;
            rs.assign((size_t)pb->n, 0.0);
            for (int i = 0; i < pb->n; ++i)
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e)
                    rs[i] += std::fabs(pb->weight ? (double)pb->weight[e] : 1.0);
            up(at(L.rowsum), rs.data(), rs.size() * 8, "upload rowsum");
            hd->rowsum = reinterpret_cast<double *>(at(L.rowsum));
        }
    }
    hd->lambda_last = pb->lambda;
    {
        int dev = 0, l2 = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) == cudaSuccess)
            hd->l2_bytes = l2;
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) hd->sm_count = sms;
    }
    hd->h = reinterpret_cast<float *>(at(L.h));
    hd->m1 = reinterpret_cast<float *>(at(L.m1));
    hd->m2 = reinterpret_cast<float *>(at(L.m2));
    hd->g[0] = reinterpret_cast<float *>(at(L.g0));
    hd->g[1] = reinterpret_cast<float *>(at(L.g1));
    hd->stage = reinterpret_cast<float *>(at(L.stage));
    hd->hW = reinterpret_cast<double *>(at(L.hW));
    hd->m1W = reinterpret_cast<double *>(at(L.m1W));
    hd->m2W = reinterpret_cast<double *>(at(L.m2W));
    hd->gW[0] = reinterpret_cast<double *>(at(L.gW0));
    hd->gW[1] = reinterpret_cast<double *>(at(L.gW1));
    hd->colsum[0] = reinterpret_cast<long long *>(at(L.colsum0));
    hd->colsum[1] = reinterpret_cast<long long *>(at(L.colsum1));
    hd->colsum[2] = reinterpret_cast<long long *>(at(L.colsum2));
    {   // |sum_i V_i D_i(s)| < sum_i V_i (= n without node weights): the largest power of two (up to 2^44) that keeps
        // that bound times the scale below 2^62
        int64_t bound = pb->n;
        if (pb->node_weight) {
            bound = 0;
            for (int i = 0; i < pb->n; ++i) bound += (int64_t)pb->node_weight[i];
        }
        int bits = 0;
        while (((int64_t)1 << bits) <= bound) ++bits;
        hd->colsum_scale = std::ldexp(1.0, std::min(44, 62 - bits));
    }
    hd->cfg = reinterpret_cast<int8_t *>(at(L.cfg));
    hd->e_part_i = reinterpret_cast<long long *>(at(L.e_part_i));
    hd->e_part_d = reinterpret_cast<double *>(at(L.e_part_d));
    hd->part_part = reinterpret_cast<int *>(at(L.part_part));
    hd->e_int = reinterpret_cast<long long *>(at(L.e_int));
    hd->e_real = reinterpret_cast<double *>(at(L.e_real));
    hd->part = reinterpret_cast<int *>(at(L.part));
    hd->best = reinterpret_cast<int *>(at(L.best));
    if (ok) ok = cuda_ok(hd, cudaMemsetAsync(hd->part, 0, (size_t)pb->q * R_cap * 4, hd->stream), "memset");
    if (ok) ok = cuda_ok(hd, cudaStreamSynchronize(hd->stream), "fem_create synchronize");
    if (!ok) {
        g_create_error = hd->err;
        delete hd;
        return FEM_ECUDA;
    }
    *out = reinterpret_cast<fem_handle *>(hd);
    return FEM_OK;
}

void fem_destroy(fem_handle *h) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (hd) l2_persist_end(hd, true);
    delete hd;
}

fem_status fem_reset(fem_handle *h) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd) return FEM_EINVAL;
    hd->t_done = 0;
    hd->injected = false;
    hd->gather_valid = false;
    hd->readout_valid = false;
    hd->wide_live = false;
    hd->tc_ready = false;
    hd->tc8_ready = false;
    hd->gather_h = hd->gather_h_want = false;
    l2_persist_end(hd, true);
    return FEM_OK;
}

fem_status fem_set_option(fem_handle *h, const char *key, int64_t value) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !key) return FEM_EINVAL;
    if (hd->t_done != 0 || hd->injected) return fail(hd, FEM_ESTATE, "options can only change before fields exist (fem_reset first)");
    if (!strcmp(key, "replica_block")) {
        if (value < 0) return fail(hd, FEM_EINVAL, "replica_block must be >= 0");
        hd->opt_replica_block = value;
    } else if (!strcmp(key, "steps_per_block")) {
        if (value < 0) return fail(hd, FEM_EINVAL, "steps_per_block must be >= 0");
        hd->opt_steps_per_block = value;
    } else if (!strcmp(key, "tc_tile_n")) {
        if (value != 0 && value != 32 && value != 64 && value != 128 && value != 256)
            return fail(hd, FEM_EINVAL, "tc_tile_n must be 0, 32, 64, 128 or 256");
        hd->opt_tc_tile_n = value;
    } else if (!strcmp(key, "persistent")) {
        if (value < 0 || value > 9) return fail(hd, FEM_EINVAL, "persistent must be 0, 1 or 1 + cluster size");
        hd->opt_persistent = value;
    } else if (!strcmp(key, "persist_chunk")) {
        if (value < 0 || value > 2048) return fail(hd, FEM_EINVAL, "persist_chunk must be 0 .. 2048");
        hd->opt_persist_chunk = value;
    } else if (!strcmp(key, "potts_tma")) {
        if (value < 0 || value > 1) return fail(hd, FEM_EINVAL, "potts_tma must be 0 or 1");
        hd->opt_potts_tma = value;
    } else if (!strcmp(key, "gather_fields")) {
        if (value < -1 || value > 1) return fail(hd, FEM_EINVAL, "gather_fields must be -1, 0 or 1");
        hd->opt_gather_fields = value;
    } else if (!strcmp(key, "tc_debug")) {
        hd->opt_tc_debug = value;
    } else if (!strcmp(key, "tc_cluster")) {
        if (value < 0 || value > 1) return fail(hd, FEM_EINVAL, "tc_cluster must be 0 or 1");
        hd->opt_tc_cluster = value;
    } else if (!strcmp(key, "long_rows")) {
        if (value < 0 || value > 1) return fail(hd, FEM_EINVAL, "long_rows must be 0 or 1");
        hd->opt_long_rows = value;
    } else if (!strcmp(key, "potts_si")) {
        if (value < 0 || value > 1) return fail(hd, FEM_EINVAL, "potts_si must be 0 or 1");
        hd->opt_potts_si = value;
    } else if (!strcmp(key, "l2_persist")) {
        if (value < 0 || value > 1) return fail(hd, FEM_EINVAL, "l2_persist must be 0 or 1");
        hd->opt_l2_persist = value;
    } else if (!strcmp(key, "tensor_cores")) {
        if (value < 0 || value > 2) return fail(hd, FEM_EINVAL, "tensor_cores must be 0, 1 or 2");
        hd->opt_tensor_cores = value;
    } else {
        return fail(hd, FEM_EINVAL, "unknown option");
    }
    return FEM_OK;
}

int64_t fem_get_info(const fem_handle *h, const char *key) {
    const Handle *hd = reinterpret_cast<const Handle *>(h);
    if (!hd || !key) return -1;
    if (!strcmp(key, "launches")) return hd->launches;
    if (!strcmp(key, "tc_launches")) return hd->tc_launches;
    if (!strcmp(key, "tc8_launches")) return hd->tc8_launches;
    if (!strcmp(key, "persist_launches")) return hd->persist_launches;
    if (!strcmp(key, "persist_cluster")) return hd->persist_cluster;
    if (!strcmp(key, "tma_launches")) return hd->tma_launches;
    if (!strcmp(key, "si_launches")) return hd->si_launches;
    if (!strcmp(key, "l2_persist_bytes")) return hd->l2_persist_on ? hd->l2_persist_bytes : 0;
    if (!strcmp(key, "gather_fields")) return hd->gather_h || hd->gather_h_want ? 1 : 0;
    if (!strcmp(key, "t_done")) return hd->t_done;
    if (!strcmp(key, "R")) return hd->R;
    if (!strcmp(key, "replica_block")) return hd->Rb;
    if (!strcmp(key, "nnz")) return hd->dp.kind == FEM_MAXSAT ? hd->pb.m : hd->dp.nnz;
    if (!strcmp(key, "uniform_degree")) return hd->dp.uniform_deg;
    if (!strcmp(key, "max_degree")) return hd->dp.max_deg;
    if (!strcmp(key, "long_rows")) return hd->dp.n_long;
    if (!strcmp(key, "integral_weights")) return hd->integral_weights;
    if (!strcmp(key, "step_bytes")) {
        // algorithmic HBM bytes of one fused step: 24 B per field (read and write h, m1, m2)
        // plus the problem structure once
        // (8 B per moment array the optimiser of the last fem_anneal does not keep less: SGD has no second moment,
        // RMSprop / SGD without momentum no first)
        const int64_t fields = (int64_t)hd->dp.n * hd->dp.F * hd->R;
        return hd->bytes_per_field * fields + hd->structure_bytes;  // (the same 24 B per field in gather-the-fields mode)
    }
    return -1;
}


fem_status fem_set_fields(fem_handle *h, int32_t R, const float *fields) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !fields) return FEM_EINVAL;
    if (R < 1 || R > hd->R_cap) return fail(hd, FEM_EINVAL, "R must be in 1..R_cap");
    configure_R(hd, R);
    const size_t bytes = (size_t)hd->dp.n * hd->dp.F * R * sizeof(float);
    if (!cuda_ok(hd, cudaMemcpyAsync(hd->stage, fields, bytes, cudaMemcpyHostToDevice, hd->stream), "upload fields")) return FEM_ECUDA;
    launch_transpose_in(hd, hd->stage, hd->h);
    if (!cuda_ok(hd, cudaStreamSynchronize(hd->stream), "fem_set_fields")) return FEM_ECUDA;
    hd->t_done = 0;
    hd->injected = true;
    hd->gather_valid = false;
    hd->readout_valid = false;
    hd->wide_live = false;
    hd->tc_ready = false;
    hd->tc8_ready = false;
    hd->gather_h = hd->gather_h_want = false;  // the injected fields are in hd->h
    return FEM_OK;
}

// device-layout array (fp32 `src`, or its fp64 twin `srcW` while the wide phase is live) -> logical host array
static fem_status fetch_state(Handle *hd, const float *src, const double *srcW, float *dst_host) {
    if (hd->R < 1) return fail(hd, FEM_ESTATE, "no fields yet");
    if (hd->wide_live && srcW) launch_transpose_out_wide(hd, srcW, hd->stage);
    else launch_transpose_out(hd, src, hd->stage);
    const size_t bytes = (size_t)hd->dp.n * hd->dp.F * hd->R * sizeof(float);
    if (!cuda_ok(hd, cudaMemcpyAsync(dst_host, hd->stage, bytes, cudaMemcpyDeviceToHost, hd->stream), "download")) return FEM_ECUDA;
    if (!cuda_ok(hd, cudaStreamSynchronize(hd->stream), "synchronize")) return FEM_ECUDA;
    return FEM_OK;
}

fem_status fem_get_fields(fem_handle *h, float *fields) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !fields) return FEM_EINVAL;
    return fetch_state(hd, hd->fields(), hd->hW, fields);
}

fem_status fem_get_moments(fem_handle *h, float *m1, float *m2) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd) return FEM_EINVAL;
    fem_status st = FEM_OK;
    if (m1) st = fetch_state(hd, hd->m1, hd->m1W, m1);
    if (st == FEM_OK && m2) st = fetch_state(hd, hd->m2, hd->m2W, m2);
    return st;
}

static void ensure_gather(Handle *hd) {
    if (hd->gather_valid || (hd->gather_h && !hd->wide_live)) return;  // (gather_h: the fp32 steps gather from the fields themselves)
    StepScalars sc{};
    sc.t = hd->t_done;
    if (hd->dp.kind == FEM_BMINCUT) launch_potts(hd, sc, hd->wide_live, /*step=*/false, 0, hd->R / hd->Rb);
    else if (hd->dp.lit_state) launch_qsat(hd, sc, hd->wide_live, /*step=*/false, 0, hd->R / hd->Rb);
    else launch_prepare_q2(hd, hd->wide_live);
    hd->gather_valid = true;
}

fem_status fem_get_marginals(fem_handle *h, float *marginals) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !marginals) return FEM_EINVAL;
    if (hd->R < 1) return fail(hd, FEM_ESTATE, "no fields yet");
    // the fp32 scratch array (g[cur ^ 1]) is free here: the next step (or the narrowing) overwrites it anyway
    float *scratch = hd->scratch();
    if (hd->dp.F > 1) launch_potts_softmax(hd, scratch);
    else launch_sigmoid(hd, scratch);
    return fetch_state(hd, scratch, nullptr, marginals);
}

fem_status fem_anneal(fem_handle *h, const fem_schedule *sch, int32_t R, uint64_t seed, int32_t stop_after) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !sch) return FEM_EINVAL;
    if (sch->struct_bytes != sizeof(fem_schedule)) return fail(hd, FEM_EINVAL, "fem_schedule.struct_bytes != sizeof(fem_schedule): caller built against another ABI version");
    if (R < 1 || R > hd->R_cap) return fail(hd, FEM_EINVAL, "R must be in 1..R_cap");
    if (sch->steps < 0 || (sch->steps > 0 && !sch->beta)) return fail(hd, FEM_EINVAL, "schedule needs beta[steps]");
    if (stop_after < hd->t_done || stop_after > sch->steps) return fail(hd, FEM_EINVAL, "stop_after must be in [t_done, steps]");
    if ((hd->t_done > 0 || hd->injected) && R != hd->R) return fail(hd, FEM_EINVAL, "R differs from the replicas already in flight");
    if (sch->optimizer < FEM_ADAM || sch->optimizer > FEM_SGD) return fail(hd, FEM_EINVAL, "unknown optimizer");
    if (!(sch->lr > 0) || !(sch->eps >= 0) || !std::isfinite(sch->weight_decay)) return fail(hd, FEM_EINVAL, "bad lr / eps / weight_decay");
    if (sch->optimizer == FEM_ADAM && (!(sch->beta1 >= 0 && sch->beta1 < 1) || !(sch->beta2 >= 0 && sch->beta2 < 1)))
        return fail(hd, FEM_EINVAL, "bad Adam parameters");
    if (sch->optimizer == FEM_RMSPROP && (!(sch->alpha >= 0 && sch->alpha < 1) || !(sch->momentum >= 0)))
        return fail(hd, FEM_EINVAL, "bad RMSprop parameters");
    if (sch->optimizer == FEM_SGD && (!(sch->momentum >= 0) || !(sch->dampening >= 0 && sch->dampening <= 1)))
        return fail(hd, FEM_EINVAL, "bad SGD parameters");
    if (sch->manipulated != 0 && sch->manipulated != 1) return fail(hd, FEM_EINVAL, "manipulated must be 0 or 1");
    if (sch->manipulated && (!(sch->gamma_grad > 0) || !std::isfinite(sch->gamma_grad)))
        return fail(hd, FEM_EINVAL, "gamma_grad must be finite and > 0");
    // the moment arrays and the gather buffers mean different things under another optimiser / gradient mode
    if (hd->t_done > 0 && (sch->optimizer != hd->traj_optimizer || sch->manipulated != hd->traj_manipulated))
        return fail(hd, FEM_EINVAL, "optimizer / manipulated cannot change inside a trajectory (fem_reset first)");
    for (int t = hd->t_done; t < stop_after; ++t)
        if (!(sch->beta[t] > 0) || !std::isfinite(sch->beta[t])) return fail(hd, FEM_EINVAL, "beta[t] must be finite and > 0");

    const int K = std::max(0, sch->precise_steps);
    if (hd->t_done == 0) {
        hd->traj_optimizer = sch->optimizer;
        hd->traj_manipulated = sch->manipulated;
        if (!hd->injected) {
            configure_R(hd, R);
            launch_init_fields(hd, seed, sch->init_scale);
        }
        if (K > 0) {  // wide phase: fp64 arithmetic and fp64 storage for the first K steps
            launch_widen(hd);
            hd->wide_live = true;
        } else {
            launch_zero_moments(hd);
            hd->wide_live = false;
        }
        hd->gather_valid = false;
        hd->tc_ready = false;
        hd->tc8_ready = false;
        hd->gather_h = hd->gather_h_want = false;
    }
    const int nb = hd->R / hd->Rb;
    // one-hot neighbours only where the paper manipulates the gradient (graph kinds with a CSR)
    const bool disc = sch->manipulated && hd->rowsum != nullptr;
    if (hd->gather_valid && hd->gather_disc != disc) hd->gather_valid = false;
    hd->gather_disc = disc;
    if (hd->t_done == 0) {
        // gather-the-fields mode (fixed for the trajectory): sparse two-state graph kinds, exact gradient, regular degree 3
        // or 4 (three or four extra tanh per field), the stepwise fp32 kernel.  Automatic choice: only when the state is
        // streamed from HBM (one replica block, too large for L2), where the 4 B per field of the gather array count.
        const bool shape_ok = (hd->dp.kind == FEM_MAXCUT || (hd->dp.kind == FEM_ISING && !hd->dp.J)) && !disc &&
                              (hd->dp.uniform_deg == 3 || hd->dp.uniform_deg == 4) && hd->Rb % 4 == 0 && !persist_eligible(hd);
        const bool streamed = nb == 1 && 20.0 * (double)hd->dp.n * hd->R > 0.45 * (double)hd->l2_bytes;
        hd->gather_h_want = shape_ok && (hd->opt_gather_fields == 1 || (hd->opt_gather_fields < 0 && streamed));
        hd->gather_h = false;
    }
    hd->plain_adam = sch->optimizer == FEM_ADAM && !sch->manipulated;
    hd->bytes_per_field = 8 + (sch->optimizer == FEM_ADAM || sch->momentum > 0 ? 8 : 0) + (sch->optimizer != FEM_SGD ? 8 : 0);
    auto scalars = [&](int t) {
        StepScalars sc;
        sc.inv_beta = 1.0 / sch->beta[t];
        sc.eps = sch->eps;
        sc.wd = sch->weight_decay;
        sc.opt = sch->optimizer;
        sc.first = t == 0;
        sc.disc = disc;
        sc.gamma = sch->manipulated ? sch->gamma_grad : 1.0;
        if (sch->optimizer == FEM_ADAM) {
            sc.step_size = sch->lr / (1.0 - std::pow(sch->beta1, (double)(t + 1)));
            sc.rsqrt_bc2 = 1.0 / std::sqrt(1.0 - std::pow(sch->beta2, (double)(t + 1)));
            sc.b1 = sch->beta1;
            sc.b2 = sch->beta2;
            sc.one_minus_b1 = 1.0 - sch->beta1;
            sc.one_minus_b2 = 1.0 - sch->beta2;
        } else {
            sc.step_size = sch->lr;
            sc.rsqrt_bc2 = 1.0;
            sc.b1 = sch->momentum;
            sc.b2 = sch->optimizer == FEM_RMSPROP ? sch->alpha : 0.0;
            sc.one_minus_b1 = 1.0 - sch->dampening;
            sc.one_minus_b2 = 1.0 - sc.b2;
        }
        sc.two_lambda = 2.0 * (sch->lambda ? sch->lambda[t] : hd->pb.lambda);
        sc.t = t;
        return sc;
    };
    ensure_gather(hd);
    auto one_step = [&](int t, int b0, int bc) {
        if (hd->dp.kind == FEM_BMINCUT) launch_potts(hd, scalars(t), hd->wide_live, true, b0, bc);
        else if (hd->dp.lit_state) launch_qsat(hd, scalars(t), hd->wide_live, true, b0, bc);
        else launch_step_q2(hd, scalars(t), hd->wide_live, b0, bc);
    };
    const int t0 = hd->t_done;
    int t = t0;
    const bool persist = persist_eligible(hd);
    auto scalars_thunk = [](void *ctx, int tt) { return (*static_cast<decltype(scalars) *>(ctx))(tt); };
    if (persist && hd->wide_live && t < K && t < stop_after) {  // wide phase inside the replica-persistent kernel
        const int te = std::min(stop_after, K);
        if (!cuda_ok(hd, persist_run(hd, true, t, te, scalars_thunk, &scalars), "persistent launch")) return FEM_ECUDA;
        t = te;
    }
    for (; t < stop_after && hd->wide_live && t < K; ++t) {  // wide phase, step-major over all blocks
        one_step(t, 0, nb);
        hd->cur ^= 1;
    }
    if (hd->wide_live && t < stop_after) {  // leave the wide phase only when fp32 steps follow
        launch_narrow(hd, false);
        hd->wide_live = false;
        hd->tc_ready = false;
        hd->tc8_ready = false;
    }
    if (hd->gather_h_want && !hd->gather_h && !hd->wide_live && t < stop_after) {
        // The first fp32 step of a trajectory takes the default path: its gather array is the accurately rounded one
        // (narrowed from the fp64 wide phase, or made from the fields with the double-precision tanh), and the early
        // dynamics amplifies that rounding.  From its output on, the gather array is exactly
        // mag_of(h) in fp32 -- what the gather-the-fields steps recompute -- so the mode switches without changing a bit.
        one_step(t, 0, nb);
        hd->cur ^= 1;
        ++t;
        hd->gather_h = true;
        hd->hpar = hd->cur;  // the fields are in hd->h
    }
    // Potts, q = 4 / 8: the fp32 steps of this call run on state-innermost replica blocks (k_step_potts_si.cu); the
    // arrays are permuted in place here and back below, so nothing outside this call sees the other layout
    const bool si = hd->dp.kind == FEM_BMINCUT && !hd->wide_live && t < stop_after && potts_si_applicable(hd);
    if (si) {
        launch_potts_si_relayout(hd, true);
        hd->si_live = true;
        l2_persist_begin(hd, (nb == 1 || hd->opt_steps_per_block == 1) ? nb : 1);
    }
    if (persist && t < stop_after) {  // small sparse two-state problem: one CTA per replica, all steps in one launch
        if (!cuda_ok(hd, persist_run(hd, false, t, stop_after, scalars_thunk, &scalars), "persistent launch")) return FEM_ECUDA;
        t = stop_after;
    } else if (nb == 1 || hd->opt_steps_per_block == 1) {
        for (; t < stop_after; ++t) {
            one_step(t, 0, nb);
            hd->cur ^= 1;
        }
    } else if (t < stop_after) {
        // replica blocks are independent: run a run of steps on one block while its state is L2-resident
        const int span = hd->opt_steps_per_block > 0 ? (int)hd->opt_steps_per_block : std::max(1, stop_after - t);
        for (int ta = t; ta < stop_after; ta += span) {
            const int tb = std::min(stop_after, ta + span);
            const int cur0 = hd->cur;
            for (int b = 0; b < nb; ++b) {
                hd->cur = cur0;
                for (int tt = ta; tt < tb; ++tt) {
                    one_step(tt, b, 1);
                    hd->cur ^= 1;
                }
            }
            hd->cur = cur0 ^ ((tb - ta) & 1);
        }
    }
    if (si) {
        launch_potts_si_relayout(hd, false);
        hd->si_live = false;
    }
    if (stop_after > t0) {
        hd->lambda_last = sch->lambda ? sch->lambda[stop_after - 1] : hd->pb.lambda;
        hd->readout_valid = false;
    }
    hd->t_done = stop_after;
    if (!cuda_ok(hd, cudaGetLastError(), "kernel launch")) return FEM_ECUDA;
    return FEM_OK;
}

fem_status fem_readout(fem_handle *h) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd) return FEM_EINVAL;
    if (hd->R < 1) return fail(hd, FEM_ESTATE, "no fields yet");
    launch_readout(hd, hd->lambda_last);
    hd->readout_valid = true;
    if (!cuda_ok(hd, cudaGetLastError(), "kernel launch")) return FEM_ECUDA;
    return FEM_OK;
}

fem_status fem_result(fem_handle *h, int32_t *best_replica, int32_t *best_config, int64_t *energy_int, double *energy,
                      int32_t *part_sizes) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd) return FEM_EINVAL;
    if (!hd->readout_valid) {
        fem_status st = fem_readout(h);
        if (st != FEM_OK) return st;
    }
    bool ok = true;
    auto down = [&](void *dst, const void *src, size_t bytes) {
        if (ok && dst) ok = cuda_ok(hd, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, hd->stream), "download result");
    };
    down(best_replica, hd->best, 4);
    down(best_config, hd->best + 1, (size_t)hd->dp.n * 4);
    down(energy_int, hd->e_int, (size_t)hd->R * 8);
    down(energy, hd->e_real, (size_t)hd->R * 8);
    down(part_sizes, hd->part, (size_t)hd->R * hd->dp.q * 4);
    if (ok) ok = cuda_ok(hd, cudaStreamSynchronize(hd->stream), "fem_result synchronize");
    l2_persist_end(hd, false);  // (the stream is idle: give the set-aside back)
    return ok ? FEM_OK : FEM_ECUDA;
}

fem_status fem_get_configs(fem_handle *h, int32_t *cfg) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !cfg) return FEM_EINVAL;
    if (!hd->readout_valid) {
        fem_status st = fem_readout(h);
        if (st != FEM_OK) return st;
    }
    int *logical = reinterpret_cast<int *>(hd->stage);
    launch_cfg_out(hd, logical);
    if (!cuda_ok(hd, cudaMemcpyAsync(cfg, logical, (size_t)hd->dp.n * hd->R * 4, cudaMemcpyDeviceToHost, hd->stream), "download configs")) return FEM_ECUDA;
    if (!cuda_ok(hd, cudaStreamSynchronize(hd->stream), "synchronize")) return FEM_ECUDA;
    return FEM_OK;
}

fem_status fem_energy_of(fem_handle *h, const int32_t *cfg, int32_t count, int64_t *energy_int, double *energy,
                         int32_t *part_sizes) {
    Handle *hd = reinterpret_cast<Handle *>(h);
    if (!hd || !cfg) return FEM_EINVAL;
    if (count < 1 || count > hd->R_cap) return fail(hd, FEM_EINVAL, "count must be in 1..R_cap");
    for (int64_t k = 0; k < (int64_t)count * hd->dp.n; ++k)
        if (cfg[k] < 0 || cfg[k] >= hd->dp.q) return fail(hd, FEM_EINVAL, "state out of range");
    int *logical = reinterpret_cast<int *>(hd->stage);
    bool ok = cuda_ok(hd, cudaMemcpyAsync(logical, cfg, (size_t)count * hd->dp.n * 4, cudaMemcpyHostToDevice, hd->stream), "upload configs");
    if (!ok) return FEM_ECUDA;
    launch_cfg_in(hd, logical, count);
    launch_energy_of(hd, count, hd->lambda_last);
    hd->readout_valid = false;  // the device configuration buffer now holds the caller's configurations
    auto down = [&](void *dst, const void *src, size_t bytes) {
        if (ok && dst) ok = cuda_ok(hd, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, hd->stream), "download energies");
    };
    down(energy_int, hd->e_int, (size_t)count * 8);
    down(energy, hd->e_real, (size_t)count * 8);
    down(part_sizes, hd->part, (size_t)count * hd->dp.q * 4);
    if (ok) ok = cuda_ok(hd, cudaStreamSynchronize(hd->stream), "fem_energy_of synchronize");
    return ok ? FEM_OK : FEM_ECUDA;
}

}  // extern "C"
