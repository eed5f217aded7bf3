// Internal declarations of libfem_b200 (not part of the ABI; see include/fem.h).
//
// Device layout.  R replicas are split into NB = R / Rb replica blocks of
// Rb replicas (Rb = R unless the "replica_block" option is set).  Inside a block a field
// (variable i, state s, replica r) lives at  (i*F + s)*Rb + r  -- replica innermost, so the row
// of a variable is F*Rb contiguous floats and a neighbour gather is one coalesced, vectorised row
// (north_star subsystem 1; the paper's listing keeps replicas outermost).  Every
// per-block array has (n*F + 1) rows: the extra last row of the gather buffers is the constant 1
// that pads short Max-SAT clauses.  Blocks are blk_stride = (n*F+1)*Rb floats apart.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
#include <set>
#include <string>
#include <utility>
#include <vector>

#include "../../include/fem.h"

namespace fem {

constexpr int kThreads = 256;
constexpr int kMaxQ = 32;
constexpr int kMaxClauseLen = 8;
// two-state graph kinds, rows from row_ptr: a "long row" has more than kLongRow entries (the hubs of a degree-skewed graph) --
// the stepwise kernel gives it a whole CTA (k_step_q2.cu) instead of one thread per VEC replicas, and the replica-persistent
// kernel is not used.  Measured on the scale-free workload (n = 1e5, hub degree 1167; us per launch of 3.2 M fields):
// threshold 32 -> 27.5, 64 -> 23.1, 80 -> 21.7, 96 -> 22.0, 128 -> 26.7, 192 -> 34.2.
constexpr int kLongRow = 80;
__host__ __device__ inline bool is_long_row(int64_t deg, int64_t /*nnz*/, int /*n*/) { return deg > kLongRow; }

// Per-step scalars, computed on the host in double and narrowed in-kernel.
struct StepScalars {
    double inv_beta;   // 1 / beta_t
    double step_size;  // lr / (1 - beta1^(t+1))
    double rsqrt_bc2;  // 1 / sqrt(1 - beta2^(t+1))
    double eps, b1, b2, one_minus_b1, one_minus_b2, wd;
    double two_lambda;  // Potts balance term 2*lambda_t
    double gamma;       // gamma_grad (S20); 1 for the exact gradient
    int opt, first, disc;  // optimiser kind, SGD first-step flag, manipulated gradients (see Sc<T>)
    int t;              // step number (the Potts column-sum buffers rotate with it)
};

// Device view of the problem (pointers into the workspace).
struct DevProblem {
    int kind, n, q, F;
    // graph kinds
    const int *row_ptr;  // [n+1]
    const int *col;      // [nnz]
    const float *w;      // [nnz] or nullptr (= +1)
    int uniform_deg;     // > 0 when every row has this many entries
    int max_deg;         // longest row
    int64_t nnz;
    const float *vw;       // BMINCUT: node weights V_i of the balance term (S33-S35), or nullptr (= all 1)
    double vtotal;         // sum_i V_i (= n without node weights)
    const int *rank;       // [n] inverse of `order` (the position of each variable), nullptr with it
    const int *order;      // [n] (Boolean Max-SAT: the variables by ascending number of occurrences.)  Two-state graph kinds with rows of different lengths: the variables sorted by degree (ascending), the
                           // order in which the stepwise kernel's threads take them, so that the variables of a warp have rows of
                           // (nearly) the same length; nullptr = index order
    const int *long_rows;  // [n_long] variables whose row has more than kLongRow entries (two-state graph kinds), ascending
    int n_long;
    const float *J;  // dense Ising, n*n
    // Max-SAT, variable-centric: occurrences of variable i are occ_ptr[i]..occ_ptr[i+1]; occurrence o
    // holds kstride = kmax-1 packed entries (stored with the stride padded to a power of two: 1, 2, 4 or 8 ints): (var << 1 | negated) of the OTHER literals of its clause,
    // padded with (n << 1 | 1) (the constant-1 row); bit 31 of entry 0 = own literal is positive.
    int m, kstride;
    const int *occ_ptr;
    const int *occ;
    const int *clause_ptr;  // [m+1], for the unsat count
    const int *lits;        // signed 1-based
    // non-Boolean SAT (F = q fields per variable): occ_ptr has n*q + 1 entries (occurrences of variable i with clause value s
    // are occ_ptr[i*q+s]..), an occurrence holds the gather ROWS k*q + W_mk of the other variables of its clause, padded with
    // row n*q; lit_state [nlits] is kept for the unsat count
    const int *lit_state;
};

// One replica block's state arrays (block base pointers; a launch with gridDim.y > 1 walks blocks).
// T = float (bulk) or double (wide phase).
template <typename T>
struct BlockArrays {
    T *h, *m1, *m2;
    const T *g_in;  // gathered quantity of step t: m = tanh(h/2) (two-state kinds), D = P - 1/q (Potts)
    T *g_out;       // same for step t+1
    int64_t blk_stride;
    int Rb;
};

struct Handle {
    fem_problem pb{};  // host copy of scalars only (pointers nulled)
    DevProblem dp{};
    cudaStream_t stream = nullptr;
    int R_cap = 0, R = 0, Rb = 0;
    int64_t rows = 0;  // n*F + 1
    bool integral_weights = true;
    // workspace carve-up (device pointers)
    float *h = nullptr, *m1 = nullptr, *m2 = nullptr, *g[2] = {nullptr, nullptr}, *stage = nullptr;
    // wide phase (first precise_steps steps): the same five arrays in fp64
    double *hW = nullptr, *m1W = nullptr, *m2W = nullptr, *gW[2] = {nullptr, nullptr};
    bool wide_live = false;                  // the fp64 arrays hold the current state
    float *field = nullptr;                  // dense Ising: J*m scratch [rows*R_cap] (fp64 in the wide phase: 2x)
    // dense Ising on the tensor cores (k_dense_tc.cu): low parts of J and of the transposed gather buffers
    float *Jlo = nullptr, *glo[2] = {nullptr, nullptr};
    alignas(64) unsigned char tc_maps[6 * 128];  // CUtensorMap x6: J, Jlo, GT[0], GTlo[0], GT[1], GTlo[1]
    int tc_maps_R = -1, tc_maps_bn = -1;     // the maps bake in R (rows of GT) and the tile height bn
    bool tc_ready = false;                   // g[cur]/glo[cur] hold GT / GT_lo of the current fields
    // dense Ising on the int8 tensor-core path (k_dense_i8.cu): digit planes of J and of the transposed magnetisations
    signed char *J8 = nullptr, *gt8[2] = {nullptr, nullptr};  // [3][n][np], [3][R_cap][np] x 2
    double *jscale = nullptr;                // [n] row scales of J (over 64)
    int i8_np = 0;                           // row pitch of the digit planes: n rounded up to 16
    alignas(64) unsigned char tc8_maps[9 * 128];  // CUtensorMap x9: J digits 0..2, GT8[0] digits, GT8[1] digits
    int tc8_maps_R = -1, tc8_maps_bn = -1;
    bool tc8_ready = false, tc8_split_done = false;  // gt8[cur] holds the digits of the current fields; J8 / jscale are made
    int64_t tc8_launches = 0;
    int64_t opt_tc_debug = 0;  // TEMPORARY
    int64_t opt_tc_cluster = 1;  // int8 dense step: 2 x 2 clusters with operand multicast where the grid allows it
    double *rowsum = nullptr;  // graph kinds: sum_j |W_ij| per node (manipulated gradients: c_i, c^f_i, c^a_i)
    int bytes_per_field = 24;  // algorithmic HBM bytes per field per step: read + write of h and of the moments in use
    bool plain_adam = true;    // Adam on the exact gradient: the only update the tcgen05 dense step implements
    bool gather_disc = false;  // the gather buffers hold one-hot values (manipulated gradients), not marginals
    long long *colsum[3] = {nullptr, nullptr, nullptr};  // Potts column sums S[q][R] in fixed point, rotating
    double colsum_scale = 1.0;                            // fixed-point scale (a power of two)
    int8_t *cfg = nullptr;                   // [rows*R_cap]
    long long *e_part_i = nullptr;
    double *e_part_d = nullptr;
    int *part_part = nullptr;
    long long *e_int = nullptr;
    double *e_real = nullptr;
    int *part = nullptr;
    int *best = nullptr;  // [0] = best replica, [1..n] = its configuration
    // "gather the fields" mode of the sparse two-state step (k_step_q2.cu): neighbours are gathered
    // from the fp32 FIELD array and m_j = tanh(h_j / 2) is recomputed per neighbour, so no separate gather array is
    // written (4 B per field per step less).  The step is synchronous, so the fields ping-pong between the arrays
    // h and g[0]: the current ones are in fields() = (cur ^ hpar) & 1 ? g[0] : h; g[1] is the hooks' scratch.
    bool gather_h = false;       // active: the fp32 fields ping-pong, steps gather from them
    bool gather_h_want = false;  // decided at the first step of a trajectory; becomes active after the first fp32 step
    int hpar = 0;
    int64_t opt_gather_fields = -1;  // -1 = automatic (degree <= 4, state streamed from HBM), 0 = never, 1 = wherever it applies
    float *fields() const { return gather_h && ((cur ^ hpar) & 1) ? g[0] : h; }
    float *fields_other() const { return gather_h && ((cur ^ hpar) & 1) ? h : g[0]; }
    float *scratch() const { return gather_h ? g[1] : g[cur ^ 1]; }  // free fp32 array of state size (hooks)
    int cur = 0;          // g[cur] holds the gathered quantity of the current fields
    int t_done = 0;
    int traj_optimizer = 0, traj_manipulated = 0;  // fixed at the first step of a trajectory
    // per-handle (hence per-device) caches of the launch helpers: kernels whose shared-memory attribute is set,
    // and resident-CTA counts from the occupancy calculator, keyed by kernel function (and shared-memory size)
    std::set<const void *> attr_done;
    std::map<std::pair<const void *, size_t>, int> resident_ctas;
    bool injected = false, readout_valid = false, gather_valid = false;
    int64_t opt_replica_block = 0, opt_steps_per_block = 0, opt_tensor_cores = 1, opt_tc_tile_n = 0;
    // small sparse two-state problems: replica-persistent kernel (k_persist_q2.cu).  0 = off, 1 = automatic cluster
    // size, 1 + CS = force clusters of CS CTAs per replica
    int64_t opt_persistent = 1;
    int64_t opt_persist_chunk = 0;  // annealing steps per launch of the persistent kernel (0 = as many as the parameters hold)
    int64_t persist_launches = 0, persist_cluster = 0;
    int64_t opt_potts_tma = 1;    // Potts step with TMA-staged rows (k_step_potts_tma.cu) where it applies
    int64_t tma_launches = 0;
    // Potts step on state-innermost replica blocks (k_step_potts_si.cu): q = 4 / 8, blocks of 4 / 8 / 16 / 32.  The fp32
    // arrays are re-laid out in place for the fp32 steps of one fem_anneal call (si_live) and back before it returns.
    int64_t opt_long_rows = 1;   // 0: long rows stay with one thread per VEC replicas (measurements only)
    int64_t opt_potts_si = 1;
    int64_t opt_l2_persist = 1;     // state-innermost Potts steps: keep the two gather buffers of a replica block in a persisting L2 set-aside
    bool l2_persist_on = false;     // the device limit is raised (fem_api.cu: l2_persist_begin / l2_persist_end)
    size_t l2_persist_prev = 0;     // cudaLimitPersistingL2CacheSize as found
    int64_t l2_persist_bytes = 0;   // set-aside in force while on (info)
    int64_t si_launches = 0;
    bool si_live = false;
    int64_t persist_ell[4] = {-1, -1, -1, -1};  // sliced-ELL entries per CTA for cluster sizes 1, 2, 4, 8
    int sm_count = 148;
    int64_t launches = 0;
    int64_t tc_launches = 0;  // launches of the tcgen05 dense step (k_dense_tc.cu)
    int64_t l2_bytes = 0;  // device L2 size (0 when unknown: no automatic replica blocking)
    int64_t structure_bytes = 0;  // problem-structure bytes one step reads (indices, weights, clause entries)
    double lambda_last = 0.0;     // balance weight of the last executed step (readout uses it)
    std::string err;
};

constexpr int kColBlocks = 592;     // CTAs of a Potts step launch (4 per SM, grid-stride over the variables)
constexpr int kEnergyChunks = 1184;  // readout partials per replica (8 node slots x 148 blocks)

// ---- launchers implemented in the .cu files (all asynchronous on hd->stream) ----
void launch_init_fields(Handle *hd, uint64_t seed, double scale);
void launch_zero_moments(Handle *hd);
void launch_widen(Handle *hd);   // fp32 h -> fp64 hW, zero wide moments
void launch_narrow(Handle *hd, bool fields_only);  // fp64 state -> fp32 arrays
void launch_transpose_in(Handle *hd, const float *logical_dev, float *dst);  // [R][n][F] -> device layout
void launch_transpose_out(Handle *hd, const float *src, float *logical_dev);
void launch_transpose_out_wide(Handle *hd, const double *src, float *logical_dev);
void launch_readout(Handle *hd, double lambda);
void launch_energy_of(Handle *hd, int count, double lambda);  // energies of hd->cfg (count replicas)
void launch_cfg_in(Handle *hd, const int *cfg_logical_dev, int count);
void launch_cfg_out(Handle *hd, int *cfg_logical_dev);

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

}  // namespace fem

namespace fem {
// typed views of the live state arrays
template <typename T> struct StateOf;
template <> struct StateOf<float> {
    static float *h(Handle *d) { return d->fields(); }
    static float *m1(Handle *d) { return d->m1; }
    static float *m2(Handle *d) { return d->m2; }
    static float *g(Handle *d, int k) { return d->g[k]; }
    static float *field(Handle *d) { return d->field; }
};
template <> struct StateOf<double> {
    static double *h(Handle *d) { return d->hW; }
    static double *m1(Handle *d) { return d->m1W; }
    static double *m2(Handle *d) { return d->m2W; }
    static double *g(Handle *d, int k) { return d->gW[k]; }
    static double *field(Handle *d) { return reinterpret_cast<double *>(d->field); }
};
}  // namespace fem
