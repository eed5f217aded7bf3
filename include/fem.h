/*
 * fem.h -- C ABI of the B200-native Free-Energy Machine annealing path (arxiv 2412.09285).
 *
 * The library runs, entirely in hand-written CUDA kernels for sm_100a, the replica-parallel
 * mean-field annealing step of the paper (Fig.2): marginals from local fields,
 * the explicit gradient of F_MF = U_MF(P) - S_MF(P)/beta (S18-S30), an Adam
 * update of the fields under an annealed beta, for R
 * independent replicas, followed by rounding (Eq.4), the integer energy of every
 * replica (Eq.6-8) and the best-replica reduction (Eq.5).
 * There is no CPU fallback: without a CUDA device every compute entry point fails with FEM_ECUDA.
 *
 * Conventions
 *   - All pointers in fem_problem / fem_schedule and all result pointers are HOST pointers.
 *     fem_create validates the problem on the host (symmetry, self loops, repeated variables: the
 *     checks need the host copy) and uploads the device formats it builds (CSR / padded occurrence
 *     table / split dense couplings).  The only DEVICE pointer in this ABI is `workspace`
 *     (caller-owned, e.g. a torch tensor).  DESIGN.md section 3 (R15) records this reading.
 *   - Coupling convention (R1): the exact gradient is that of U_MF = <E>, every edge counted
 *     ONCE (Eq.6/Eq.9): dU/dp_i = sum_j W_ij m_j for MAXCUT, -sum_j W_ij P_j(s) for
 *     BMINCUT.  The paper's listing and S21/S24/S26 count ordered pairs (a factor 2 on the coupling
 *     term), so hyper-parameters quoted for the listing correspond to HALF the
 *     temperature here (beta_here = 2 beta_listing for the coupling/entropy balance; for BMINCUT also
 *     lambda_here = 2 lambda_listing).  The manipulated gradients (S25/S27/S30) carry no such factor
 *     and are implemented term for term.
 *   - The library allocates no device memory: all state lives in the caller's workspace, which
 *     must stay alive and untouched until fem_destroy.  Host-side bookkeeping is freed by
 *     fem_destroy.
 *   - Work is enqueued on the caller's CUDA stream (`cuda_stream` is a cudaStream_t cast to
 *     void*, NULL = legacy default stream).  fem_anneal and fem_readout are ASYNCHRONOUS; the
 *     fem_result / fem_get_* / fem_energy_of calls synchronise that stream before returning.
 *     Host arrays passed to fem_anneal are consumed before it returns.
 *   - Logical host layouts are replica-outermost, row-major: fields h[R][n][F] with F = q for
 *     FEM_BMINCUT and F = 1 otherwise (the two-state kinds keep h_i = h_i(+1) - h_i(-1),
 *     PAPER.md:661); configurations cfg[R][n] with states 0..q-1 (two-state: 1 <=> sigma = +1 /
 *     Boolean true).  The device layout (replica-innermost n x R rows) is private.
 *   - Determinism: same inputs and seed give bit-identical outputs run to run (no float atomics).
 *   - Errors: status codes only.  Argument errors are reported synchronously (FEM_EINVAL) and
 *     leave the handle unchanged; CUDA errors surface as FEM_ECUDA at the call that observes
 *     them.  fem_last_error returns a static or handle-owned message.
 */
#ifndef FEM_H_
#define FEM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fem_handle fem_handle; /* opaque */

typedef enum { FEM_OK = 0, FEM_EINVAL = 1, FEM_ENOMEM = 2, FEM_ECUDA = 3, FEM_ESTATE = 4 } fem_status;

typedef enum {
    FEM_MAXCUT = 0,  /* E = -sum_{(i,j) in E} W_ij [1 - delta(s_i,s_j)]          Eq.6  */
    FEM_ISING = 1,   /* E = -sum_{i<j} J_ij s_i s_j, s = +-1 (sparse CSR or dense) PAPER.md:43         */
    FEM_BMINCUT = 2, /* E = cut + lambda * sum_k (n_k - n/q)^2, q-state Potts      Eq.7  */
    FEM_MAXSAT = 3   /* E = number of unsatisfied clauses                          Eq.8  */
} fem_kind;

/* Problem description; every pointer is a HOST pointer, read only during fem_create /
 * fem_workspace_bytes. */
typedef struct {
    int32_t kind; /* fem_kind */
    int32_t n;    /* number of variables, >= 1 */
    int32_t q;    /* states per variable: 2 for MAXCUT / ISING / MAXSAT, 2..32 for BMINCUT */
    /* Graph kinds (MAXCUT, BMINCUT, sparse ISING): symmetric CSR with BOTH directions stored, no self
     * loops, no repeated entries, columns ascending in each row.  weight NULL = all +1.  For BMINCUT
     * the weights must be > 0. */
    const int64_t *row_ptr; /* [n+1] */
    const int32_t *col_idx; /* [row_ptr[n]] */
    const float *weight;    /* [row_ptr[n]] or NULL */
    /* ISING only, instead of the CSR: dense n*n row-major symmetric couplings, zero diagonal. */
    const float *dense_J;
    /* MAXSAT: m clauses; clause c holds lits[clause_ptr[c] .. clause_ptr[c+1]) as signed 1-based
     * literals (+v = variable v, -v = NOT v, i.e. W_mi = 1 / 0 in Eq.8).  A clause must not repeat a
     * variable (S15); clause length 1..8. */
    int32_t m;
    const int64_t *clause_ptr; /* [m+1] */
    const int32_t *lits;       /* [clause_ptr[m]] */
    double lambda;             /* BMINCUT balance weight when the schedule gives no per-step lambda */
    /* ---- ABI version 4 ---- BMINCUT only, optional: node weights V_i of the balance term (S33-S35),
     * HOST [n], integral values in 1 .. 2^20, or NULL (= all 1).  The energy becomes cut + lambda * sum_k (sum_{i in k} V_i
     * - sum_i V_i / q)^2, part_sizes the sums of V_i per part, and the balance term of the gradient
     * 2 lambda V_i [sum_j V_j P_j(s) - V_i P_i(s)].  Must be NULL for the other kinds. */
    const float *node_weight;
    /* MAXSAT only, optional: non-Boolean SAT ("W_mi has q > 2 states").  HOST [clause_ptr[m]]: lit_state[x] =
     * W_mi in 0..q-1 of literal slot x, lits[x] = +v (1-based variable, must be > 0), q in 2..8.  Every variable then has q
     * states and q fields (softmax marginals; logical layouts as for BMINCUT, F = q), the energy is the number of clauses in
     * which NO variable takes its clause value (Eq.8), and the gradient is S28 per state with the
     * chain rule S20.  NULL = Boolean SAT (q must be 2). */
    const int32_t *lit_state;
} fem_problem;

/* Annealing schedule and optimiser.  Step t = 0..steps-1 uses beta[t]
 * (inverse temperature) and Adam step count t+1. */
typedef struct {
    uint32_t struct_bytes; /* sizeof(fem_schedule) as the CALLER compiled it; fem_anneal returns FEM_EINVAL on any other
                            * value, so a caller built against another ABI version is never read out of bounds */
    int32_t steps;
    const double *beta;   /* HOST [steps], > 0 */
    const double *lambda; /* HOST [steps] per-step balance weight, or NULL */
    double lr, beta1, beta2, eps, weight_decay; /* Adam, PyTorch semantics */
    double init_scale;     /* h(0) = init_scale * N(0,1); used when fields were not injected */
    int32_t precise_steps; /* wide phase: the first K steps keep state AND arithmetic in fp64, then the state is
                            * rounded to fp32 once and the rest of the anneal is fp32 */
    /* ---- ABI version 2: the optimisers and gradient manipulations the paper benchmarks with ---- */
    int32_t optimizer;     /* fem_optimizer; FEM_ADAM uses lr, beta1, beta2, eps, weight_decay above.
                            * FEM_RMSPROP (torch.optim.RMSprop, not centered): lr, alpha, eps, weight_decay, momentum.
                            * FEM_SGD (torch.optim.SGD, no Nesterov): lr, momentum, dampening, weight_decay */
    double alpha;          /* RMSprop smoothing constant, in [0, 1) */
    double momentum;       /* RMSprop / SGD momentum, >= 0 */
    double dampening;      /* SGD dampening, in [0, 1] */
    int32_t manipulated;   /* 0: exact gradient of F_MF (gamma_grad ignored).  1: manipulated gradients:
                            * MAXCUT / sparse ISING S29-S30: neighbours enter as sgn(m_j), coupling term times
                            * c_i = 1 / sum_j |W_ij| (Ising: |2 J_ij|); BMINCUT S27: one-hot neighbours e_j, c^f_i =
                            * q / sum_j W_ij on the cut term and lambda * c^a_i, c^a_i = q / sqrt(sum_j W_ij), on the balance
                            * term; MAXSAT and dense ISING: no modification; all kinds: g^h times gamma_grad (S20) */
    double gamma_grad;     /* > 0; used when manipulated = 1 */
} fem_schedule;

typedef enum { FEM_ADAM = 0, FEM_RMSPROP = 1, FEM_SGD = 2 } fem_optimizer;

/* The two annealing schedules of the paper, t = 0..N-1, written to HOST beta_out[N]:
 *   inverse-proportional (linear in temperature): T(t) = T_max + (T_min - T_max) t/(N-1), beta(t) = 1/T(t)
 *   exponential: beta(t) = exp((ln beta_max - ln beta_min) t/(N-1) + ln beta_min)
 * so that beta(0) = beta_min = 1/T_max and beta(N-1) = beta_max = 1/T_min; N = 1 gives beta(0).
 * FEM_EINVAL: N < 1, NULL output, non-positive or non-finite endpoints.  Pure host arithmetic in double. */
fem_status fem_schedule_inverse_proportional(double T_max, double T_min, int32_t N, double *beta_out);
fem_status fem_schedule_exponential(double beta_min, double beta_max, int32_t N, double *beta_out);

/* Bytes of device workspace fem_create needs for this problem with up to R_cap replicas
 * (0 on invalid arguments).  Pure host arithmetic. */
size_t fem_workspace_bytes(const fem_problem *problem, int32_t R_cap);

/* Validate `problem`, build the device formats inside `workspace` (DEVICE pointer, 256-byte aligned,
 * >= fem_workspace_bytes) and return a handle.  Synchronises `cuda_stream` once at the end.
 * FEM_EINVAL: bad sizes, asymmetric CSR, self loop, unsorted/repeated column, literal out of range,
 * repeated variable in a clause, q out of range, workspace too small or misaligned. */
fem_status fem_create(const fem_problem *problem, int32_t R_cap, void *workspace, size_t workspace_bytes,
                      void *cuda_stream, fem_handle **out);

/* Run steps [t_done, stop_after) of the schedule on R replicas, where t_done is the number of steps
 * already run since the last reset.  When t_done == 0 the Adam moments are zeroed and, unless fields
 * were injected with fem_set_fields, the fields are drawn from `seed` with the counter-based
 * generator of DESIGN.md section 3 (R4).  Asynchronous.  FEM_EINVAL: R < 1 or > R_cap, R differs
 * from the R of the steps already run, stop_after outside [t_done, steps], beta[t] <= 0, struct_bytes !=
 * sizeof(fem_schedule), or optimizer / manipulated differ from the ones the trajectory was started with (t_done > 0).
 * One launch of the fused step kernel per step and replica block (one iteration
 * of the listing's loop). */
fem_status fem_anneal(fem_handle *h, const fem_schedule *schedule, int32_t R, uint64_t seed, int32_t stop_after);

/* Forget the trajectory: t_done = 0, injected fields dropped. */
fem_status fem_reset(fem_handle *h);

/* Enqueue rounding (Eq.4), per-replica energies (Eq.6-8) and the best-replica argmin (Eq.5) on the
 * current fields.  Asynchronous; results stay on the device until fem_result. */
fem_status fem_readout(fem_handle *h);

/* Run fem_readout if the fields changed since the last one, copy the results to the host and
 * synchronise.  Any output pointer may be NULL.
 *   best_replica : argmin_a energy[a], lowest a on ties
 *   best_config  : HOST [n], configuration of the best replica
 *   energy_int   : HOST [R]; MAXCUT: -cut, BMINCUT: cut, MAXSAT: unsat count, with weights rounded to
 *                  nearest integer (exact when they are integral); ISING: 0
 *   energy       : HOST [R] fp64; MAXCUT/MAXSAT: (double)energy_int when weights are integral, else the
 *                  fp64 sum; BMINCUT: cut + lambda*sum_k (n_k - n/q)^2; ISING: -sum_{i<j} J_ij s_i s_j
 *   part_sizes   : HOST [R][q] (BMINCUT; zeros otherwise) */
fem_status fem_result(fem_handle *h, int32_t *best_replica, int32_t *best_config, int64_t *energy_int,
                      double *energy, int32_t *part_sizes);

/* ---- parity hooks (logical layouts, HOST pointers, synchronous) ---- */
fem_status fem_set_fields(fem_handle *h, int32_t R, const float *fields /* [R][n][F] */); /* resets t_done */
fem_status fem_get_fields(fem_handle *h, float *fields /* [R][n][F] */);
fem_status fem_get_moments(fem_handle *h, float *m1, float *m2 /* [R][n][F] each, may be NULL */);
/* marginals computed on the device from the current fields; two-state kinds: [R][n] = P(state 1) */
fem_status fem_get_marginals(fem_handle *h, float *marginals /* [R][n][F] */);
fem_status fem_get_configs(fem_handle *h, int32_t *cfg /* [R][n] */);
/* energies of caller-supplied configurations (count <= R_cap), same definitions as fem_result */
fem_status fem_energy_of(fem_handle *h, const int32_t *cfg /* [count][n] */, int32_t count, int64_t *energy_int,
                         double *energy, int32_t *part_sizes /* [count][q] or NULL */);

/* Tuning knobs (all optional): "replica_block" (replicas per L2-resident block; 0 = chosen from the
 * device's L2 size, the default; >= R = no blocking), "steps_per_block" (steps run on one replica
 * block before moving to the next; 0 = the whole anneal per block, the default; 1 = step-major).
 * Results do not depend on either (replicas are independent).  Dense ISING only: "tensor_cores"
 * (1 = the default: the int8 digit step on tcgen05 (kind::i8, k_dense_i8.cu) where it applies -- R a multiple of 32, plain
 * Adam on the exact gradient --, else the 3xTF32 step; 2 = the 3xTF32 step (kind::tf32; n % 4 == 0); 0 = CUDA-core GEMM)
 * and "tc_tile_n" (replica columns per tensor-core tile: 0 = default, 32/64/128, and 256 for the 3xTF32 step only),
 * "tc_cluster" (int8 step: 1 = 2 x 2 thread-block clusters with operand multicast where the tile grid is even in both
 * directions, the default; 0 = off; bit-identical either way).
 * "persistent" (small sparse MAXCUT / ISING / MAXSAT problems with few enough replicas to run in at most three
 * waves of clusters: 1 = replica-persistent cluster kernel where the problem fits, the default; 0 = one launch per step; 1 + CS = force clusters of CS = 1, 2, 4 or 8 CTAs per replica),
 * "persist_chunk" (annealing steps per launch of that kernel: 0 = as many as its parameters hold, 2048 in fp32, the default;
 * 1 .. 2048 = at most that many; no effect on the result) and
 * "long_rows" (two-state graph kinds: 1 = rows with many entries are summed by a CTA each in a fixed order, the default;
 * 0 = one thread per row as for short rows -- this one does change the summation order of those rows),
 * "potts_si" (BMINCUT, q = 4 or 8, replica blocks of 4 / 8 / 16 / 32 with n a multiple of 32 / block: 1 = fp32 steps on
 * state-innermost replica blocks, k_step_potts_si.cu, the default; 0 = off),
 * "l2_persist" (state-innermost Potts steps: 1 = the two gather buffers of the replica block(s) a launch works on are kept
 * in a persisting L2 set-aside under an access-policy window while h, m1, m2 stream past them, the default, used when both
 * fit in 47% of the L2; 0 = off.  The set-aside is the DEVICE-wide limit cudaLimitPersistingL2CacheSize: fem_anneal raises it
 * when such steps begin, and fem_result, fem_reset and fem_destroy put the old value back after synchronising; while it is
 * raised, other work on the device has that much less L2 for ordinary accesses.  A cache policy: no bit of the result
 * changes),
 * "potts_tma" (BMINCUT shapes the state-innermost kernel does not take, or with "potts_si" = 0: 1 = rows staged by bulk
 * asynchronous copies where the shape allows, the default; 0 = register path).  Apart from "long_rows" and
 * the three "tensor_cores" modes (different roundings of the dense product) none of them changes a single bit of the
 * results.  Unknown key: FEM_EINVAL. */
fem_status fem_set_option(fem_handle *h, const char *key, int64_t value);
/* Introspection for benchmarks: "launches" (kernels enqueued so far), "tc_launches" (of which tcgen05
 * dense steps; "tc8_launches": of those, int8 digit steps), "l2_persist_bytes" (persisting L2 set-aside in force, 0 when none), "persist_launches", "persist_cluster" (CTAs per replica of the persistent kernel),
 * "tma_launches" (TMA-staged Potts steps), "si_launches" (state-innermost Potts steps), "t_done", "R", "replica_block", "nnz", "uniform_degree",
 * "max_degree", "long_rows" (rows of a two-state graph kind with more than 80 entries:
 * the stepwise kernel gives each
 * a CTA of its own), "integral_weights", "step_bytes" (algorithmic HBM bytes of one fused step of the last schedule's optimiser,
 * DESIGN.md section 6).  Unknown key: -1. */
int64_t fem_get_info(const fem_handle *h, const char *key);

/* Measurement helper (not on the hot path): L2 -> SM read rate of the current device in GB/s.  `buffer` is a DEVICE
 * pointer (16-byte aligned) to `bytes` (1 MiB .. 96 MiB, a multiple of 16; it is overwritten with zeros), read `repeats`
 * times from all SMs with 16-byte loads that bypass L1, timed with CUDA events on `cuda_stream`; synchronous.  bench.py
 * compares the L2-resident Max-SAT step (cfg 3) with this roof.  FEM_EINVAL on bad arguments, FEM_ECUDA without a device. */
fem_status fem_probe_l2_read(void *buffer, size_t bytes, int32_t repeats, void *cuda_stream, double *gigabytes_per_second);

/* Measurement helper (not on the hot path): rate in GB/s at which all SMs gather pseudo-random rows of `row_bytes` (64, 128,
 * 256 or 512) out of a DEVICE buffer of `bytes` (1 MiB .. 1 GiB, a multiple of 512; overwritten with zeros), 8 independent
 * rows in flight per warp, `repeats` iterations per warp -- the access pattern of the neighbour gathers (a2).  With the
 * buffer size as the parameter it shows where the two-die L2 stops serving a working set at full rate (DESIGN.md section 6:
 * bench.py reports it at 32 MiB and at the footprint of cfg 2's replica block).  Synchronous; FEM_EINVAL / FEM_ECUDA as above. */
fem_status fem_probe_l2_gather(void *buffer, size_t bytes, int32_t row_bytes, int32_t repeats, void *cuda_stream,
                               double *gigabytes_per_second);

/* Cut values without any allocation (Eq.6: cut(sigma) = sum over edges (i, j), i < j, of W_ij [sigma_i != sigma_j]),
 * for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * No handle, no workspace: the per-chunk partial sums that fem_energy_of keeps in the caller's workspace live in a
 * file-scope static __device__ array of FEM_CUT_STATIC_SCRATCH_BYTES (2 MiB), which every GPU that loads the library holds
 * until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it enqueues two
 * kernels on `cuda_stream` and returns without synchronising (the first call on a device also looks up the array's device
 * address, once: make that call before capturing a graph).
 *   All pointers are DEVICE pointers on the CURRENT device, owned by the caller and neither checked nor kept:
 *   n        number of nodes (>= 1)
 *   row_ptr  int32 [n + 1], col_idx int32 [nnz]: the symmetric CSR of fem_problem (both directions of every edge, columns
 *            ascending, no self loops); weight float [nnz] or NULL (= 1), rounded to the nearest integer per edge as in the
 *            readout (a7)
 *   sigma    int8 [n][count], configuration innermost: sigma[i * count + a] in {0, 1} is node i of configuration a
 *   count    configurations, 1 .. FEM_CUT_STATIC_MAX_COUNT
 *   cut      int64 [count], written: for the same graph and configurations fem_energy_of reports energy_int = -cut
 * Returns FEM_EINVAL (count beyond the maximum: split the batch; n or count < 1; a null pointer) or FEM_ECUDA, with the reason
 * in fem_cut_static_error() (per host thread).  Every call on a device shares the scratch array and finds the previous call's
 * contents in it; nothing in it has to start at zero (each call writes every partial it reads).  Calls whose kernels may
 * overlap on the GPU (streams without an ordering between them) RACE on it: order them on one stream or by events. */
#define FEM_CUT_STATIC_MAX_COUNT 4096
#define FEM_CUT_STATIC_SCRATCH_BYTES (2u << 20)
fem_status fem_cut_static(int32_t n, const int32_t *row_ptr, const int32_t *col_idx, const float *weight, const int8_t *sigma,
                          int32_t count, int64_t *cut, void *cuda_stream);
const char *fem_cut_static_error(void);

const char *fem_last_error(const fem_handle *h); /* h may be NULL: last create-time error */
void fem_destroy(fem_handle *h);
int32_t fem_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FEM_H_ */
