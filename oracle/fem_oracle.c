/*
 * fem_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-pass, double-precision CPU restatement of the Free-Energy
 * Machine (FEM) annealing path of arxiv 2412.09285, written from PAPER.md only.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2412_09285_b200/csrc/ and neither includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  Every function cites the passage of PAPER.md it restates.
 *
 * Readings of the paper where it is silent or inconsistent are the ones listed in
 * DESIGN.md section 3 (R1..R12); the ones that matter here:
 *   R1  edge-once coupling: U_MF is the expectation of the integer energy
 *       (Eq.6/Eq.9), not the ordered-pair double count of the
 *       listing.
 *   R2  bMinCut energy reported as cut + lambda*sum_k (n_k - n/q)^2; it differs from
 *       Eq.7 by the constant lambda*(n - n^2/q).
 *   R3  rounding from the final fields h(N); ties -> lowest state index.
 *   R4  initial fields 0.001*N(0,1) from a counter-based generator (below).
 *   R5  Adam as published (Kingma & Ba), eps outside the bias-corrected sqrt,
 *       weight decay added to the gradient (PyTorch's Adam).
 *
 * Logical layouts (host, row-major):  fields h[R][n][F] with F = q for the Potts
 * kind and F = 1 for the two-state kinds (MaxCut / Ising / Max-SAT keep the single
 * field h_i = h_i(+1) - h_i(-1));  configurations cfg[R][n] int32.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   femo_free_energy / femo_grad_h : central finite differences of F; torch autograd
 *                                    on the paper's F; sum_s g^h_i(s) = 0; q=2 softmax
 *                                    path == sigmoid path; mean-field fixed point S40
 *   femo_marginals / entropy       : closed forms at h=0, shift invariance, saturation
 *   femo_adam                      : torch.optim.Adam (float64, CPU)
 *   femo_schedule_*                : endpoints, 1/linspace
 *   femo_energy                    : brute-force enumeration, saturation U_MF == E
 *   femo_anneal                    : brute-force optima on n<=20
 *   femo_rmsprop / femo_sgd        : torch.optim.RMSprop / torch.optim.SGD (float64, CPU)
 *   femo_grad_h_manipulated        : the general-q S25 + S20 form written out in numpy (S29/S30 are its
 *                                    two-state reduction); saturated fields reduce it to the exact
 *                                    gradient on row-normalised weights; sum_s g^h_i(s) = 0; brute-force optima
 *   femo_init_fields               : moments / reproducibility only (a generator, not a
 *                                    formula of the paper)
 *   Solution quality against the paper's tables (G-set, K2000, Walshaw, MaxSAT-2016):
 *   parity unpinned -- those instances are not available.
 *
 * Build:  gcc -O2 -ffp-contract=off -fPIC -shared [-fopenmp] fem_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define FEMO_MAXCUT 0  /* E = -sum_{(i,j) in E} W_ij [1 - delta(s_i,s_j)]   Eq.6 */
#define FEMO_ISING 1   /* E = -sum_{i<j} W_ij s_i s_j, s = +-1    */
#define FEMO_BMINCUT 2 /* E = cut + lambda * balance                        Eq.7 */
#define FEMO_MAXSAT 3  /* E = number of unsatisfied clauses                 Eq.8 */

typedef struct {
    int32_t kind, n, q;
    /* graph kinds: symmetric CSR, both directions stored, no self loops */
    const int64_t *row_ptr;
    const int32_t *col_idx;
    const double *weight; /* NULL = all +1 */
    /* ISING only, optional: dense n*n row-major symmetric J with zero diagonal */
    const double *dense_J;
    /* MAXSAT: m clauses; lits are signed 1-based: +v = variable v, -v = NOT v */
    int32_t m;
    const int64_t *clause_ptr;
    const int32_t *lits;
    /* BMINCUT only, optional: node weights V_i > 0 of the balance term (S33-S35); NULL = all 1 */
    const double *node_weight;
    /* MAXSAT only, optional: non-Boolean SAT ("W_mi has q > 2 states").  lit_state[x] = W_mi in 0..q-1 of the
     * x-th literal slot, lits[x] = +v (1-based variable); every variable then has q states and q fields (softmax marginals,
     * PAPER.md:76), and E = sum_m prod_{i in dm} [1 - delta(W_mi, sigma_i)] (Eq.8).  NULL = Boolean SAT. */
    const int32_t *lit_state;
} femo_problem;

typedef struct {
    double lr, beta1, beta2, eps, weight_decay;
} femo_adam_cfg;

/* q fields per variable for the Potts kind and for non-Boolean SAT, one (h(+1) - h(-1)) otherwise */
static int multistate(const femo_problem *pb) { return pb->kind == FEMO_BMINCUT || (pb->kind == FEMO_MAXSAT && pb->lit_state); }
int32_t femo_fields_per_var(const femo_problem *pb) { return multistate(pb) ? pb->q : 1; }

/* ------------------------------------------------------------------------------------------
 * Marginals from fields.  P_i(s) = exp h_i(s) / sum_s' exp h_i(s');
 * two states: P_i = sigmoid(h_i), h_i = h_i(+1) - h_i(-1).
 * ---------------------------------------------------------------------------------------- */
static double sigmoid(double x) {
    if (x >= 0.0) return 1.0 / (1.0 + exp(-x));
    double e = exp(x);
    return e / (1.0 + e);
}

static double logsumexp(const double *h, int q) {
    double mx = h[0];
    for (int s = 1; s < q; ++s)
        if (h[s] > mx) mx = h[s];
    double z = 0.0;
    for (int s = 0; s < q; ++s) z += exp(h[s] - mx);
    return mx + log(z);
}

/* one replica: h[n*F] -> P[n*F]; two-state kinds return P_i = P_i(state 1) */
void femo_marginals(const femo_problem *pb, const double *h, double *P) {
    int n = pb->n;
    if (!multistate(pb)) {
        for (int i = 0; i < n; ++i) P[i] = sigmoid(h[i]);
        return;
    }
    int q = pb->q;
    for (int i = 0; i < n; ++i) {
        double lse = logsumexp(h + (size_t)i * q, q);
        for (int s = 0; s < q; ++s) P[(size_t)i * q + s] = exp(h[(size_t)i * q + s] - lse);
    }
}

/* ------------------------------------------------------------------------------------------
 * Mean-field entropy S_MF = -sum_i sum_s P_i(s) ln P_i(s)   (S2),
 * with ln P taken from the fields (ln P_i(s) = h_i(s) - logsumexp h_i), never log(P).
 * ---------------------------------------------------------------------------------------- */
static double entropy_two_state(double h) {
    /* ln p = -log1p(exp(-h)), ln(1-p) = -log1p(exp(h)) */
    double p = sigmoid(h), r = sigmoid(-h);
    double lnp = (h >= 0.0) ? -log1p(exp(-h)) : h - log1p(exp(h));
    double lnr = (h <= 0.0) ? -log1p(exp(h)) : -h - log1p(exp(-h));
    return -(p * lnp + r * lnr);
}

double femo_entropy(const femo_problem *pb, const double *h) {
    double S = 0.0;
    int n = pb->n;
    if (!multistate(pb)) {
        for (int i = 0; i < n; ++i) S += entropy_two_state(h[i]);
        return S;
    }
    int q = pb->q;
    for (int i = 0; i < n; ++i) {
        const double *hi = h + (size_t)i * q;
        double lse = logsumexp(hi, q);
        for (int s = 0; s < q; ++s) S -= exp(hi[s] - lse) * (hi[s] - lse);
    }
    return S;
}

static double wgt(const femo_problem *pb, int64_t e) { return pb->weight ? pb->weight[e] : 1.0; }
static double nodew(const femo_problem *pb, int i) { return pb->node_weight ? pb->node_weight[i] : 1.0; }

/* ------------------------------------------------------------------------------------------
 * Mean-field internal energy U_MF(P), one replica (reading R1: every edge once).
 *   MaxCut  (S6,  PAPER.md:417):  U = -sum_{(i,j) in E} W_ij sum_s P_i(s)[1 - P_j(s)]
 *   Ising   (S36): U = -1/2 sum_{i,j} W_ij m_i m_j,  m_i = P_i(+1) - P_i(-1)
 *   bMinCut (S11; balance() PAPER.md:536):
 *           U = sum_E W_ij sum_s P_i(s)[1 - P_j(s)] + lambda sum_s [(sum_i P_i(s))^2 - sum_i P_i(s)^2]
 *               + lambda (n - n^2/q)                                  (constant of reading R2)
 *           with node weights V_i (S33): P_i(s) -> V_i P_i(s) in both sums of the balance term, and
 *           the constant becomes lambda (sum_i V_i^2 - (sum_i V_i)^2 / q), so that one-hot marginals still give
 *           exactly cut + lambda sum_k (sum_{i in k} V_i - sum_i V_i / q)^2
 *   MaxSAT  (S16):  U = sum_m prod_{i in dm} [1 - P_i(W_mi)]
 * ---------------------------------------------------------------------------------------- */
double femo_internal_energy(const femo_problem *pb, const double *h, double lambda) {
    int n = pb->n;
    double U = 0.0;
    double *P = (double *)malloc(sizeof(double) * (size_t)n * femo_fields_per_var(pb));
    femo_marginals(pb, h, P);
    if (pb->kind == FEMO_MAXCUT) {
        for (int i = 0; i < n; ++i)
            for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                int j = pb->col_idx[e];
                if (j <= i) continue; /* each edge once */
                /* sum over the two states: p_i(1-p_j) + (1-p_i)p_j */
                double pi = P[i], pj = P[j], ri = sigmoid(-h[i]), rj = sigmoid(-h[j]);
                U -= wgt(pb, e) * (pi * rj + ri * pj);
            }
    } else if (pb->kind == FEMO_ISING) {
        if (pb->dense_J) {
            for (int i = 0; i < n; ++i)
                for (int j = i + 1; j < n; ++j)
                    U -= pb->dense_J[(size_t)i * n + j] * tanh(0.5 * h[i]) * tanh(0.5 * h[j]);
        } else {
            for (int i = 0; i < n; ++i)
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                    int j = pb->col_idx[e];
                    if (j <= i) continue;
                    U -= wgt(pb, e) * tanh(0.5 * h[i]) * tanh(0.5 * h[j]);
                }
        }
    } else if (pb->kind == FEMO_BMINCUT) {
        int q = pb->q;
        for (int i = 0; i < n; ++i)
            for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                int j = pb->col_idx[e];
                if (j <= i) continue;
                double same = 0.0;
                for (int s = 0; s < q; ++s) same += P[(size_t)i * q + s] * P[(size_t)j * q + s];
                U += wgt(pb, e) * (1.0 - same);
            }
        for (int s = 0; s < q; ++s) {
            double col = 0.0, sq = 0.0;
            for (int i = 0; i < n; ++i) {
                double vp = nodew(pb, i) * P[(size_t)i * q + s];
                col += vp;
                sq += vp * vp;
            }
            U += lambda * (col * col - sq);
        }
        double v1 = 0.0, v2 = 0.0;
        for (int i = 0; i < n; ++i) {
            v1 += nodew(pb, i);
            v2 += nodew(pb, i) * nodew(pb, i);
        }
        U += lambda * (v2 - v1 * v1 / (double)q);
    } else if (pb->lit_state) { /* non-Boolean SAT, S16 with q states: U = sum_m prod_i [1 - P_i(W_mi)] */
        int q = pb->q;
        for (int c = 0; c < pb->m; ++c) {
            double prod = 1.0;
            for (int64_t x = pb->clause_ptr[c]; x < pb->clause_ptr[c + 1]; ++x)
                prod *= 1.0 - P[(size_t)(pb->lits[x] - 1) * q + pb->lit_state[x]];
            U += prod;
        }
    } else { /* MAXSAT */
        for (int c = 0; c < pb->m; ++c) {
            double prod = 1.0;
            for (int64_t x = pb->clause_ptr[c]; x < pb->clause_ptr[c + 1]; ++x) {
                int lit = pb->lits[x];
                int v = (lit > 0 ? lit : -lit) - 1;
                /* literal false with probability 1-p (positive literal) or p (negated) */
                prod *= (lit > 0) ? sigmoid(-h[v]) : sigmoid(h[v]);
            }
            U += prod;
        }
    }
    free(P);
    return U;
}

/* F_MF = U_MF - S_MF / beta   (S1; Eq.3) */
double femo_free_energy(const femo_problem *pb, const double *h, double beta, double lambda) {
    return femo_internal_energy(pb, h, lambda) - femo_entropy(pb, h) / beta;
}

/* ------------------------------------------------------------------------------------------
 * Explicit gradient g^h = dF_MF/dh, one replica, gamma_grad = 1, exact g^p (no manipulation).
 *
 * Potts kind: g^p_i(s) from S26 in the edge-once reading,
 *     g^p_i(s) = -sum_j W_ij P_j(s) + 2 lambda [S_s - P_i(s)] + (1/beta)[ln P_i(s) + 1],
 *   with node weights (S34): 2 lambda V_i [sum_j V_j P_j(s) - V_i P_i(s)] for the balance part,
 * then the chain rule S20:
 *     g^h_i(s) = P_i(s) [ g^p_i(s) - sum_s' P_i(s') g^p_i(s') ].
 * Two-state kinds: S29 with c_i = 1 and P_j in place of e_j,
 *     g^h_i = [ dU/dp_i + (1/beta) ln(p_i/(1-p_i)) ] p_i (1 - p_i),   ln(p/(1-p)) = h_i,
 *   MaxCut : dU/dp_i = sum_j W_ij (2 p_j - 1) = sum_j W_ij m_j          (S21/S30)
 *   Ising  : dU/dp_i = 2 dU/dm_i = -2 sum_j W_ij m_j                    (S36/S39)
 *   MaxSAT : dU/dp_i = sum_{m ni i} s_mi prod_{k in dm, k != i} u_mk     (S28)
 *            u_mk = probability literal k of clause m is false; s_mi = -1 (positive) / +1 (negated)
 * ---------------------------------------------------------------------------------------- */
void femo_grad_h(const femo_problem *pb, const double *h, double beta, double lambda, double *g) {
    int n = pb->n;
    if (pb->kind == FEMO_BMINCUT) {
        int q = pb->q;
        double *P = (double *)malloc(sizeof(double) * (size_t)n * q);
        double *col = (double *)calloc((size_t)q, sizeof(double));
        double *gp = (double *)malloc(sizeof(double) * (size_t)q);
        femo_marginals(pb, h, P);
        for (int i = 0; i < n; ++i)
            for (int s = 0; s < q; ++s) col[s] += nodew(pb, i) * P[(size_t)i * q + s];
        for (int i = 0; i < n; ++i) {
            const double *hi = h + (size_t)i * q;
            const double *Pi = P + (size_t)i * q;
            double lse = logsumexp(hi, q);
            double Vi = nodew(pb, i);
            for (int s = 0; s < q; ++s) {
                double f = 0.0;
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e)
                    f += wgt(pb, e) * P[(size_t)pb->col_idx[e] * q + s];
                gp[s] = -f + 2.0 * lambda * Vi * (col[s] - Vi * Pi[s]) + (hi[s] - lse + 1.0) / beta;
            }
            double gbar = 0.0;
            for (int s = 0; s < q; ++s) gbar += Pi[s] * gp[s];
            for (int s = 0; s < q; ++s) g[(size_t)i * q + s] = Pi[s] * (gp[s] - gbar);
        }
        free(P);
        free(col);
        free(gp);
        return;
    }
    if (pb->kind == FEMO_MAXSAT && pb->lit_state) {
        /* non-Boolean SAT: S28 per state, dU/dP_i(s) = -sum_{m ni i, W_mi = s} prod_{k != i} [1 - P_k(W_mk)],
         * g^p_i(s) = dU/dP_i(s) + (1/beta)[ln P_i(s) + 1], then the chain rule S20 */
        int q = pb->q;
        double *P = (double *)malloc(sizeof(double) * (size_t)n * q);
        double *dP = (double *)calloc((size_t)n * q, sizeof(double));
        femo_marginals(pb, h, P);
        for (int c = 0; c < pb->m; ++c) {
            int64_t a = pb->clause_ptr[c], b = pb->clause_ptr[c + 1];
            for (int64_t x = a; x < b; ++x) {
                double loo = 1.0; /* leave-one-out product, by multiplication only */
                for (int64_t y = a; y < b; ++y)
                    if (y != x) loo *= 1.0 - P[(size_t)(pb->lits[y] - 1) * q + pb->lit_state[y]];
                dP[(size_t)(pb->lits[x] - 1) * q + pb->lit_state[x]] -= loo;
            }
        }
        for (int i = 0; i < n; ++i) {
            const double *hi = h + (size_t)i * q;
            const double *Pi = P + (size_t)i * q;
            double lse = logsumexp(hi, q);
            double gbar = 0.0;
            for (int s = 0; s < q; ++s) gbar += Pi[s] * (dP[(size_t)i * q + s] + (hi[s] - lse + 1.0) / beta);
            for (int s = 0; s < q; ++s)
                g[(size_t)i * q + s] = Pi[s] * (dP[(size_t)i * q + s] + (hi[s] - lse + 1.0) / beta - gbar);
        }
        free(P);
        free(dP);
        return;
    }
    double *dU = (double *)calloc((size_t)n, sizeof(double));
    if (pb->kind == FEMO_MAXCUT || pb->kind == FEMO_ISING) {
        double *mag = (double *)malloc(sizeof(double) * (size_t)n);
        for (int i = 0; i < n; ++i) mag[i] = tanh(0.5 * h[i]); /* m_i = 2P_i - 1 */
        double sign = (pb->kind == FEMO_MAXCUT) ? 1.0 : -2.0;
        for (int i = 0; i < n; ++i) {
            double f = 0.0;
            if (pb->kind == FEMO_ISING && pb->dense_J) {
                for (int j = 0; j < n; ++j) f += pb->dense_J[(size_t)i * n + j] * mag[j];
            } else {
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e)
                    f += wgt(pb, e) * mag[pb->col_idx[e]];
            }
            dU[i] = sign * f;
        }
        free(mag);
    } else { /* MAXSAT, S28 */
        for (int c = 0; c < pb->m; ++c) {
            int64_t a = pb->clause_ptr[c], b = pb->clause_ptr[c + 1];
            for (int64_t x = a; x < b; ++x) {
                double loo = 1.0; /* leave-one-out product, by multiplication only */
                for (int64_t y = a; y < b; ++y) {
                    if (y == x) continue;
                    int lit = pb->lits[y];
                    int v = (lit > 0 ? lit : -lit) - 1;
                    loo *= (lit > 0) ? sigmoid(-h[v]) : sigmoid(h[v]);
                }
                int lit = pb->lits[x];
                int v = (lit > 0 ? lit : -lit) - 1;
                dU[v] += (lit > 0) ? -loo : loo;
            }
        }
    }
    for (int i = 0; i < n; ++i) g[i] = (dU[i] + h[i] / beta) * sigmoid(h[i]) * sigmoid(-h[i]);
    free(dU);
}

/* ------------------------------------------------------------------------------------------
 * Adam (ref.[29] of the paper), step counter t >= 1:
 *   g  <- g + wd * h
 *   m1 <- b1 m1 + (1-b1) g ;  m2 <- b2 m2 + (1-b2) g^2
 *   h  <- h - lr * [m1/(1-b1^t)] / ( sqrt(m2/(1-b2^t)) + eps )
 * ---------------------------------------------------------------------------------------- */
void femo_adam(const femo_adam_cfg *cfg, int32_t t, int64_t count, double *h, double *m1, double *m2, const double *g) {
    double bc1 = 1.0 - pow(cfg->beta1, (double)t);
    double bc2 = 1.0 - pow(cfg->beta2, (double)t);
    for (int64_t k = 0; k < count; ++k) {
        double gk = g[k] + cfg->weight_decay * h[k];
        m1[k] = cfg->beta1 * m1[k] + (1.0 - cfg->beta1) * gk;
        m2[k] = cfg->beta2 * m2[k] + (1.0 - cfg->beta2) * gk * gk;
        double mhat = m1[k] / bc1;
        double vhat = m2[k] / bc2;
        h[k] -= cfg->lr * mhat / (sqrt(vhat) + cfg->eps);
    }
}

/* ------------------------------------------------------------------------------------------
 * Manipulated gradients: what the paper benchmarks with.
 * The marginals of the NEIGHBOURS are replaced by their one-hot vectors e_j ("discretization",
 * PAPER.md:626), the coupling term is normalised per node, and gamma_grad scales the result.
 *
 * Two-state graph kinds, S29/S30:
 *     g^h_i = gamma [ c_i sum_j W_ij sgn(m_j) + h_i/beta ] p_i (1 - p_i),   c_i = 1 / sum_j |W_ij|
 *   (S30 writes gamma/4 (1 - m_i^2); p(1-p) = (1 - m^2)/4.)  sgn(m_j) = sgn(h_j), sgn(0) = 0.
 *   Ising: the same with dU/dp_i = -2 sum_j J_ij m_j (see femo_grad_h), i.e. W_ij -> -2 J_ij, and
 *   c_i = 1 / sum_j |2 J_ij| so that the normalised coupling term stays within [-1, 1] as PAPER.md:630 states.
 * Potts kind, S27 taken literally (coefficient lambda, not 2 lambda, on the balance term):
 *     ghat^p_i(s) = -c^f_i sum_j W_ij e_j(s) + lambda c^a_i [ sum_j e_j(s) - e_i(s) ] + (1/beta)[ln P_i(s) + 1]
 *     c^f_i = q / sum_j W_ij,  c^a_i = q / sqrt(sum_j W_ij)
 *   with node weights (S35): lambda c^a_i V_i [ sum_j V_j e_j(s) - V_i e_i(s) ] for the balance part,
 *   then S20:  g^h_i(s) = gamma P_i(s) [ ghat^p_i(s) - sum_s' P_i(s') ghat^p_i(s') ].
 *   e_j = one-hot of argmax_s h_j(s), ties -> lowest state (the rounding rule R3).
 * Max-SAT: the paper makes no modification: exact gradient times gamma.
 * Nodes without neighbours have no coupling term; their c is taken as 0 (reading R13).
 * ---------------------------------------------------------------------------------------- */
void femo_grad_h_manipulated(const femo_problem *pb, const double *h, double beta, double lambda, double gamma,
                             double *g) {
    int n = pb->n;
    if (pb->kind == FEMO_MAXSAT || (pb->kind == FEMO_ISING && pb->dense_J)) {
        femo_grad_h(pb, h, beta, lambda, g);
        for (int64_t i = 0; i < (int64_t)n * femo_fields_per_var(pb); ++i) g[i] *= gamma;
        return;
    }
    if (pb->kind == FEMO_BMINCUT) {
        int q = pb->q;
        double *P = (double *)malloc(sizeof(double) * (size_t)n * q);
        int *hot = (int *)malloc(sizeof(int) * (size_t)n);
        double *cnt = (double *)calloc((size_t)q, sizeof(double));
        double *gp = (double *)malloc(sizeof(double) * (size_t)q);
        femo_marginals(pb, h, P);
        for (int i = 0; i < n; ++i) {
            int best = 0;
            for (int s = 1; s < q; ++s)
                if (h[(size_t)i * q + s] > h[(size_t)i * q + best]) best = s;
            hot[i] = best;
            cnt[best] += nodew(pb, i);
        }
        for (int i = 0; i < n; ++i) {
            const double *hi = h + (size_t)i * q;
            const double *Pi = P + (size_t)i * q;
            double lse = logsumexp(hi, q);
            double rowsum = 0.0;
            for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) rowsum += wgt(pb, e);
            double cf = rowsum > 0.0 ? (double)q / rowsum : 0.0;
            double ca = rowsum > 0.0 ? (double)q / sqrt(rowsum) : 0.0;
            for (int s = 0; s < q; ++s) {
                double f = 0.0;
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e)
                    if (hot[pb->col_idx[e]] == s) f += wgt(pb, e);
                double ei = (hot[i] == s) ? 1.0 : 0.0;
                double Vi = nodew(pb, i);
                gp[s] = -cf * f + lambda * ca * Vi * (cnt[s] - Vi * ei) + (hi[s] - lse + 1.0) / beta;
            }
            double gbar = 0.0;
            for (int s = 0; s < q; ++s) gbar += Pi[s] * gp[s];
            for (int s = 0; s < q; ++s) g[(size_t)i * q + s] = gamma * Pi[s] * (gp[s] - gbar);
        }
        free(P);
        free(hot);
        free(cnt);
        free(gp);
        return;
    }
    /* MaxCut / sparse Ising */
    double scale = (pb->kind == FEMO_MAXCUT) ? 1.0 : -2.0;
    for (int i = 0; i < n; ++i) {
        double f = 0.0, l1 = 0.0;
        for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
            double hj = h[pb->col_idx[e]];
            double sg = (hj > 0.0) ? 1.0 : (hj < 0.0 ? -1.0 : 0.0);
            f += scale * wgt(pb, e) * sg;
            l1 += fabs(scale * wgt(pb, e));
        }
        double c = l1 > 0.0 ? 1.0 / l1 : 0.0;
        g[i] = gamma * (c * f + h[i] / beta) * sigmoid(h[i]) * sigmoid(-h[i]);
    }
}

/* ------------------------------------------------------------------------------------------
 * RMSprop and SGD with momentum ("the Python
 * implementations of these optimizers as provided by PyTorch", tuned: lr, weight decay, momentum,
 * dampening (SGD); lr, weight decay, momentum, alpha (RMSprop); everything else PyTorch's default:
 * RMSprop eps = 1e-8 added OUTSIDE the square root, not centered; SGD without Nesterov).
 *   RMSprop:  g <- g + wd h;  v <- alpha v + (1-alpha) g^2;  d = g / (sqrt(v) + eps);
 *             momentum > 0:  b <- momentum b + d;  h <- h - lr b      else  h <- h - lr d
 *   SGD:      g <- g + wd h;  momentum > 0:  b <- g at the first step, b <- momentum b + (1-dampening) g after;
 *             h <- h - lr b   (momentum = 0: h <- h - lr g)
 * m1 holds the momentum buffer b, m2 the running square average v.  t is the 1-based step count.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t kind; /* 0 Adam, 1 RMSprop, 2 SGD */
    double lr, beta1, beta2, eps, weight_decay; /* Adam: beta1, beta2 */
    double alpha, momentum, dampening;          /* RMSprop: alpha, momentum; SGD: momentum, dampening */
} femo_opt_cfg;

void femo_rmsprop(const femo_opt_cfg *cfg, int64_t count, double *h, double *m1, double *m2, const double *g) {
    for (int64_t k = 0; k < count; ++k) {
        double gk = g[k] + cfg->weight_decay * h[k];
        m2[k] = cfg->alpha * m2[k] + (1.0 - cfg->alpha) * gk * gk;
        double d = gk / (sqrt(m2[k]) + cfg->eps);
        if (cfg->momentum > 0.0) {
            m1[k] = cfg->momentum * m1[k] + d;
            h[k] -= cfg->lr * m1[k];
        } else {
            h[k] -= cfg->lr * d;
        }
    }
}

void femo_sgd(const femo_opt_cfg *cfg, int32_t t, int64_t count, double *h, double *m1, const double *g) {
    for (int64_t k = 0; k < count; ++k) {
        double gk = g[k] + cfg->weight_decay * h[k];
        if (cfg->momentum > 0.0) {
            m1[k] = (t == 1) ? gk : cfg->momentum * m1[k] + (1.0 - cfg->dampening) * gk;
            h[k] -= cfg->lr * m1[k];
        } else {
            h[k] -= cfg->lr * gk;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Annealing schedules, t = 0..N-1.
 *   inverse-proportional: T(t) = T_max + (T_min - T_max) t/(N-1), beta = 1/T
 *   exponential         : beta(t) = exp( (ln bmax - ln bmin) t/(N-1) + ln bmin )
 * ---------------------------------------------------------------------------------------- */
void femo_schedule_inverse_proportional(double T_max, double T_min, int32_t N, double *beta) {
    for (int t = 0; t < N; ++t) {
        double T = (N > 1) ? T_max + (T_min - T_max) * (double)t / (double)(N - 1) : T_max;
        beta[t] = 1.0 / T;
    }
}

void femo_schedule_exponential(double beta_min, double beta_max, int32_t N, double *beta) {
    for (int t = 0; t < N; ++t) {
        double x = (N > 1) ? (double)t / (double)(N - 1) : 0.0;
        beta[t] = exp((log(beta_max) - log(beta_min)) * x + log(beta_min));
    }
}

/* ------------------------------------------------------------------------------------------
 * Initial fields h = scale * N(0,1), reading R4: a counter-based
 * generator on the logical index c = (a*n + i)*F + s so that replica a does not depend on R.
 *   mix(z): z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31
 *   x  = mix(seed + G),  G = 0x9E3779B97F4A7C15
 *   r1 = mix(x + (2c+1) G), r2 = mix(x + (2c+2) G)
 *   U1 = ((r1>>11) + 1) 2^-53 in (0,1],  U2 = (r2>>11) 2^-53 in [0,1)
 *   z  = sqrt(-2 ln U1) cos(2 pi U2);  h = (float)(scale * z)     (rounded to fp32, stored as double)
 * ---------------------------------------------------------------------------------------- */
static uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

void femo_init_fields(uint64_t seed, int32_t R, int32_t n, int32_t F, double scale, double *h) {
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    uint64_t x = mix64(seed + G);
    int64_t total = (int64_t)R * n * F;
    for (int64_t c = 0; c < total; ++c) {
        uint64_t r1 = mix64(x + (2ULL * (uint64_t)c + 1ULL) * G);
        uint64_t r2 = mix64(x + (2ULL * (uint64_t)c + 2ULL) * G);
        double U1 = ((double)(r1 >> 11) + 1.0) * 0x1.0p-53;
        double U2 = (double)(r2 >> 11) * 0x1.0p-53;
        double z = sqrt(-2.0 * log(U1)) * cos(6.283185307179586476925286766559 * U2);
        h[c] = (double)(float)(scale * z);
    }
}

/* ------------------------------------------------------------------------------------------
 * One synchronous FEM step for all replicas: marginals of every variable
 * from h(t), gradient at P(t), then Adam with step count t+1.  lambda is this step's value.
 * ---------------------------------------------------------------------------------------- */
void femo_step(const femo_problem *pb, int32_t R, double *h, double *m1, double *m2, int32_t t, double beta,
               double lambda, const femo_adam_cfg *adam) {
    int64_t per = (int64_t)pb->n * femo_fields_per_var(pb);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int a = 0; a < R; ++a) {
        double *g = (double *)malloc(sizeof(double) * (size_t)per);
        femo_grad_h(pb, h + a * per, beta, lambda, g);
        femo_adam(adam, t + 1, per, h + a * per, m1 + a * per, m2 + a * per, g);
        free(g);
    }
}

/* steps t_begin .. t_end-1 of an anneal with schedule beta[0..N-1]; lambda_t may be NULL */
void femo_anneal(const femo_problem *pb, int32_t R, double *h, double *m1, double *m2, const double *beta,
                 const double *lambda_t, double lambda, int32_t t_begin, int32_t t_end, const femo_adam_cfg *adam) {
    for (int t = t_begin; t < t_end; ++t)
        femo_step(pb, R, h, m1, m2, t, beta[t], lambda_t ? lambda_t[t] : lambda, adam);
}

/* The same synchronous step with the section 8(f) choices: optimiser kind and exact (manipulated = 0) or
 * manipulated gradients (manipulated = 1, with gamma_grad).  manipulated = 0 ignores gamma (exact gradient). */
void femo_step_ex(const femo_problem *pb, int32_t R, double *h, double *m1, double *m2, int32_t t, double beta,
                  double lambda, const femo_opt_cfg *opt, int32_t manipulated, double gamma) {
    int64_t per = (int64_t)pb->n * femo_fields_per_var(pb);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int a = 0; a < R; ++a) {
        double *g = (double *)malloc(sizeof(double) * (size_t)per);
        if (manipulated) femo_grad_h_manipulated(pb, h + a * per, beta, lambda, gamma, g);
        else femo_grad_h(pb, h + a * per, beta, lambda, g);
        if (opt->kind == 0) {
            femo_adam_cfg ac = {opt->lr, opt->beta1, opt->beta2, opt->eps, opt->weight_decay};
            femo_adam(&ac, t + 1, per, h + a * per, m1 + a * per, m2 + a * per, g);
        } else if (opt->kind == 1) {
            femo_rmsprop(opt, per, h + a * per, m1 + a * per, m2 + a * per, g);
        } else {
            femo_sgd(opt, t + 1, per, h + a * per, m1 + a * per, g);
        }
        free(g);
    }
}

void femo_anneal_ex(const femo_problem *pb, int32_t R, double *h, double *m1, double *m2, const double *beta,
                    const double *lambda_t, double lambda, int32_t t_begin, int32_t t_end, const femo_opt_cfg *opt,
                    int32_t manipulated, double gamma) {
    for (int t = t_begin; t < t_end; ++t)
        femo_step_ex(pb, R, h, m1, m2, t, beta[t], lambda_t ? lambda_t[t] : lambda, opt, manipulated, gamma);
}

/* ------------------------------------------------------------------------------------------
 * Readout sigma_i = argmax_s P_i(s)  (Eq.4), reading R3: taken on the fields
 * (argmax h == argmax P); two-state: state 1 iff h_i > 0; ties -> lowest state.
 * ---------------------------------------------------------------------------------------- */
void femo_round(const femo_problem *pb, int32_t R, const double *h, int32_t *cfg) {
    int n = pb->n, F = femo_fields_per_var(pb);
    for (int64_t k = 0; k < (int64_t)R * n; ++k) {
        const double *hk = h + k * F;
        if (F == 1) {
            cfg[k] = hk[0] > 0.0 ? 1 : 0;
        } else {
            int best = 0;
            for (int s = 1; s < F; ++s)
                if (hk[s] > hk[best]) best = s;
            cfg[k] = best;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Energy of ONE configuration cfg[n] (plain definitions; the bit-exact gate).
 *   MaxCut : cut = sum_{(i,j) in E, s_i != s_j} W_ij ; E = -cut            (Eq.6)
 *   bMinCut: cut as above; n_k = #{i : s_i = k};
 *            energy = cut + lambda * sum_k (n_k - n/q)^2  (k ascending)     (Eq.7, R2)
 *            with node weights (integral, S33 PAPER.md:892): n_k = sum_{i : s_i = k} V_i and n = sum_i V_i
 *   MaxSAT : unsat = #{m : every literal of m is false}                     (Eq.8)
 *   Ising  : E = -sum_{i<j} W_ij s_i s_j, s = 2 cfg - 1, row-major order
 * e_int is the integer energy (weights rounded to nearest; meaningful when they are integral),
 * e_real the same sum in double.  part[q] (may be NULL) receives n_k for the Potts kind.
 * ---------------------------------------------------------------------------------------- */
void femo_energy(const femo_problem *pb, const int32_t *cfg, double lambda, int64_t *e_int, double *e_real,
                 int32_t *part) {
    int n = pb->n;
    int64_t ei = 0;
    double er = 0.0;
    if (pb->kind == FEMO_MAXCUT || pb->kind == FEMO_BMINCUT) {
        int64_t cut_i = 0;
        double cut_r = 0.0;
        for (int i = 0; i < n; ++i)
            for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                int j = pb->col_idx[e];
                if (j <= i || cfg[i] == cfg[j]) continue;
                cut_i += llround(wgt(pb, e));
                cut_r += wgt(pb, e);
            }
        if (pb->kind == FEMO_MAXCUT) {
            ei = -cut_i;
            er = -cut_r;
        } else {
            int q = pb->q;
            int32_t *cnt = (int32_t *)calloc((size_t)q, sizeof(int32_t));
            int64_t total = 0;
            for (int i = 0; i < n; ++i) {
                cnt[cfg[i]] += (int32_t)llround(nodew(pb, i));
                total += llround(nodew(pb, i));
            }
            double pen = 0.0;
            for (int k = 0; k < q; ++k) {
                double d = (double)cnt[k] - (double)total / (double)q;
                pen = pen + d * d;
            }
            ei = cut_i;
            er = cut_r + lambda * pen;
            if (part) memcpy(part, cnt, sizeof(int32_t) * (size_t)q);
            free(cnt);
        }
    } else if (pb->kind == FEMO_MAXSAT && pb->lit_state) { /* a clause is satisfied when some variable takes its clause value */
        for (int c = 0; c < pb->m; ++c) {
            int sat = 0;
            for (int64_t x = pb->clause_ptr[c]; x < pb->clause_ptr[c + 1]; ++x)
                if (cfg[pb->lits[x] - 1] == pb->lit_state[x]) sat = 1;
            if (!sat) ei += 1;
        }
        er = (double)ei;
    } else if (pb->kind == FEMO_MAXSAT) {
        for (int c = 0; c < pb->m; ++c) {
            int sat = 0;
            for (int64_t x = pb->clause_ptr[c]; x < pb->clause_ptr[c + 1]; ++x) {
                int lit = pb->lits[x];
                int v = (lit > 0 ? lit : -lit) - 1;
                if ((lit > 0 && cfg[v] == 1) || (lit < 0 && cfg[v] == 0)) sat = 1;
            }
            if (!sat) ei += 1;
        }
        er = (double)ei;
    } else { /* ISING */
        if (pb->dense_J) {
            for (int i = 0; i < n; ++i)
                for (int j = i + 1; j < n; ++j) {
                    double w = pb->dense_J[(size_t)i * n + j];
                    double ss = (double)((2 * cfg[i] - 1) * (2 * cfg[j] - 1));
                    er -= w * ss;
                    ei -= llround(w) * (int64_t)((2 * cfg[i] - 1) * (2 * cfg[j] - 1));
                }
        } else {
            for (int i = 0; i < n; ++i)
                for (int64_t e = pb->row_ptr[i]; e < pb->row_ptr[i + 1]; ++e) {
                    int j = pb->col_idx[e];
                    if (j <= i) continue;
                    int ss = (2 * cfg[i] - 1) * (2 * cfg[j] - 1);
                    er -= wgt(pb, e) * (double)ss;
                    ei -= llround(wgt(pb, e)) * (int64_t)ss;
                }
        }
    }
    *e_int = ei;
    *e_real = er;
}

/* all replicas: cfg[R][n] -> e_int[R], e_real[R], part[R][q] (NULL allowed) */
void femo_energies(const femo_problem *pb, int32_t R, const int32_t *cfg, double lambda, int64_t *e_int,
                   double *e_real, int32_t *part) {
    for (int a = 0; a < R; ++a)
        femo_energy(pb, cfg + (size_t)a * pb->n, lambda, e_int + a, e_real + a,
                    part ? part + (size_t)a * pb->q : NULL);
}

/* Best replica: argmin_a E(sigma^a)  (Eq.5); ties -> lowest a. */
int32_t femo_argmin(int32_t R, const double *e_real) {
    int best = 0;
    for (int a = 1; a < R; ++a)
        if (e_real[a] < e_real[best]) best = a;
    return best;
}

int32_t femo_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
