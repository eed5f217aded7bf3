"""Pins for the oracle's SURVEY.md section 8(f) rows (CPU only): RMSprop / SGD optimisers and the
manipulated gradients (one-hot discretisation, per-node normalisation, gamma_grad).

None of these retypes the oracle's formula: the optimisers are pinned to torch.optim (the library the
paper names); the two-state manipulated gradient (the oracle follows the REDUCED form S29/S30)
is pinned to the GENERAL form S25 + S20 written over two explicit states (the paper proves the reduction,
PAPER.md:661-671); saturated fields reduce the manipulated gradient to the exact one on normalised weights
(one-hot = marginal there); plus the invariants sum_s g^h_i(s) = 0, MaxCut == Ising with J = -W/2, and
brute-force optima reached by the whole anneal.
"""
import itertools

import numpy as np
import pytest
import torch

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem, small_graph


# ------------------------------------------------------------------------------------------------ optimisers
def _torch_run(make_opt, grads, h0):
    p = torch.nn.Parameter(torch.tensor(h0, dtype=torch.float64))
    opt = make_opt([p])
    out = []
    for g in grads:
        opt.zero_grad()
        p.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        out.append(p.detach().numpy().copy())
    return out


@pytest.mark.parametrize("momentum,alpha,wd", [(0.0, 0.99, 0.0), (0.9, 0.9, 0.0), (0.5, 0.99, 0.013), (0.0, 0.5, 0.2)])
def test_rmsprop_matches_torch(momentum, alpha, wd):
    rng = np.random.default_rng(3)
    h0 = rng.normal(size=37)
    grads = [rng.normal(size=37) * 10.0 ** rng.integers(-4, 2) for _ in range(25)]
    ref = _torch_run(lambda ps: torch.optim.RMSprop(ps, lr=0.03, alpha=alpha, eps=1e-8, weight_decay=wd,
                                                    momentum=momentum), grads, h0)
    opt = fo.Optimizer(kind=fo.RMSPROP, lr=0.03, alpha=alpha, eps=1e-8, weight_decay=wd, momentum=momentum)
    h, m1, m2 = h0.copy(), np.zeros(37), np.zeros(37)
    for t, g in enumerate(grads):
        fo.rmsprop_update(opt, h, m1, m2, g)
        assert np.max(np.abs(h - ref[t])) <= 1e-13 * max(1.0, np.max(np.abs(ref[t]))), t


@pytest.mark.parametrize("momentum,dampening,wd", [(0.0, 0.0, 0.0), (0.9, 0.0, 0.0), (0.8, 0.3, 0.0), (0.7, 0.1, 0.05)])
def test_sgd_matches_torch(momentum, dampening, wd):
    rng = np.random.default_rng(4)
    h0 = rng.normal(size=29)
    grads = [rng.normal(size=29) for _ in range(25)]
    ref = _torch_run(lambda ps: torch.optim.SGD(ps, lr=0.07, momentum=momentum, dampening=dampening,
                                                weight_decay=wd), grads, h0)
    opt = fo.Optimizer(kind=fo.SGD, lr=0.07, momentum=momentum, dampening=dampening, weight_decay=wd)
    h, m1 = h0.copy(), np.zeros(29)
    for t, g in enumerate(grads):
        fo.sgd_update(opt, t + 1, h, m1, g)
        assert np.max(np.abs(h - ref[t])) <= 1e-13 * max(1.0, np.max(np.abs(ref[t]))), t


def test_anneal_ex_with_adam_and_exact_gradient_is_anneal():
    inst = small_graph(14, 0.4, 21)
    pb = as_problem(inst)
    beta = fo.schedule_inverse_proportional(1.0, 0.05, 40)
    h0 = fo.init_fields(1, 3, inst.n, 1)
    a = fo.anneal(fo.State(pb, h0), beta, fo.Adam(lr=0.2, weight_decay=0.01))
    b = fo.anneal_ex(fo.State(pb, h0), beta, fo.Optimizer(kind=fo.ADAM, lr=0.2, weight_decay=0.01))
    assert np.array_equal(a.h, b.h) and np.array_equal(a.m2, b.m2)


# ------------------------------------------------------------------------------------ manipulated gradients
def _general_form_two_state(inst, h, beta, gamma, ising=False):
    """S25 + S20 over the two explicit states (+1, -1) with fields h(+1) = h, h(-1) = 0:
    ghat^p_i(s) = c_i sum_j W_ij e_j(s) + (1/beta)[ln P_i(s) + 1];  g^h_i(s) = gamma P_i(s)[ghat_i(s) - <ghat_i>_P].
    Returns g^h_i(+1) (= -g^h_i(-1), the gradient of the single field h_i = h_i(+1) - h_i(-1))."""
    n = inst.n
    W = np.zeros((n, n))
    rows = np.repeat(np.arange(n), np.diff(inst.row_ptr))
    w = np.ones(inst.nnz) if inst.weight is None else inst.weight.astype(np.float64)
    W[rows, inst.col_idx] = w
    if ising:
        W = -2.0 * W                                   # dU/dp = -2 sum_j J_ij m_j; MaxCut has dU/dp = sum_j W_ij m_j
    hh = np.stack([h, np.zeros(n)], axis=1)            # states (+1, -1)
    P = np.exp(hh - hh.max(1, keepdims=True))
    P /= P.sum(1, keepdims=True)
    e = np.zeros((n, 2))
    e[np.arange(n), np.where(h > 0, 0, 1)] = 1.0
    e[h == 0] = 0.5                                    # sgn(0) = 0  <=>  e = (1/2, 1/2)
    l1 = np.abs(W).sum(1)
    c = np.where(l1 > 0, 1.0 / np.where(l1 > 0, l1, 1.0), 0.0)
    # S24 -> S25 drops the factor 2 of S24 together with P -> e: the coupling part of ghat^p is c_i sum_j W_ij e_j(s)
    ghat = c[:, None] * (W @ e) + (np.log(P) + 1.0) / beta
    gh = gamma * P * (ghat - (P * ghat).sum(1, keepdims=True))
    assert np.allclose(gh[:, 0], -gh[:, 1], atol=1e-15)
    return gh[:, 0]


@pytest.mark.parametrize("beta,gamma", [(0.4, 1.0), (2.0, 0.7), (9.0, 3.0)])
def test_two_state_manipulated_gradient_is_the_reduction_of_the_general_form(beta, gamma):
    rng = np.random.default_rng(8)
    for inst, ising in ((small_graph(11, 0.5, 31, real=True), False), (small_graph(12, 0.4, 32), False),
                        (wl.sparse_ising_from(small_graph(10, 0.5, 33, real=True), scale=0.6), True)):
        h = rng.normal(size=inst.n) * 1.5
        h[3] = 0.0                                     # sgn(0) = 0
        g = fo.grad_h_manipulated(as_problem(inst), h, beta, 0.0, gamma)
        ref = _general_form_two_state(inst, h, beta, gamma, ising)
        assert np.max(np.abs(g - ref)) < 1e-13


def test_manipulated_maxcut_equals_manipulated_ising_with_J_minus_half_W():
    g = small_graph(13, 0.45, 34, real=True)
    isg = wl.sparse_ising_from(g, scale=-0.5)
    h = np.random.default_rng(9).normal(size=g.n)
    a = fo.grad_h_manipulated(as_problem(g), h, 1.3, 0.0, 0.8)
    b = fo.grad_h_manipulated(as_problem(isg), h, 1.3, 0.0, 0.8)
    assert np.max(np.abs(a - b)) < 1e-14


def _row_normalised(inst, scale_of_rowsum):
    """Copy of a graph instance whose CSR entry (i, j) carries W_ij * scale_of_rowsum(sum_j |W_ij|) (per ROW)."""
    w = np.ones(inst.nnz) if inst.weight is None else inst.weight.astype(np.float64)
    rows = np.repeat(np.arange(inst.n), np.diff(inst.row_ptr))
    l1 = np.bincount(rows, weights=np.abs(w), minlength=inst.n)
    return w * scale_of_rowsum(l1)[rows]


def test_saturated_fields_reduce_the_manipulated_gradient_to_the_exact_one_on_normalised_weights():
    """|h| = 40: m_j = +-1 exactly in double, so e_j = P_j and the manipulated gradient is the exact gradient of a
    problem whose rows are divided by sum_j |W_ij| (the oracle's exact gradient never assumes symmetric weights)."""
    rng = np.random.default_rng(10)
    g = small_graph(12, 0.5, 35, real=True)
    h = 40.0 * rng.choice([-1.0, 1.0], size=g.n)
    pb = as_problem(g)
    pbn = fo.Problem(kind=fo.MAXCUT, n=g.n, q=2, row_ptr=g.row_ptr, col_idx=g.col_idx,
                     weight=_row_normalised(g, lambda l1: 1.0 / l1))
    a = fo.grad_h_manipulated(pb, h, 0.9, 0.0, 1.7)
    b = 1.7 * fo.grad_h(pbn, h, 0.9)
    assert np.max(np.abs(a - b)) <= 1e-15 + 1e-12 * np.max(np.abs(b))
    # Potts, regular graph (uniform c^f, c^a): exact gradient with W c^f and lambda c^a / 2 (S26 has 2 lambda, S27 lambda)
    reg = wl.random_regular(20, 4, 36, wl.BMINCUT, 3, lam=0.3)
    q, d = 3, 4.0
    hp = np.zeros((reg.n, q))
    hp[np.arange(reg.n), rng.integers(0, q, reg.n)] = 60.0
    pbp = as_problem(reg)
    pbs = fo.Problem(kind=fo.BMINCUT, n=reg.n, q=q, row_ptr=reg.row_ptr, col_idx=reg.col_idx,
                     weight=np.full(reg.nnz, q / d))
    a = fo.grad_h_manipulated(pbp, hp.ravel(), 1.1, 0.3, 1.0)
    b = fo.grad_h(pbs, hp.ravel(), 1.1, 0.3 * (q / np.sqrt(d)) / 2.0)
    assert np.max(np.abs(a - b)) <= 1e-13


def test_potts_manipulated_gradient_rows_sum_to_zero_and_isolated_nodes_feel_no_coupling():
    b = small_graph(9, 0.3, 37, pm1=False)
    inst = wl.Instance(wl.BMINCUT, b.n, 4, b.row_ptr, b.col_idx, None, lam=0.2)
    deg = np.diff(inst.row_ptr)
    h = np.random.default_rng(11).normal(size=(inst.n, 4))
    g = fo.grad_h_manipulated(as_problem(inst), h.ravel(), 2.0, 0.2, 1.0).reshape(inst.n, 4)
    assert np.max(np.abs(g.sum(1))) < 1e-14                         # S20: sum_s g^h_i(s) = 0
    assert np.all(np.isfinite(g))
    if np.any(deg == 0):                                             # c^f = c^a = 0: only the entropy term is left
        i = int(np.argmax(deg == 0))
        P = np.exp(h[i] - h[i].max()); P /= P.sum()
        ent = np.log(P) / 2.0
        assert np.allclose(g[i], P * (ent - (P * ent).sum()), atol=1e-14)


def test_max_sat_and_dense_ising_are_not_manipulated_only_scaled():
    inst = wl.random_ksat(9, 30, 3, 38)
    h = np.random.default_rng(12).normal(size=inst.n)
    pb = as_problem(inst)
    assert np.array_equal(fo.grad_h_manipulated(pb, h, 1.5, 0.0, 2.5), 2.5 * fo.grad_h(pb, h, 1.5))


def _brute_force_maxcut(inst):
    n = inst.n
    rows = np.repeat(np.arange(n), np.diff(inst.row_ptr))
    w = np.ones(inst.nnz) if inst.weight is None else inst.weight
    best = -1e30
    for bits in itertools.product((0, 1), repeat=n - 1):
        s = np.array((0,) + bits)
        best = max(best, 0.5 * float(np.sum(w[s[rows] != s[inst.col_idx]])))
    return best


@pytest.mark.parametrize("kind", ["rmsprop", "sgd", "adam"])
def test_manipulated_anneal_reaches_brute_force_optimum(kind):
    """The paper's benchmarked recipe (manipulated gradients, RMSprop / SGD / Adam) finds the optimum of small graphs."""
    opt = {"rmsprop": fo.Optimizer(kind=fo.RMSPROP, lr=0.05, alpha=0.9, momentum=0.5),
           "sgd": fo.Optimizer(kind=fo.SGD, lr=1.0, momentum=0.8, dampening=0.1),
           "adam": fo.Optimizer(kind=fo.ADAM, lr=0.1)}[kind]
    hits = 0
    for k in range(8):
        inst = small_graph(14, 0.4, 50 + k)
        pb = as_problem(inst)
        beta = fo.schedule_exponential(0.5, 40.0, 300)
        st = fo.anneal_ex(fo.State(pb, fo.init_fields(k, 24, inst.n, 1)), beta, opt, manipulated=True, gamma=1.0)
        e = fo.energies(pb, fo.round_configs(pb, st.h))[1]
        hits += int(round(-e.min()) == round(_brute_force_maxcut(inst)))
    assert hits >= 7, hits


# --------------------------------------------------- Potts manipulated gradient on a weighted, irregular graph
def _general_form_potts(inst, h, beta, lam, gamma, global_rowsum=False):
    """S27 + S20 written over explicit states with a DENSE weight matrix:
    ghat^p = -c^f (W e) + lambda c^a [1 (1^T e) - e] + (1/beta)[ln P + 1],  c^f_i = q / sum_j W_ij,
    c^a_i = q / sqrt(sum_j W_ij) per NODE;  g^h = gamma P (ghat^p - <ghat^p>_P)."""
    n, q = inst.n, inst.q
    W = np.zeros((n, n))
    rows = np.repeat(np.arange(n), np.diff(inst.row_ptr))
    W[rows, inst.col_idx] = np.ones(inst.nnz) if inst.weight is None else inst.weight.astype(np.float64)
    assert np.array_equal(W, W.T)
    H = h.reshape(n, q)
    P = np.exp(H - H.max(1, keepdims=True))
    P /= P.sum(1, keepdims=True)
    e = np.zeros((n, q))
    e[np.arange(n), np.argmax(H, axis=1)] = 1.0        # numpy's argmax returns the lowest index among ties (R3)
    rs = W.sum(1)
    ok = rs > 0
    if global_rowsum:                                  # (deliberately wrong variant, used to show the pin has teeth)
        rs = np.where(ok, rs[ok].mean(), 0.0)
    cf = np.where(ok, q / np.where(ok, rs, 1.0), 0.0)
    ca = np.where(ok, q / np.sqrt(np.where(ok, rs, 1.0)), 0.0)
    ghat = -cf[:, None] * (W @ e) + lam * ca[:, None] * (e.sum(0)[None, :] - e) + (np.log(P) + 1.0) / beta
    return (gamma * P * (ghat - (P * ghat).sum(1, keepdims=True))).ravel()


def _weighted_irregular_potts(n, q, seed, lam):
    """Erdos-Renyi graph (irregular degrees, maybe an isolated node) with real positive weights of very different sizes."""
    rng = np.random.default_rng(seed)
    iu, ju = np.triu_indices(n, k=1)
    keep = rng.random(iu.size) < 0.3
    keep[iu == n - 1] = False
    keep[ju == n - 1] = False                          # node n-1 isolated: c^f = c^a = 0
    u, v = iu[keep], ju[keep]
    w = (rng.random(u.size) * 3.0 + 0.05) * 10.0 ** rng.integers(-1, 2, size=u.size)
    row_ptr, col, weight = wl.csr_from_edges(n, u, v, w)
    return wl.Instance(wl.BMINCUT, n, q, row_ptr, col, weight, lam=lam)


@pytest.mark.parametrize("q,beta,gamma", [(3, 0.7, 1.0), (5, 2.5, 0.6), (8, 11.0, 2.0)])
def test_potts_manipulated_gradient_on_a_weighted_irregular_graph_is_s27_with_per_node_factors(q, beta, gamma):
    inst = _weighted_irregular_potts(13, q, 40 + q, lam=0.37)
    deg = np.diff(inst.row_ptr)
    assert deg.min() == 0 and len(set(deg.tolist())) > 3            # irregular, with an isolated node
    rs = np.bincount(np.repeat(np.arange(inst.n), deg), weights=inst.weight.astype(np.float64), minlength=inst.n)
    assert rs[rs > 0].max() / rs[rs > 0].min() > 3.0                 # per-node factors differ a lot
    rng = np.random.default_rng(41)
    h = rng.normal(size=(inst.n, q)) * 1.2
    h[2, 1] = h[2, 3 % q] = h[2].max() + 0.5                          # a tie among the maxima: lowest state wins
    g = fo.grad_h_manipulated(as_problem(inst), h.ravel(), beta, inst.lam, gamma)
    ref = _general_form_potts(inst, h.ravel(), beta, inst.lam, gamma)
    assert np.max(np.abs(g - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # a mistake this pin is there to catch -- one global row sum instead of one per node -- is far outside the tolerance
    wrong = _general_form_potts(inst, h.ravel(), beta, inst.lam, gamma, global_rowsum=True)
    assert np.max(np.abs(wrong - ref)) > 1e-3 * np.max(np.abs(ref))


# -------------------------------------------------------------------------------------- per-step lambda (the ramp)
@pytest.mark.parametrize("manipulated", [False, True])
def test_anneal_with_a_lambda_ramp_is_step_by_step_grad_with_that_steps_lambda(manipulated):
    """PAPER.md:828, Table S3 :842: lambda is incremented linearly from 0 to lambda_max over the N steps.  anneal(lam_t)
    must equal: for t, g = grad(h, beta[t], lam_t[t]); Adam(t + 1) -- composed here from the separately pinned pieces."""
    inst = _weighted_irregular_potts(12, 4, 77, lam=123.0)            # inst.lam must be IGNORED when lam_t is given
    pb = as_problem(inst)
    N, R = 30, 3
    beta = fo.schedule_exponential(0.3, 20.0, N)
    lam_t = np.linspace(0.0, 0.2, N)
    h0 = fo.init_fields(5, R, inst.n, inst.q)
    adam = fo.Adam(lr=0.05, weight_decay=0.01)
    if manipulated:
        st = fo.anneal_ex(fo.State(pb, h0), beta, fo.Optimizer(kind=fo.ADAM, lr=0.05, weight_decay=0.01), inst.lam,
                          lam_t=lam_t, manipulated=True, gamma=0.9)
    else:
        st = fo.anneal(fo.State(pb, h0), beta, adam, inst.lam, lam_t=lam_t)
    h = h0.reshape(R, -1).copy()
    m1, m2 = np.zeros_like(h), np.zeros_like(h)
    for t in range(N):
        for a in range(R):
            g = (fo.grad_h_manipulated(pb, h[a], beta[t], lam_t[t], 0.9) if manipulated
                 else fo.grad_h(pb, h[a], beta[t], lam_t[t]))
            fo.adam_update(adam, t + 1, h[a], m1[a], m2[a], g)
    assert np.array_equal(st.h.reshape(R, -1), h)
    # and the ramp matters: the constant-lambda anneal ends elsewhere
    other = fo.anneal(fo.State(pb, h0), beta, adam, 0.2)
    assert np.max(np.abs(other.h - st.h)) > 1e-3
    # lambda_t[t] = lambda for all t is the constant-lambda anneal, bit for bit
    same = fo.anneal(fo.State(pb, h0), beta, adam, 999.0, lam_t=np.full(N, 0.2))
    assert np.array_equal(same.h, other.h)
