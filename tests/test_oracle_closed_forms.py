"""Closed forms, invariants and limits that pin the oracle's marginals, entropy, schedules, Adam,
integer energies and initial-field generator (CPU only).  Citations are PAPER.md lines."""
import itertools
import math
import os

import numpy as np
import pytest
import torch

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem, small_graph, dense_W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- marginals and entropy
@pytest.mark.parametrize("q", [2, 3, 8])
def test_uniform_start_is_maximal_entropy(q):
    """h = 0 => P = 1/q and S = n ln q."""
    b = small_graph(7, 0.5, 31, pm1=False)
    if q == 2:
        pb = as_problem(b)
        h = np.zeros(b.n)
        assert np.allclose(fo.marginals(pb, h), 0.5, atol=0)
    else:
        pb = as_problem(wl.Instance(wl.BMINCUT, b.n, q, b.row_ptr, b.col_idx, None))
        h = np.zeros(b.n * q)
        assert np.max(np.abs(fo.marginals(pb, h) - 1.0 / q)) < 1e-16
    assert abs(fo.entropy(pb, h) - b.n * math.log(q)) < 1e-13


def test_softmax_shift_invariance_and_normalisation():
    b = small_graph(6, 0.5, 32, pm1=False)
    pb = as_problem(wl.Instance(wl.BMINCUT, b.n, 5, b.row_ptr, b.col_idx, None))
    rng = np.random.default_rng(0)
    h = rng.normal(size=(b.n, 5)) * 3
    P = fo.marginals(pb, h.ravel()).reshape(b.n, 5)
    P2 = fo.marginals(pb, (h + rng.normal(size=(b.n, 1)) * 50).ravel()).reshape(b.n, 5)
    assert np.max(np.abs(P.sum(1) - 1)) < 1e-15
    assert np.max(np.abs(P - P2)) < 1e-13
    ref = torch.softmax(torch.tensor(h), dim=1).numpy()          # library routine as the special case
    assert np.max(np.abs(P - ref)) < 1e-15


def test_two_state_marginal_is_sigmoid_and_tanh_identity():
    """P = sigmoid(h), m = 2P - 1 = tanh(h/2); stable in both tails."""
    b = small_graph(9, 0.5, 33)
    h = np.array([-800.0, -40.0, -3.0, -1e-9, 0.0, 1e-9, 3.0, 40.0, 800.0])
    P = fo.marginals(as_problem(b), h)
    assert P[0] == 0.0 and P[-1] == 1.0 and P[4] == 0.5
    assert np.max(np.abs(2 * P - 1 - np.tanh(h / 2))) < 1e-15
    assert np.all(np.isfinite(fo.grad_h(as_problem(b), h, 3.0)))
    assert math.isfinite(fo.entropy(as_problem(b), h))


def test_entropy_matches_definition_S2():
    """S = -sum P ln P (S2) evaluated literally on moderate fields."""
    b = small_graph(8, 0.5, 34)
    h = np.random.default_rng(1).normal(size=b.n) * 2
    p = 1 / (1 + np.exp(-h))
    assert abs(fo.entropy(as_problem(b), h) + np.sum(p * np.log(p) + (1 - p) * np.log(1 - p))) < 1e-13


# ---------------------------------------------------------------- beta -> infinity (north_star check 3)
def brute_cut(W, cfg):
    iu, ju = np.triu_indices(W.shape[0], 1)
    return float(np.sum(W[iu, ju] * (cfg[iu] != cfg[ju])))


def test_saturation_maxcut_and_ising():
    inst = small_graph(12, 0.5, 35, pm1=True)
    pb = as_problem(inst)
    W = dense_W(inst)
    rng = np.random.default_rng(2)
    for _ in range(5):
        cfg = rng.integers(0, 2, size=inst.n)
        h = (2.0 * cfg - 1.0) * 800.0                    # one-hot marginals to double precision
        assert fo.internal_energy(pb, h) == -brute_cut(W, cfg)
        assert abs(fo.entropy(pb, h)) < 1e-20
        assert np.max(np.abs(fo.grad_h(pb, h, 100.0))) < 1e-20
        e_int, e_real, _ = fo.energies(pb, cfg[None])
        assert e_int[0] == -int(brute_cut(W, cfg)) and e_real[0] == float(e_int[0])
        # Ising with J = -W/2: E_ising = -sum_{i<j} J s_i s_j = (sum_E W)/2 - cut
        ipb = as_problem(wl.sparse_ising_from(inst, -0.5))
        s = 2 * cfg - 1
        iu, ju = np.triu_indices(inst.n, 1)
        assert abs(fo.internal_energy(ipb, h) - np.sum(0.5 * W[iu, ju] * s[iu] * s[ju])) < 1e-12


def test_saturation_bmincut_includes_balance_identity():
    """One-hot P => U_MF = cut + lambda * sum_k (n_k - n/q)^2 exactly (Eq.7, reading R2)."""
    b = small_graph(12, 0.5, 36, pm1=False)
    q, lam = 4, 0.3
    inst = wl.Instance(wl.BMINCUT, b.n, q, b.row_ptr, b.col_idx, None)
    pb = as_problem(inst)
    W = dense_W(inst)
    rng = np.random.default_rng(3)
    for _ in range(5):
        cfg = rng.integers(0, q, size=b.n)
        h = np.full((b.n, q), -800.0)
        h[np.arange(b.n), cfg] = 800.0
        cnt = np.bincount(cfg, minlength=q)
        expect = brute_cut(W, cfg) + lam * np.sum((cnt - b.n / q) ** 2)
        assert abs(fo.internal_energy(pb, h.ravel(), lam) - expect) < 1e-12
        e_int, e_real, part = fo.energies(pb, cfg[None], lam)
        assert e_int[0] == int(brute_cut(W, cfg)) and abs(e_real[0] - expect) < 1e-12
        assert np.array_equal(part[0], cnt)
        # Eq.7's own form differs by the constant lambda (n - n^2/q)
        eq7 = brute_cut(W, cfg) + lam * (np.sum(cnt * cnt) - b.n)
        assert abs(eq7 + lam * (b.n - b.n ** 2 / q) - expect) < 1e-12


def test_saturation_maxsat():
    inst = wl.random_ksat(14, 60, 3, 37)
    pb = as_problem(inst)
    lits = inst.lits.reshape(inst.m, 3)
    rng = np.random.default_rng(4)
    for _ in range(5):
        cfg = rng.integers(0, 2, size=inst.n)
        unsat = sum(1 for c in lits if not any((cfg[abs(l) - 1] == 1) == (l > 0) for l in c))
        h = (2.0 * cfg - 1.0) * 800.0
        assert fo.internal_energy(pb, h) == float(unsat)
        assert fo.energies(pb, cfg[None])[0][0] == unsat


# ---------------------------------------------------------------- integer energies by enumeration
def test_paper_cnf_example_truth_table():
    clauses = []
    with open(os.path.join(GOLDEN, "cnf_example.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                clauses.append([int(x) for x in line.split()])
    lits = np.array([l for c in clauses for l in c], dtype=np.int32)
    ptr = np.cumsum([0] + [len(c) for c in clauses]).astype(np.int64)
    pb = fo.Problem(kind=fo.MAXSAT, n=4, q=2, m=len(clauses), clause_ptr=ptr, lits=lits)
    n_sat_assignments = 0
    for bits in itertools.product([0, 1], repeat=4):
        s1, s2, s3, s4 = [bool(b) for b in bits]
        truth = [s1 or (not s2), (not s1) or s4, s2 or (not s3) or (not s4)]
        unsat = sum(1 for t in truth if not t)
        assert fo.energies(pb, np.array(bits, dtype=np.int32)[None])[0][0] == unsat
        n_sat_assignments += unsat == 0
        # mean-field energy on one-hot marginals equals the count
        assert fo.internal_energy(pb, (2.0 * np.array(bits) - 1.0) * 800.0) == float(unsat)
    assert n_sat_assignments > 0


def test_energy_enumeration_small_graphs():
    inst = small_graph(10, 0.5, 38, pm1=True)
    pb = as_problem(inst)
    W = dense_W(inst)
    cfgs = np.array(list(itertools.product([0, 1], repeat=10)), dtype=np.int32)
    e_int, e_real, _ = fo.energies(pb, cfgs)
    iu, ju = np.triu_indices(10, 1)
    ref = -np.sum(W[iu, ju][None] * (cfgs[:, iu] != cfgs[:, ju]), axis=1)
    assert np.array_equal(e_int, ref.astype(np.int64))
    assert fo.argmin(e_real) == int(np.argmin(ref))           # numpy argmin also takes the first minimum
    # dense Ising energy, E = -sum_{i<j} J s_i s_j
    sk = wl.sk_dense(9, 39)
    cf = np.array(list(itertools.product([0, 1], repeat=9)), dtype=np.int32)
    s = 2.0 * cf - 1.0
    J = sk.dense_J.astype(np.float64)
    ref = -0.5 * np.einsum("ai,ij,aj->a", s, J, s)
    assert np.max(np.abs(fo.energies(as_problem(sk), cf)[1] - ref)) < 1e-12


# ---------------------------------------------------------------- schedules
def test_schedules():
    """beta(0) = beta_min, beta(N-1) = beta_max; inverse-proportional == 1/linspace
    (PAPER.md:572); exponential is geometric."""
    b = fo.schedule_inverse_proportional(1.0, 0.01, 500)
    assert b[0] == 1.0 and abs(b[-1] - 100.0) < 1e-10
    assert np.max(np.abs(1 / b - np.linspace(1.0, 0.01, 500))) < 1e-15
    assert np.max(np.abs(1 / b - torch.linspace(1.0, 0.01, 500, dtype=torch.float64).numpy())) < 1e-15
    e = fo.schedule_exponential(0.02, 750.0, 100)
    assert abs(e[0] - 0.02) < 1e-15 and abs(e[-1] - 750.0) < 1e-9
    assert np.max(np.abs(e[1:] / e[:-1] - (750.0 / 0.02) ** (1 / 99))) < 1e-12


# ---------------------------------------------------------------- Adam against the library routine
@pytest.mark.parametrize("wd", [0.0, 0.013])
def test_adam_matches_torch_optim(wd):
    rng = np.random.default_rng(5)
    h0 = rng.normal(size=40)
    grads = rng.normal(size=(30, 40)) * np.logspace(-6, 1, 40)[None]
    adam = fo.Adam(lr=0.1, beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=wd)
    h, m1, m2 = h0.copy(), np.zeros(40), np.zeros(40)
    p = torch.tensor(h0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([p], lr=0.1, betas=(0.9, 0.999), eps=1e-8, weight_decay=wd)
    for t in range(30):
        fo.adam_update(adam, t + 1, h, m1, m2, grads[t])
        p.grad = torch.tensor(grads[t])
        opt.step()
        assert np.max(np.abs(h - p.detach().numpy())) < 1e-13


# ---------------------------------------------------------------- initial fields
def test_init_fields_generator():
    h = fo.init_fields(0, 64, 500, 1, 1e-3)
    assert h.shape == (64, 500)
    assert np.array_equal(h, h.astype(np.float32).astype(np.float64))         # fp32-representable
    z = h / 1e-3
    assert abs(z.mean()) < 0.02 and abs(z.std() - 1) < 0.02
    assert abs(np.mean(z ** 4) - 3) < 0.15                                     # Gaussian kurtosis
    assert np.array_equal(h, fo.init_fields(0, 64, 500, 1, 1e-3))             # reproducible
    assert not np.array_equal(h, fo.init_fields(1, 64, 500, 1, 1e-3))
    assert np.array_equal(h[:8], fo.init_fields(0, 8, 500, 1, 1e-3))          # replica a independent of R
    hq = fo.init_fields(3, 4, 50, 8, 1e-3)
    assert hq.shape == (4, 50, 8) and abs(hq.std() / 1e-3 - 1) < 0.1
