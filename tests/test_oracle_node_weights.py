"""Pins for the node-weighted balance term of bMinCut (S33-S35), CPU only.

None of these retypes the oracle's loops: (i) S33 is written as a DENSE double sum over (i, j) in torch and autograd
gives the gradient w.r.t. the fields; (ii) one-hot marginals turn U_MF into the integer energy
cut + lambda sum_k (sum_{i in k} V_i - sum_i V_i / q)^2; (iii) a node of integral weight V_i is V_i unit-weight copies
that must sit in the same part -- the energy of the EXPANDED unit-weight graph (the path without node weights, pinned by
enumeration elsewhere) is the reference; (iv) S35 is written with dense matrices over explicit states; (v) V = 1 is
today's path bit for bit.  The finite-difference pin of g^h against F lives in test_oracle_gradient.py (case
bmincut_q4_node_weights).
"""
import itertools

import numpy as np
import pytest
import torch

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem, small_graph, dense_W


def weighted_instance(n, q, seed, lam, vmax=9, real_edges=True):
    b = small_graph(n, 0.5, seed, real=real_edges, pm1=False)
    w = None if b.weight is None else np.abs(b.weight)
    rng = np.random.default_rng(seed + 1000)
    V = rng.integers(1, vmax + 1, size=n).astype(np.float32)
    V[0] = 1.0
    V[1] = float(vmax)
    return wl.Instance(wl.BMINCUT, n, q, b.row_ptr, b.col_idx, w, lam=lam, node_weight=V)


@pytest.mark.parametrize("beta", [0.6, 3.0])
def test_gradient_is_autograd_of_the_dense_double_sum_S33(beta):
    """F = sum_E W_ij sum_s P_i(s)[1 - P_j(s)] + lambda sum_{i,j} sum_s [V_i V_j P_i(s) P_j(s) - V_i^2 P_i(s)^2] - S/beta,
    the balance term written literally as the double sum of S33: the V_i^2 P_i^2 term is subtracted once
    per i, i.e. the printed sum over (i, j) is read like `balance()` (:536, reading R2): (sum_i V_i P_i)^2 - sum_i V_i^2 P_i^2."""
    inst = weighted_instance(8, 4, 61, lam=0.17)
    n, q = inst.n, inst.q
    V = torch.tensor(inst.node_weight.astype(np.float64))
    W = torch.tensor(dense_W(inst))
    h = np.random.default_rng(2).normal(size=(n, q))
    ht = torch.tensor(h, dtype=torch.float64, requires_grad=True)
    P = torch.softmax(ht, dim=1)
    cut = ((W @ P) * (1 - P)).sum() / 2                               # every edge once (reading R1)
    bal = 0.0
    for i in range(n):
        for j in range(n):
            bal = bal + (V[i] * V[j] * P[i] * P[j]).sum()
        bal = bal - (V[i] ** 2 * P[i] ** 2).sum()
    S = -(P * P.log()).sum()
    (cut + inst.lam * bal - S / beta).backward()
    g = fo.grad_h(as_problem(inst), h.ravel(), beta, inst.lam).reshape(n, q)
    assert np.max(np.abs(ht.grad.numpy() - g)) < 1e-12
    # the weights matter: the unweighted gradient is far away
    plain = wl.Instance(wl.BMINCUT, n, q, inst.row_ptr, inst.col_idx, inst.weight, lam=inst.lam)
    assert np.max(np.abs(fo.grad_h(as_problem(plain), h.ravel(), beta, inst.lam).reshape(n, q) - g)) > 1e-2


def expanded_unit_graph(inst):
    """Every node i becomes V_i unit-weight nodes; the edges of i hang on its first copy.  A configuration of the
    weighted graph maps to the one where all copies of i carry s_i: same cut, part sizes n_k = sum_{i in k} V_i."""
    V = inst.node_weight.astype(np.int64)
    first = np.concatenate([[0], np.cumsum(V)[:-1]])
    rows = np.repeat(np.arange(inst.n), np.diff(inst.row_ptr))
    keep = rows < inst.col_idx
    w = None if inst.weight is None else inst.weight[keep]
    row_ptr, col, weight = wl.csr_from_edges(int(V.sum()), first[rows[keep]], first[inst.col_idx[keep]], w)
    return wl.Instance(wl.BMINCUT, int(V.sum()), inst.q, row_ptr, col, weight, lam=inst.lam), np.repeat(np.arange(inst.n), V)


def test_integer_energy_is_that_of_the_expanded_unit_weight_graph():
    b = small_graph(9, 0.5, 62, pm1=False)                               # unit edge weights: integer energies
    V = np.array([3, 1, 7, 2, 1, 5, 4, 1, 2], dtype=np.float32)
    inst = wl.Instance(wl.BMINCUT, b.n, 3, b.row_ptr, b.col_idx, None, lam=0.25, node_weight=V)
    big, owner = expanded_unit_graph(inst)
    rng = np.random.default_rng(3)
    cfg = rng.integers(0, 3, size=(6, inst.n)).astype(np.int32)
    e_int, e_real, part = fo.energies(as_problem(inst), cfg, inst.lam)
    e_int2, e_real2, part2 = fo.energies(as_problem(big), cfg[:, owner], inst.lam)
    assert np.array_equal(e_int, e_int2) and np.array_equal(e_real, e_real2) and np.array_equal(part, part2)
    # and by the definition, enumerated: cut + lambda sum_k (sum_{i in k} V_i - sum V / q)^2
    W = dense_W(inst)
    iu, ju = np.triu_indices(inst.n, 1)
    for a in range(cfg.shape[0]):
        cut = float(np.sum(W[iu, ju] * (cfg[a, iu] != cfg[a, ju])))
        sizes = np.array([V[cfg[a] == k].sum() for k in range(3)], dtype=np.float64)
        assert e_int[a] == int(cut)
        assert abs(e_real[a] - (cut + 0.25 * np.sum((sizes - V.sum() / 3.0) ** 2))) < 1e-12
        assert np.array_equal(part[a], sizes.astype(part.dtype))


def test_saturation_one_hot_marginals_give_the_integer_energy():
    inst = weighted_instance(10, 4, 63, lam=0.031, real_edges=False)
    pb = as_problem(inst)
    rng = np.random.default_rng(4)
    for _ in range(5):
        cfg = rng.integers(0, inst.q, size=inst.n).astype(np.int32)
        h = np.zeros((inst.n, inst.q))
        h[np.arange(inst.n), cfg] = 800.0
        e_real = fo.energies(pb, cfg[None], inst.lam)[1][0]
        assert abs(fo.internal_energy(pb, h.ravel(), inst.lam) - e_real) < 1e-10 * max(1.0, abs(e_real))
        assert abs(fo.entropy(pb, h.ravel())) < 1e-300 or fo.entropy(pb, h.ravel()) == 0.0


def _s35_dense(inst, h, beta, lam, gamma):
    """S27 with the balance part replaced by S35, dense matrices over explicit states, then S20."""
    n, q = inst.n, inst.q
    W = dense_W(inst)
    V = inst.node_weight.astype(np.float64)
    H = h.reshape(n, q)
    P = np.exp(H - H.max(1, keepdims=True))
    P /= P.sum(1, keepdims=True)
    e = np.zeros((n, q))
    e[np.arange(n), np.argmax(H, axis=1)] = 1.0
    rs = W.sum(1)
    ok = rs > 0
    cf = np.where(ok, q / np.where(ok, rs, 1.0), 0.0)
    ca = np.where(ok, q / np.sqrt(np.where(ok, rs, 1.0)), 0.0)
    bal = V[:, None] * ((V[:, None] * e).sum(0)[None, :] - V[:, None] * e)      # V_i [sum_j V_j e_j(s) - V_i e_i(s)]
    ghat = -cf[:, None] * (W @ e) + lam * ca[:, None] * bal + (np.log(P) + 1.0) / beta
    return (gamma * P * (ghat - (P * ghat).sum(1, keepdims=True))).ravel()


@pytest.mark.parametrize("q,beta,gamma", [(3, 0.8, 1.0), (6, 4.0, 0.5)])
def test_manipulated_gradient_is_S35_over_explicit_states(q, beta, gamma):
    inst = weighted_instance(11, q, 64 + q, lam=0.29)
    h = np.random.default_rng(5).normal(size=inst.n * q) * 1.3
    g = fo.grad_h_manipulated(as_problem(inst), h, beta, inst.lam, gamma)
    ref = _s35_dense(inst, h, beta, inst.lam, gamma)
    assert np.max(np.abs(g - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # a plausible mistake -- V_i applied once instead of to both factors of the self term -- is outside the tolerance
    inst1 = wl.Instance(wl.BMINCUT, inst.n, q, inst.row_ptr, inst.col_idx, inst.weight, lam=inst.lam,
                        node_weight=np.ones(inst.n, dtype=np.float32))
    assert np.max(np.abs(fo.grad_h_manipulated(as_problem(inst1), h, beta, inst.lam, gamma) - ref)) > 1e-3


def test_unit_node_weights_are_the_unweighted_path_bit_for_bit():
    inst = weighted_instance(12, 5, 66, lam=0.2)
    ones = wl.Instance(wl.BMINCUT, inst.n, 5, inst.row_ptr, inst.col_idx, inst.weight, lam=0.2,
                       node_weight=np.ones(inst.n, dtype=np.float32))
    none = wl.Instance(wl.BMINCUT, inst.n, 5, inst.row_ptr, inst.col_idx, inst.weight, lam=0.2)
    a, b = as_problem(ones), as_problem(none)
    h = np.random.default_rng(6).normal(size=inst.n * 5)
    assert np.array_equal(fo.grad_h(a, h, 1.7, 0.2), fo.grad_h(b, h, 1.7, 0.2))
    assert np.array_equal(fo.grad_h_manipulated(a, h, 1.7, 0.2, 0.9), fo.grad_h_manipulated(b, h, 1.7, 0.2, 0.9))
    assert fo.internal_energy(a, h, 0.2) == fo.internal_energy(b, h, 0.2)
    cfg = np.random.default_rng(7).integers(0, 5, size=(4, inst.n)).astype(np.int32)
    for x, y in zip(fo.energies(a, cfg, 0.2), fo.energies(b, cfg, 0.2)):
        assert np.array_equal(x, y)


def test_anneal_balances_node_weight_not_node_count():
    """Whole-path sanity on a tiny instance: the best replica reaches the brute-force optimum of the
    node-weighted energy (parts balanced in sum-of-V, not in node count)."""
    b = small_graph(10, 0.4, 67, pm1=False)
    V = np.array([6, 1, 1, 1, 1, 1, 1, 1, 1, 4], dtype=np.float32)
    inst = wl.Instance(wl.BMINCUT, b.n, 2, b.row_ptr, b.col_idx, None, lam=0.2, node_weight=V)
    pb = as_problem(inst)
    best = min(fo.energies(pb, np.array([(0,) + bits], dtype=np.int32), 0.2)[1][0]
               for bits in itertools.product((0, 1), repeat=b.n - 1))
    st = fo.anneal(fo.State(pb, fo.init_fields(1, 32, inst.n, 2)), fo.schedule_inverse_proportional(2.0, 0.02, 400),
                   fo.Adam(lr=0.1), 0.2)
    e = fo.energies(pb, fo.round_configs(pb, st.h), 0.2)[1]
    assert abs(e.min() - best) < 1e-12, (e.min(), best)
