"""Pins for the oracle's free energy and explicit gradient (CPU only).

Nothing here retypes the oracle's formulas: the gradient is pinned by central finite differences of
F (north_star check 1), by torch autograd on the paper's own listing (which
the paper says equals the explicit gradient), and by the identities the paper states
(S20 row sums PAPER.md:599; q=2 reduction PAPER.md:661; Ising/MaxCut map PAPER.md:43,114).
"""
import numpy as np
import pytest
import torch

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl


def as_problem(inst: wl.Instance) -> fo.Problem:
    return fo.Problem(kind=inst.kind, n=inst.n, q=inst.q, row_ptr=inst.row_ptr, col_idx=inst.col_idx,
                      weight=inst.weight, dense_J=inst.dense_J, m=inst.m, clause_ptr=inst.clause_ptr, lits=inst.lits,
                      node_weight=inst.node_weight, lit_state=getattr(inst, "lit_state", None))


def small_graph(n, p, seed, pm1=True, real=False):
    g = wl.erdos_renyi_maxcut(n, p, seed, pm1=pm1)
    if real:
        rng = np.random.default_rng(seed + 7)
        # symmetric real weights: draw per undirected edge, mirror
        w = {}
        rows = np.repeat(np.arange(n), np.diff(g.row_ptr))
        ww = np.empty(g.nnz, dtype=np.float32)
        for e, (i, j) in enumerate(zip(rows, g.col_idx)):
            key = (min(i, j), max(i, j))
            if key not in w:
                w[key] = rng.normal()
            ww[e] = w[key]
        g.weight = ww
    return g


def cases():
    out = []
    g = small_graph(10, 0.5, 11, real=True)
    out.append(("maxcut_real", g, 0.0))
    out.append(("maxcut_pm1", small_graph(12, 0.4, 12), 0.0))
    out.append(("ising_sparse", wl.sparse_ising_from(small_graph(9, 0.6, 13, real=True), scale=0.7), 0.0))
    sk = wl.sk_dense(8, 14)
    out.append(("ising_dense", sk, 0.0))
    b = small_graph(8, 0.6, 15, pm1=False)
    out.append(("bmincut_q3", wl.Instance(wl.BMINCUT, b.n, 3, b.row_ptr, b.col_idx, None), 0.37))
    b2 = small_graph(7, 0.7, 16, real=True)
    b2.weight = np.abs(b2.weight)
    out.append(("bmincut_q5_w", wl.Instance(wl.BMINCUT, b2.n, 5, b2.row_ptr, b2.col_idx, b2.weight), 0.11))
    vb = wl.Instance(wl.BMINCUT, b2.n, 4, b2.row_ptr, b2.col_idx, b2.weight,
                     node_weight=np.array([3, 1, 7, 2, 1, 5, 4], dtype=np.float32))   # node-weighted balance term (S33-S34)
    out.append(("bmincut_q4_node_weights", vb, 0.23))
    out.append(("maxsat_k3", wl.random_ksat(9, 30, 3, 17), 0.0))
    out.append(("maxsat_k4", wl.random_ksat(10, 40, 4, 18), 0.0))
    return out


@pytest.mark.parametrize("name,inst,lam", cases(), ids=[c[0] for c in cases()])
@pytest.mark.parametrize("beta", [0.3, 1.0, 7.0])
def test_gradient_matches_finite_differences(name, inst, lam, beta):
    pb = as_problem(inst)
    rng = np.random.default_rng(5)
    h = rng.normal(scale=0.8, size=inst.n * pb.fields_per_var)
    g = fo.grad_h(pb, h, beta, lam)
    eps = 1e-6
    fd = np.empty_like(h)
    for k in range(h.size):
        hp, hm = h.copy(), h.copy()
        hp[k] += eps
        hm[k] -= eps
        fd[k] = (fo.free_energy(pb, hp, beta, lam) - fo.free_energy(pb, hm, beta, lam)) / (2 * eps)
    assert np.max(np.abs(fd - g)) < 2e-8 * max(1.0, np.max(np.abs(g)))


def dense_W(inst):
    W = np.zeros((inst.n, inst.n))
    rows = np.repeat(np.arange(inst.n), np.diff(inst.row_ptr))
    W[rows, inst.col_idx] = 1.0 if inst.weight is None else inst.weight
    return W


def listing_F(problem, W, p, penalty, beta):
    """The paper's listing with cut() halved: reading R1 (edge once)."""
    cut = ((W @ p) * (1 - p)).sum((1, 2)) / 2
    S = -(p * p.log()).sum(2).sum(1)
    balance = (p.sum(1) ** 2).sum(1) - (p ** 2).sum(2).sum(1)
    if problem == "maxcut":
        return -cut - S / beta
    return cut + penalty * balance - S / beta


@pytest.mark.parametrize("beta", [0.5, 4.0])
def test_bmincut_gradient_matches_autograd_of_listing(beta):
    b = small_graph(9, 0.5, 21, pm1=False)
    inst = wl.Instance(wl.BMINCUT, b.n, 4, b.row_ptr, b.col_idx, None)
    pb = as_problem(inst)
    lam = 0.23
    rng = np.random.default_rng(3)
    h = rng.normal(size=(1, inst.n, 4))
    ht = torch.tensor(h, dtype=torch.float64, requires_grad=True)
    F = listing_F("bmincut", torch.tensor(dense_W(inst)), torch.softmax(ht, dim=2), lam, beta)
    F.backward(gradient=torch.ones_like(F))
    g = fo.grad_h(pb, h.ravel(), beta, lam).reshape(1, inst.n, 4)
    assert np.max(np.abs(ht.grad.numpy() - g)) < 1e-12


@pytest.mark.parametrize("beta", [0.5, 4.0])
def test_maxcut_gradient_matches_autograd_of_listing(beta):
    inst = small_graph(11, 0.5, 22, real=True)
    pb = as_problem(inst)
    rng = np.random.default_rng(4)
    h = rng.normal(size=inst.n)
    # two-state softmax with h(+1) = h, h(-1) = 0; d/dh(+1) is the gradient w.r.t. the single field
    h2 = np.stack([np.zeros_like(h), h], axis=1)[None]          # state index 1 == "+1"
    ht = torch.tensor(h2, dtype=torch.float64, requires_grad=True)
    F = listing_F("maxcut", torch.tensor(dense_W(inst)), torch.softmax(ht, dim=2), 0.0, beta)
    F.backward(gradient=torch.ones_like(F))
    g = fo.grad_h(pb, h, beta)
    assert np.max(np.abs(ht.grad.numpy()[0, :, 1] - g)) < 1e-12
    # q=2 identity g^h(+1) = -g^h(-1)
    assert np.max(np.abs(ht.grad.numpy()[0, :, 1] + ht.grad.numpy()[0, :, 0])) < 1e-12


def test_maxsat_gradient_matches_autograd_of_eq11():
    inst = wl.random_ksat(12, 50, 4, 23)
    pb = as_problem(inst)
    beta = 1.7
    rng = np.random.default_rng(6)
    h = rng.normal(size=inst.n)
    ht = torch.tensor(h, dtype=torch.float64, requires_grad=True)
    p = torch.sigmoid(ht)
    U = 0.0
    lits = inst.lits.reshape(inst.m, -1)
    for c in range(inst.m):                      # Eq.11: prod_i [1 - P_i(W_mi)]
        prod = 1.0
        for lit in lits[c]:
            v = abs(int(lit)) - 1
            prod = prod * ((1 - p[v]) if lit > 0 else p[v])
        U = U + prod
    S = -(p * p.log() + (1 - p) * (1 - p).log()).sum()
    (U - S / beta).backward()
    assert np.max(np.abs(ht.grad.numpy() - fo.grad_h(pb, h, beta))) < 1e-12


def test_potts_gradient_rows_sum_to_zero():
    b = small_graph(10, 0.5, 24, pm1=False)
    inst = wl.Instance(wl.BMINCUT, b.n, 6, b.row_ptr, b.col_idx, None)
    g = fo.grad_h(as_problem(inst), np.random.default_rng(1).normal(size=inst.n * 6), 2.0, 0.4).reshape(inst.n, 6)
    assert np.max(np.abs(g.sum(axis=1))) < 1e-14


def test_two_state_potts_path_equals_sigmoid_path():
    """MaxCut(W) has the same free energy as the q=2 Potts cut with weights -W and lambda = 0, up to a
    constant (Eq.9 vs Eq.10); the softmax code path must reproduce the sigmoid one."""
    inst = small_graph(12, 0.5, 25, real=True)
    potts = wl.Instance(wl.BMINCUT, inst.n, 2, inst.row_ptr, inst.col_idx, -inst.weight)
    rng = np.random.default_rng(2)
    h = rng.normal(size=inst.n)
    off = rng.normal(size=inst.n)                       # softmax shift invariance too
    h2 = np.stack([off, off + h], axis=1).ravel()
    g_sig = fo.grad_h(as_problem(inst), h, 1.3)
    g_soft = fo.grad_h(as_problem(potts), h2, 1.3, 0.0).reshape(inst.n, 2)
    assert np.max(np.abs(g_soft[:, 1] - g_sig)) < 1e-13
    assert np.max(np.abs(g_soft[:, 0] + g_sig)) < 1e-13


def test_maxcut_is_ising_with_J_minus_half_W():
    inst = small_graph(12, 0.5, 26, real=True)
    ising = wl.sparse_ising_from(inst, scale=-0.5)
    h = np.random.default_rng(8).normal(size=inst.n)
    a = fo.grad_h(as_problem(inst), h, 0.9)
    b = fo.grad_h(as_problem(ising), h, 0.9)
    assert np.max(np.abs(a - b)) < 1e-14
    # free energies differ by the constant -sum_E W/2
    const = -0.5 * dense_W(inst)[np.triu_indices(inst.n, 1)].sum()
    assert abs(fo.free_energy(as_problem(inst), h, 0.9) - fo.free_energy(as_problem(ising), h, 0.9) - const) < 1e-12


def test_dense_and_sparse_ising_agree():
    sk = wl.sk_dense(10, 27)
    J = sk.dense_J.astype(np.float64)
    iu, ju = np.triu_indices(10, 1)
    row_ptr, col, w = wl.csr_from_edges(10, iu, ju, J[iu, ju].astype(np.float32))
    sp = wl.Instance(wl.ISING, 10, 2, row_ptr, col, w)
    h = np.random.default_rng(9).normal(size=10)
    assert np.max(np.abs(fo.grad_h(as_problem(sk), h, 2.0) - fo.grad_h(as_problem(sp), h, 2.0))) < 1e-14
