"""Pins for the oracle's non-Boolean SAT ("W_mi has q > 2 states"; Eq.8
PAPER.md:173, Eq.11 PAPER.md:218, S28 PAPER.md:650, S20 PAPER.md:599).  None of them re-types the oracle's formula: central
finite differences of F, torch autograd on Eq.11 written over explicit tensors, enumeration of the energy, the reduction
to the Boolean oracle at q = 2, saturation, and the brute-force optimum."""
import itertools

import numpy as np
import torch

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem


def tiny(q=3, n=7, m=12, k=3, seed=3, kmin=None):
    return wl.random_qsat(n, m, k, q, seed, kmin=kmin)


def test_gradient_matches_finite_differences_of_the_free_energy():
    for q, kmin in ((3, None), (5, 1), (2, 2)):
        inst = tiny(q=q, kmin=kmin)
        pb = as_problem(inst)
        rng = np.random.default_rng(q)
        for beta in (0.7, 3.0):
            h = rng.normal(0, 0.8, inst.n * q)
            g = fo.grad_h(pb, h, beta)
            for idx in rng.choice(h.size, 12, replace=False):
                e = np.zeros_like(h)
                e[idx] = 1e-5
                fd = (fo.free_energy(pb, h + e, beta) - fo.free_energy(pb, h - e, beta)) / 2e-5
                assert abs(fd - g[idx]) < 2e-8, (q, beta, idx)
            assert np.max(np.abs(g.reshape(inst.n, q).sum(axis=1))) < 1e-14      # S20: sum_s g^h_i(s) = 0


def test_gradient_matches_autograd_on_eq11():
    """Eq.11: F = sum_m prod_{i in dm} [1 - P_i(W_mi)] + (1/beta) sum_i sum_s P_i(s) ln P_i(s), P = softmax(h)."""
    inst = tiny(q=4, n=9, m=20, k=4, seed=8, kmin=2)
    pb = as_problem(inst)
    beta = 1.7
    h = torch.tensor(np.random.default_rng(1).normal(0, 1, (inst.n, 4)), dtype=torch.float64, requires_grad=True)
    P = torch.softmax(h, dim=1)
    U = 0.0
    for c in range(inst.m):
        sl = slice(int(inst.clause_ptr[c]), int(inst.clause_ptr[c + 1]))
        U = U + torch.prod(1.0 - P[torch.tensor(inst.lits[sl] - 1, dtype=torch.long), torch.tensor(inst.lit_state[sl], dtype=torch.long)])
    F = U + (P * torch.log_softmax(h, dim=1)).sum() / beta
    F.backward()
    g = fo.grad_h(pb, h.detach().numpy().ravel(), beta)
    assert np.max(np.abs(g - h.grad.numpy().ravel())) < 1e-13
    assert abs(fo.free_energy(pb, h.detach().numpy().ravel(), beta) - float(F.detach())) < 1e-12


def test_two_states_reduce_to_the_boolean_oracle():
    """q = 2 with clause values W: literal +v <=> W = 1, -v <=> W = 0; fields h(0) = a, h(1) = a + h_bool
    (PAPER.md:661).  Energy, free energy, marginals and g^h(1) = -g^h(0) = the two-state gradient."""
    q2 = tiny(q=2, n=8, m=15, k=3, seed=5)
    signed = np.where(q2.lit_state == 1, q2.lits, -q2.lits).astype(np.int32)
    boolean = wl.Instance(wl.MAXSAT, q2.n, 2, m=q2.m, clause_ptr=q2.clause_ptr, lits=signed)
    pq, pbool = as_problem(q2), as_problem(boolean)
    rng = np.random.default_rng(2)
    hb = rng.normal(0, 1.2, q2.n)
    a = rng.normal(0, 1, q2.n)
    hq = np.stack([a, a + hb], axis=1).ravel()
    assert abs(fo.free_energy(pq, hq, 2.0) - fo.free_energy(pbool, hb, 2.0)) < 1e-12
    assert np.max(np.abs(fo.marginals(pq, hq).reshape(-1, 2)[:, 1] - fo.marginals(pbool, hb))) < 1e-15
    gq, gb = fo.grad_h(pq, hq, 2.0).reshape(-1, 2), fo.grad_h(pbool, hb, 2.0)
    assert np.max(np.abs(gq[:, 1] - gb)) < 1e-13 and np.max(np.abs(gq[:, 0] + gb)) < 1e-13
    cfg = rng.integers(0, 2, (5, q2.n)).astype(np.int32)
    assert np.array_equal(fo.energies(pq, cfg)[0], fo.energies(pbool, cfg)[0])


def test_energy_by_enumeration_and_saturation():
    inst = tiny(q=3, n=6, m=14, k=3, seed=11, kmin=1)
    pb = as_problem(inst)
    cfgs = np.array(list(itertools.product(range(3), repeat=inst.n)), dtype=np.int32)
    e_int, e_real, _ = fo.energies(pb, cfgs)
    # plain definition (Eq.8): a clause counts when no variable takes its clause value
    want = np.zeros(len(cfgs), dtype=np.int64)
    for c in range(inst.m):
        sl = slice(int(inst.clause_ptr[c]), int(inst.clause_ptr[c + 1]))
        want += np.all(cfgs[:, inst.lits[sl] - 1] != inst.lit_state[sl][None, :], axis=1)
    assert np.array_equal(e_int, want) and np.array_equal(e_real, want.astype(np.float64))
    # one-hot marginals: U_MF is the integer energy, entropy and gradient vanish
    for row in (0, 100, 517):
        h = np.full((inst.n, 3), -40.0)
        h[np.arange(inst.n), cfgs[row]] = 40.0
        assert abs(fo.internal_energy(pb, h.ravel()) - want[row]) < 1e-12
        assert abs(fo.entropy(pb, h.ravel())) < 1e-12 and np.max(np.abs(fo.grad_h(pb, h.ravel(), 5.0))) < 1e-12
    assert np.array_equal(fo.round_configs(pb, h.ravel()[None, :]), cfgs[517][None, :])


def test_anneal_reaches_the_brute_force_optimum():
    hits = 0
    for seed in range(6):
        inst = tiny(q=3, n=8, m=30, k=3, seed=40 + seed)
        pb = as_problem(inst)
        cfgs = np.array(list(itertools.product(range(3), repeat=inst.n)), dtype=np.int32)
        best = fo.energies(pb, cfgs)[0].min()
        st = fo.State(pb, fo.init_fields(seed, 16, inst.n, 3))
        fo.anneal(st, fo.schedule_inverse_proportional(1.0, 0.01, 300), fo.Adam())
        hits += fo.energies(pb, fo.round_configs(pb, st.h))[0].min() == best
    assert hits >= 5
