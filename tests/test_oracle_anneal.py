"""Pins for the oracle's iteration: mean-field fixed points (S40), the step plumbing, and
brute-force optima on n <= 20 (north_star check 4).  CPU only."""
import itertools
import math

import numpy as np
import pytest

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem, small_graph, dense_W


def test_two_node_antiferromagnetic_fixed_point():
    """Single edge W=1: stationary points of F obey m1 = -m2 = m with m = tanh(beta m / 2), non-zero iff
    beta > 2 (S39-S40, PAPER.md:1924-1932 with J = -W/2)."""
    row_ptr, col, _ = wl.csr_from_edges(2, np.array([0]), np.array([1]), None)
    pb = fo.Problem(kind=fo.MAXCUT, n=2, q=2, row_ptr=row_ptr, col_idx=col)
    for beta in (1.5, 3.0, 6.0):
        if beta <= 2:                                  # only the paramagnet: descent ends at m = 0
            h = np.array([0.3, -0.2])
            for _ in range(20000):
                h -= 0.5 * fo.grad_h(pb, h, beta)
            assert np.max(np.abs(np.tanh(h / 2))) < 1e-6
            continue
        x = 0.9                                        # solve m = tanh(beta m / 2) by iteration
        for _ in range(10000):
            x = math.tanh(beta * x / 2)
        assert x > 0.1
        hstar = 2 * math.atanh(x)
        assert np.max(np.abs(fo.grad_h(pb, np.array([hstar, -hstar]), beta))) < 1e-14      # stationary
        assert np.max(np.abs(fo.grad_h(pb, np.array([hstar, hstar]), beta))) > 1e-3        # ferro is not
        if beta == 3.0:                                # and descent from a generic start finds it
            h = np.array([0.3, -0.2])
            for _ in range(40000):
                h -= 0.5 * fo.grad_h(pb, h, beta)
            m = np.tanh(h / 2)
            assert abs(m[0] + m[1]) < 1e-9 and abs(abs(m[0]) - x) < 1e-8


def test_gradient_descent_reaches_mean_field_equations():
    """At constant beta the minimiser of F satisfies m_i = tanh(beta sum_j J_ij m_j) (S40);
    MaxCut maps to J = -W/2."""
    inst = small_graph(14, 0.4, 41, pm1=True)
    pb = as_problem(inst)
    J = -0.5 * dense_W(inst)
    beta = 1.2
    h = np.random.default_rng(0).normal(size=inst.n) * 0.5
    for _ in range(40000):
        h -= 0.3 * fo.grad_h(pb, h, beta)
    for _ in range(2000):                              # saturated spins move slowly: finish with steps scaled by 1/(p(1-p))
        p = 1 / (1 + np.exp(-h))
        h -= 0.3 * fo.grad_h(pb, h, beta) / (p * (1 - p))
    m = np.tanh(h / 2)
    assert np.max(np.abs(m - np.tanh(beta * J @ m))) < 1e-12
    assert np.max(np.abs(m)) > 0.05                    # a non-trivial solution, not the paramagnet


@pytest.mark.parametrize("kind", ["maxcut", "bmincut", "maxsat"])
def test_step_is_synchronous_gradient_then_adam(kind):
    """femo_anneal == for each t: g = grad_h(h(t)) on every replica, Adam with count t+1, beta[t]
    (p for the whole tensor, then backward, then optimizer.step())."""
    if kind == "maxcut":
        inst, lam = small_graph(12, 0.5, 42), 0.0
    elif kind == "bmincut":
        b = small_graph(10, 0.5, 43, pm1=False)
        inst, lam = wl.Instance(wl.BMINCUT, b.n, 3, b.row_ptr, b.col_idx, None), 0.2
    else:
        inst, lam = wl.random_ksat(12, 40, 3, 44), 0.0
    pb = as_problem(inst)
    R, N = 3, 7
    beta = fo.schedule_inverse_proportional(1.0, 0.1, N)
    adam = fo.Adam()
    h0 = fo.init_fields(5, R, inst.n, pb.fields_per_var, 1e-3)
    st = fo.anneal(fo.State(pb, h0), beta, adam, lam)
    h = h0.reshape(R, -1).copy()
    m1, m2 = np.zeros_like(h), np.zeros_like(h)
    for t in range(N):
        g = np.stack([fo.grad_h(pb, h[a], beta[t], lam) for a in range(R)])
        for a in range(R):
            fo.adam_update(adam, t + 1, h[a], m1[a], m2[a], g[a])
    assert np.array_equal(st.h.reshape(R, -1), h)
    # resumability: 3 steps + 4 steps == 7 steps
    st2 = fo.anneal(fo.State(pb, h0), beta, adam, lam, t_end=3)
    st2 = fo.anneal(st2, beta, adam, lam)
    assert np.array_equal(st2.h, st.h)
    # OpenMP build shards replicas only: identical numbers
    st3 = fo.anneal(fo.State(pb, h0), beta, adam, lam, openmp=True)
    assert np.array_equal(st3.h, st.h)


def brute_force_maxcut(W):
    n = W.shape[0]
    iu, ju = np.triu_indices(n, 1)
    w = W[iu, ju]
    best = -np.inf
    codes = np.arange(1 << (n - 1), dtype=np.int64)          # fix spin n-1 = 0 (global flip symmetry)
    bits = ((codes[:, None] >> np.arange(n)[None]) & 1).astype(np.int8)
    for lo in range(0, codes.size, 1 << 14):
        b = bits[lo:lo + (1 << 14)]
        cut = ((b[:, iu] != b[:, ju]) * w[None]).sum(1)
        best = max(best, cut.max())
    return best


def test_anneal_reaches_brute_force_optimum_small_graphs():
    """Config-0 schedule (R=32, 500 steps, T 1 -> 0.01, Adam 0.1) on a fixed seeded set of 12 graphs,
    n = 14..18, unit and +-1 weights; at least 90% must reach the exact optimum."""
    hits, total = 0, 0
    beta = fo.schedule_inverse_proportional(1.0, 0.01, 500)
    for k in range(12):
        n = 14 + k % 5
        inst = small_graph(n, 0.5, 100 + k, pm1=(k % 2 == 1))
        pb = as_problem(inst)
        st = fo.anneal(fo.State(pb, fo.init_fields(0, 32, n, 1, 1e-3)), beta, fo.Adam())
        cfg = fo.round_configs(pb, st.h)
        e_int, e_real, _ = fo.energies(pb, cfg)
        best = -e_int[fo.argmin(e_real)]
        opt = brute_force_maxcut(dense_W(inst))
        assert best <= opt
        hits += int(best == opt)
        total += 1
    assert hits >= math.ceil(0.9 * total), (hits, total)


def test_anneal_small_maxsat_and_bmincut_reach_brute_force():
    beta = fo.schedule_inverse_proportional(1.0, 0.01, 500)
    # Max-3-SAT, n = 12: enumerate 4096 assignments
    inst = wl.random_ksat(12, 70, 3, 45)
    pb = as_problem(inst)
    allcfg = np.array(list(itertools.product([0, 1], repeat=12)), dtype=np.int32)
    opt = fo.energies(pb, allcfg)[0].min()
    st = fo.anneal(fo.State(pb, fo.init_fields(0, 32, 12, 1, 1e-3)), beta, fo.Adam())
    e_int, e_real, _ = fo.energies(pb, fo.round_configs(pb, st.h))
    assert e_int.min() >= opt and e_int[fo.argmin(e_real)] == opt
    # bMinCut q=3, n = 9: enumerate 3^9 configurations of the stated energy
    b = small_graph(9, 0.5, 46, pm1=False)
    lam = 0.5
    binst = wl.Instance(wl.BMINCUT, 9, 3, b.row_ptr, b.col_idx, None)
    bpb = as_problem(binst)
    allcfg = np.array(list(itertools.product([0, 1, 2], repeat=9)), dtype=np.int32)
    opt = fo.energies(bpb, allcfg, lam)[1].min()
    st = fo.anneal(fo.State(bpb, fo.init_fields(0, 32, 9, 3, 1e-3)), beta, fo.Adam(), lam)
    e_int, e_real, part = fo.energies(bpb, fo.round_configs(bpb, st.h), lam)
    assert e_real.min() >= opt - 1e-12 and abs(e_real[fo.argmin(e_real)] - opt) < 1e-12


def test_rounding_rule():
    b = small_graph(4, 0.9, 47)
    assert fo.round_configs(as_problem(b), np.array([[-1.0, 0.0, 1e-30, 2.0]])).tolist() == [[0, 0, 1, 1]]
    pb = as_problem(wl.Instance(wl.BMINCUT, 2, 3, b.row_ptr[:3], b.col_idx, None))
    assert fo.round_configs(pb, np.array([[[0.5, 0.5, 0.1], [0.0, 0.2, 0.2]]])).tolist() == [[0, 1]]
