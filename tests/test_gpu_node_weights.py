"""GPU parity for the node-weighted balance term of bMinCut (S33-S35):
the CUDA path (fem_problem.node_weight, ABI 4) against the oracle.  Same bars as tests/test_gpu_parity.py: wide phase
over all steps <= 2e-7 on the marginals, default launch configuration <= 1e-4 at step 50, energies and part sizes of the
GPU's configurations bit-exact, mean final energy within 0.5%."""
import numpy as np
import pytest

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem
from test_gpu_parity import MARGINAL_TOL, WIDE_TOL, edge_ids

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fem():
    from paper_2412_09285_b200 import fem as femlib
    return femlib


def weighted_instance(name):
    rng = np.random.default_rng(17)
    if name == "q8_reg10_R16_rb8":              # state-innermost kernel (cfg 2's shape), two replica blocks
        b = wl.random_regular(1200, 10, 2031, wl.BMINCUT, 8, lam=0.02)
        w, R, rb = None, 16, 8
    elif name == "q4_reg6_weighted_R32":        # state-innermost kernel, weighted edges, one variable per group
        b = wl.random_regular(1201, 6, 2032, wl.BMINCUT, 4, lam=0.03)
        w = rng.integers(1, 4, b.nnz // 2).astype(np.float32)[edge_ids(b)]
        w, R, rb = w, 32, 32
    elif name == "q5_er_irregular_R12":         # register path: q not 4 / 8, rows of different lengths, isolated nodes
        er = wl.erdos_renyi_maxcut(700, 0.008, 2033, pm1=False)
        b = wl.Instance(wl.BMINCUT, er.n, 5, er.row_ptr, er.col_idx, None, lam=0.05)
        w, R, rb = None, 12, 0
    else:                                        # q = 8 but n not a multiple of 32 / Rb: register path at q = 8
        b = wl.random_regular(1202, 3, 2034, wl.BMINCUT, 8, lam=0.04)
        w, R, rb = None, 8, 8
    V = rng.integers(1, 7, b.n).astype(np.float32)
    V[rng.integers(0, b.n, 5)] = 40.0            # a few heavy nodes
    return wl.Instance(wl.BMINCUT, b.n, b.q, b.row_ptr, b.col_idx, w, lam=b.lam, node_weight=V, name=name), R, rb


CASES = ["q8_reg10_R16_rb8", "q4_reg6_weighted_R32", "q5_er_irregular_R12", "q8_reg3_odd_n_R8"]


@pytest.mark.parametrize("manipulated", [False, True])
@pytest.mark.parametrize("name", CASES)
def test_node_weighted_marginals_and_energies(fem, name, manipulated):
    inst, R, rb = weighted_instance(name)
    pb = as_problem(inst)
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(2, R, inst.n, inst.q).astype(np.float32)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, fo.Optimizer(), inst.lam, t_end=50,
                      manipulated=manipulated, gamma=0.8)
    P_ref = fo.marginals(pb, st.h)
    for K, tol in ((50, WIDE_TOL), (8, MARGINAL_TOL)):
        if manipulated and K == 8:
            continue                               # fp32 argmax decisions: covered step by step in test_gpu_next_rows.py
        eng = fem.Fem(inst, R)
        if rb:
            eng.set_option("replica_block", rb)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=K, manipulated=manipulated, gamma_grad=0.8), R, stop_after=50)
        P = eng.get_marginals().astype(np.float64)
        assert np.max(np.abs(P - P_ref.reshape(P.shape))) < tol, (name, K)
        if K == 8 and name in ("q8_reg10_R16_rb8", "q4_reg6_weighted_R32"):
            assert eng.info("si_launches") == 42 * (R // eng.info("replica_block"))   # the state-innermost kernel ran
        res = eng.result()
        cfg = eng.get_configs()
        e_int, e_real, part = fo.energies(pb, cfg, inst.lam)
        assert np.array_equal(res["energy_int"], e_int) and np.array_equal(res["energy"], e_real)
        assert np.array_equal(res["part_sizes"], part)           # sums of V_i per part
        assert part.sum(axis=-1).min() == part.sum(axis=-1).max() == int(inst.node_weight.sum())
        eng.close()


def test_unit_node_weights_change_nothing(fem):
    """V = 1 given explicitly is the unweighted problem bit for bit (fields, energies), on both Potts kernels."""
    for name in ("q8_reg10_R16_rb8", "q5_er_irregular_R12"):
        inst, R, rb = weighted_instance(name)
        ones = wl.Instance(wl.BMINCUT, inst.n, inst.q, inst.row_ptr, inst.col_idx, inst.weight, lam=inst.lam,
                           node_weight=np.ones(inst.n, np.float32))
        none = wl.Instance(wl.BMINCUT, inst.n, inst.q, inst.row_ptr, inst.col_idx, inst.weight, lam=inst.lam)
        out = []
        for x in (ones, none):
            eng = fem.Fem(x, R)
            if rb:
                eng.set_option("replica_block", rb)
            eng.anneal(fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.05, 60), precise_steps=4), R, seed=9)
            out.append((eng.get_fields(), eng.result()))
            eng.close()
        assert np.array_equal(out[0][0], out[1][0])
        assert np.array_equal(out[0][1]["energy"], out[1][1]["energy"])
        assert np.array_equal(out[0][1]["part_sizes"], out[1][1]["part_sizes"])


def test_node_weighted_full_anneal_energy_distribution(fem):
    """north_star criterion 3 with node weights: whole anneal, mean final energy within 0.5% of the oracle's."""
    inst, R, rb = weighted_instance("q8_reg10_R16_rb8")
    pb = as_problem(inst)
    steps = 400
    beta = fem.linear_temperature_schedule(1.0, 0.01, steps)
    h0 = fo.init_fields(5, R, inst.n, inst.q)
    st = fo.anneal_ex(fo.State(pb, h0), beta, fo.Optimizer(), inst.lam, t_end=steps, openmp=True)
    _, e_ref, _ = fo.energies(pb, fo.round_configs(pb, st.h), inst.lam)
    eng = fem.Fem(inst, R)
    eng.set_option("replica_block", rb)
    eng.anneal(fem.Schedule(beta=beta), R, seed=5)
    res = eng.result()
    cfg = eng.get_configs()
    e_int, e_real, part = fo.energies(pb, cfg, inst.lam)
    assert np.array_equal(res["energy"], e_real) and np.array_equal(res["part_sizes"], part)
    assert abs(res["energy"].mean() - e_ref.mean()) <= 0.005 * abs(e_ref.mean())
    eng.close()


def test_bad_node_weights_are_rejected(fem):
    inst, R, _ = weighted_instance("q5_er_irregular_R12")
    for bad in ("zero", "fraction", "huge", "wrong_kind"):
        V = inst.node_weight.copy()
        kind, q = wl.BMINCUT, inst.q
        if bad == "zero":
            V[3] = 0.0
        elif bad == "fraction":
            V[3] = 1.5
        elif bad == "huge":
            V[3] = 4.0e6
        else:
            kind, q = wl.MAXCUT, 2
        x = wl.Instance(kind, inst.n, q, inst.row_ptr, inst.col_idx, None, lam=inst.lam, node_weight=V)
        with pytest.raises(fem.FemError):
            fem.Fem(x, 4)
