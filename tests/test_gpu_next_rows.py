"""GPU parity for the SURVEY.md section 8(f) rows: RMSprop / SGD optimisers and the manipulated gradients
(one-hot neighbours, per-node normalisation, gamma_grad), CUDA path against the oracle.

Floating point decides an integer here (sgn(m_j), the argmax behind the one-hot vectors), so:
  * with the wide phase over all steps both sides hold fp64 state and take every such decision alike: the
    marginals must agree to the fp32 rounding of the returned values;
  * the fp32 bulk kernels are checked ONE STEP AT A TIME from the GPU's own fp32 state handed to the oracle
    (fields and moments are exactly representable), skipping the rare variables next to a decision within
    rounding distance of a tie.
"""
import numpy as np
import pytest

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem
from test_gpu_parity import get, MARGINAL_TOL, WIDE_TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fem():
    from paper_2412_09285_b200 import fem as femlib
    return femlib


OPTS = {
    "rmsprop_mom": dict(optimizer=1, lr=0.02, alpha=0.9, momentum=0.5, weight_decay=0.001),
    "rmsprop": dict(optimizer=1, lr=0.02, alpha=0.99),
    "sgd_mom": dict(optimizer=2, lr=0.5, momentum=0.8, dampening=0.1),
    "sgd": dict(optimizer=2, lr=0.5, weight_decay=0.002),
    "adam": dict(optimizer=0, lr=0.1),
}


def oracle_opt(o):
    return fo.Optimizer(kind=o["optimizer"], lr=o["lr"], alpha=o.get("alpha", 0.99), momentum=o.get("momentum", 0.0),
                        dampening=o.get("dampening", 0.0), weight_decay=o.get("weight_decay", 0.0))


NAMES = ["maxcut_torus_30x34", "maxcut_reg3_pm1", "maxcut_er_odd_R", "ising_sparse", "ising_dense_sk",
         "bmincut_q8_reg10", "bmincut_q5_weighted", "maxsat_k4"]


@pytest.mark.parametrize("opt", ["rmsprop_mom", "rmsprop", "sgd_mom", "sgd"])
@pytest.mark.parametrize("name", NAMES)
def test_optimisers_exact_gradient(fem, name, opt):
    inst, R = get(name)
    o = OPTS[opt]
    steps = 500
    beta = fem.linear_temperature_schedule(1.0, 0.01, steps)
    h0 = fo.init_fields(1, R, inst.n, inst.fields_per_var).astype(np.float32)
    pb = as_problem(inst)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, oracle_opt(o), inst.lam, t_end=50)
    P_ref = fo.marginals(pb, st.h)
    # fp32 from step 8 on: north_star's 1e-4 bar was set for Adam; RMSprop with a short memory (alpha = 0.9) renormalises
    # rounding-level gradients every few steps and is chaotic at that level: its fp32 kernel is
    # covered by the step-by-step test below instead
    legs = ((50, WIDE_TOL),) if opt == "rmsprop_mom" else ((50, WIDE_TOL), (8, MARGINAL_TOL))
    for K, tol in legs:
        eng = fem.Fem(inst, R)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=K, **o), R, stop_after=50)
        P = eng.get_marginals().astype(np.float64)
        err = np.max(np.abs(P - P_ref.reshape(P.shape)))
        assert err < tol, (K, err)
        m1, m2 = eng.get_moments()
        if K == 50:
            assert np.max(np.abs(m1 - st.m1.reshape(m1.shape))) <= 1e-5 * max(1.0, np.max(np.abs(st.m1)))
            assert np.max(np.abs(m2 - st.m2.reshape(m2.shape))) <= 1e-5 * max(1e-12, np.max(np.abs(st.m2)))
        eng.close()


MANIP = ["maxcut_torus_30x34", "maxcut_reg3_pm1", "maxcut_er_odd_R", "cfg0_maxcut_er800", "ising_sparse",
         "bmincut_q8_reg10", "bmincut_q3_reg6_odd_R", "bmincut_q5_weighted", "maxsat_k4", "ising_dense_sk"]


@pytest.mark.parametrize("opt", ["rmsprop_mom", "adam", "sgd_mom"])
@pytest.mark.parametrize("name", MANIP)
def test_manipulated_gradients_wide_phase(fem, name, opt):
    """fp64 state on both sides: every sgn / argmax decision is taken alike, marginals agree after 50 steps."""
    inst, R = get(name)
    o = OPTS[opt]
    beta = fem.exponential_schedule(0.5, 50.0, 400)
    h0 = fo.init_fields(2, R, inst.n, inst.fields_per_var).astype(np.float32)
    pb = as_problem(inst)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, oracle_opt(o), inst.lam, t_end=50, manipulated=True,
                      gamma=0.8)
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    eng.anneal(fem.Schedule(beta=beta, precise_steps=50, manipulated=True, gamma_grad=0.8, **o), R, stop_after=50)
    P = eng.get_marginals().astype(np.float64)
    err = np.max(np.abs(P - fo.marginals(pb, st.h).reshape(P.shape)))
    assert err < WIDE_TOL, err
    eng.close()


@pytest.mark.parametrize("manipulated", [True, False])
@pytest.mark.parametrize("opt", ["rmsprop_mom", "sgd_mom"])
@pytest.mark.parametrize("name", ["maxcut_torus_30x34", "maxcut_reg3_pm1", "ising_sparse", "bmincut_q8_reg10",
                                  "bmincut_q5_weighted", "maxsat_k4", "ising_dense_sk"])
def test_fp32_kernels_step_by_step(fem, name, opt, manipulated):
    """The fp32 bulk kernels (stepwise, persistent, Potts, dense CUDA-core): six single steps, each from the GPU's
    own state (fields and moments are exactly representable in the oracle's doubles)."""
    inst, R = get(name)
    o = OPTS[opt]
    beta = fem.exponential_schedule(0.5, 50.0, 400)
    pb = as_problem(inst)
    sch = fem.Schedule(beta=beta, precise_steps=30, manipulated=manipulated, gamma_grad=1.3, **o)
    eng = fem.Fem(inst, R)
    eng.anneal(sch, R, seed=6, stop_after=30)
    checked = 0
    for t in range(30, 36):
        h = eng.get_fields()
        m1, m2 = eng.get_moments()
        st = fo.State(pb, h.astype(np.float64))
        st.m1, st.m2, st.t = m1.astype(np.float64).reshape(st.h.shape), m2.astype(np.float64).reshape(st.h.shape), t
        fo.anneal_ex(st, beta, oracle_opt(o), inst.lam, t_end=t + 1, manipulated=manipulated, gamma=1.3)
        eng.anneal(sch, R, stop_after=t + 1)
        h1 = eng.get_fields().astype(np.float64)
        # both sides start the step from the SAME fp32 state, so every sgn / argmax decision of this step is identical
        diff = np.abs(h1 - st.h.reshape(h1.shape))
        scale = np.maximum(1.0, np.abs(h1))
        assert np.all(diff <= 2e-5 * scale), (t, float(diff.max()))
        checked += diff.size
    assert checked == 6 * h1.size
    eng.close()


def test_manipulated_full_anneal_quality_cfg0(fem):
    """The paper's recipe on config 0's graph (RMSprop + manipulated gradients, exponential schedule): the GPU's
    mean final cut is within 0.5% of the oracle's (energy distribution, not trajectories)."""
    c = wl.CONFIGS["cfg0"]
    inst = c.make()
    pb = as_problem(inst)
    o = dict(optimizer=1, lr=0.05, alpha=0.9, momentum=0.5)
    beta = fem.exponential_schedule(0.5, 40.0, 400)
    h0 = fo.init_fields(0, c.R, inst.n, 1).astype(np.float32)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, oracle_opt(o), manipulated=True, gamma=1.0, openmp=True)
    ref = fo.energies(pb, fo.round_configs(pb, st.h))[0]
    eng = fem.Fem(inst, c.R)
    eng.set_fields(h0)
    eng.anneal(fem.Schedule(beta=beta, manipulated=True, **o), c.R)
    res = eng.result()
    assert eng.info("persist_launches") > 0
    assert abs(res["energy_int"].mean() - ref.mean()) <= 0.005 * abs(ref.mean())
    cfg = eng.get_configs()
    assert np.array_equal(fo.energies(pb, cfg)[0], res["energy_int"])
    eng.close()


@pytest.mark.parametrize("manipulated", [False, True])
@pytest.mark.parametrize("name", ["bmincut_q8_reg10", "bmincut_q5_weighted", "bmincut_q3_reg6_odd_R"])
def test_lambda_ramp(fem, name, manipulated):
    """The balance weight incremented linearly from 0 to lambda_max over the N steps (Table S3 :842)
    through fem_schedule.lambda[]: wide phase over 50 steps against the oracle's anneal(lam_t), then the fp32 kernels
    (TMA-staged and register Potts paths) for the rest of the ramp; the readout uses the LAST step's lambda."""
    inst, R = get(name)
    N = 120
    beta = fem.exponential_schedule(0.5, 30.0, N)
    lam = np.linspace(0.0, 0.2, N)
    h0 = fo.init_fields(4, R, inst.n, inst.fields_per_var).astype(np.float32)
    pb = as_problem(inst)
    opt = fo.Optimizer(kind=fo.ADAM, lr=0.05)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, opt, 123.0, lam_t=lam, t_end=50,
                      manipulated=manipulated, gamma=0.9)
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    eng.anneal(fem.Schedule(beta=beta, lam=lam, lr=0.05, precise_steps=50, manipulated=manipulated, gamma_grad=0.9), R,
               stop_after=50)
    P = eng.get_marginals().astype(np.float64)
    err = np.max(np.abs(P - fo.marginals(pb, st.h).reshape(P.shape)))
    assert err < WIDE_TOL, err
    eng.close()
    if not manipulated:
        # north_star's fp32 bar (1e-4 at step 50, default precise_steps) is stated for the BASELINE schedule shape (T linear
        # 1.0 -> 0.01, Adam lr 0.1): the same ramp under that schedule
        N2 = 500
        beta2, lam2 = fem.linear_temperature_schedule(1.0, 0.01, N2), np.linspace(0.0, 0.2, N2)
        st2 = fo.anneal(fo.State(pb, h0.astype(np.float64)), beta2, fo.Adam(), 123.0, lam_t=lam2, t_end=50)
        eng = fem.Fem(inst, R)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta2, lam=lam2, precise_steps=8), R, stop_after=50)
        P = eng.get_marginals().astype(np.float64)
        err = np.max(np.abs(P - fo.marginals(pb, st2.h).reshape(P.shape)))
        assert err < MARGINAL_TOL, err
        eng.close()
    # fp32 kernels one step at a time along the ramp, from the GPU's own state
    sch = fem.Schedule(beta=beta, lam=lam, lr=0.05, precise_steps=4, manipulated=manipulated, gamma_grad=0.9)
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    eng.anneal(sch, R, stop_after=60)
    for t in range(60, 64):
        h = eng.get_fields()
        m1, m2 = eng.get_moments()
        s2 = fo.State(pb, h.astype(np.float64))
        s2.m1, s2.m2, s2.t = m1.astype(np.float64).reshape(s2.h.shape), m2.astype(np.float64).reshape(s2.h.shape), t
        fo.anneal_ex(s2, beta, opt, 123.0, lam_t=lam, t_end=t + 1, manipulated=manipulated, gamma=0.9)
        eng.anneal(sch, R, stop_after=t + 1)
        h1 = eng.get_fields().astype(np.float64)
        assert np.all(np.abs(h1 - s2.h.reshape(h1.shape)) <= 2e-5 * np.maximum(1.0, np.abs(h1))), t
    # the whole ramp; energies reported with lambda_max (the last step's value)
    eng.anneal(sch, R)
    res = eng.result()
    cfg = eng.get_configs()
    e_int, e_real, part = fo.energies(pb, cfg, float(lam[-1]))
    assert np.array_equal(res["energy_int"], e_int) and np.array_equal(res["energy"], e_real)
    assert np.array_equal(res["part_sizes"], part)
    eng.close()


def test_optimiser_cannot_change_inside_a_trajectory(fem):
    inst, R = get("maxcut_torus_30x34")
    beta = fem.linear_temperature_schedule(1.0, 0.01, 20)
    eng = fem.Fem(inst, R)
    eng.anneal(fem.Schedule(beta=beta), R, stop_after=10)
    with pytest.raises(fem.FemError):
        eng.anneal(fem.Schedule(beta=beta, optimizer=2, lr=0.5), R)
    with pytest.raises(fem.FemError):
        eng.anneal(fem.Schedule(beta=beta, manipulated=True), R)
    eng.anneal(fem.Schedule(beta=beta), R)           # the same optimiser continues
    eng.reset()
    eng.anneal(fem.Schedule(beta=beta, optimizer=2, lr=0.5), R)   # a new trajectory may use another
    eng.close()


def test_bad_optimiser_arguments_are_rejected(fem):
    inst, R = get("maxcut_torus_30x34")
    beta = fem.linear_temperature_schedule(1.0, 0.01, 10)
    eng = fem.Fem(inst, R)
    for bad in (dict(optimizer=3), dict(optimizer=1, alpha=1.0), dict(optimizer=2, dampening=1.5),
                dict(optimizer=2, momentum=-0.1), dict(manipulated=True, gamma_grad=0.0)):
        with pytest.raises(fem.FemError):
            eng.anneal(fem.Schedule(beta=beta, **bad), R)
    eng.close()
