"""GPU parity for non-Boolean SAT: fem_problem.lit_state (ABI 4),
k_step_qsat.cu against the oracle.  Bars as in tests/test_gpu_parity.py."""
import numpy as np
import pytest

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem
from test_gpu_parity import MARGINAL_TOL, WIDE_TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fem():
    from paper_2412_09285_b200 import fem as femlib
    return femlib


CASES = {
    # name: (q, k, kmin, n, m, R, replica_block)
    "q3_k3_R8": (3, 3, None, 150, 900, 8, 0),
    "q5_k1to4_R6": (5, 4, 1, 120, 700, 6, 0),             # clause lengths 1..4, R not a multiple of 4 (one replica per thread)
    "q8_k2_R16_rb4": (8, 2, None, 100, 1500, 16, 4),      # four replica blocks
    "q2_k5_R8": (2, 5, 3, 90, 500, 8, 0),                 # two states through the q-state path
}


def make(name):
    q, k, kmin, n, m, R, rb = CASES[name]
    return wl.random_qsat(n, m, k, q, 2100 + q, kmin=kmin), R, rb


@pytest.mark.parametrize("opt", ["adam", "sgd_mom"])
@pytest.mark.parametrize("name", list(CASES))
def test_qsat_marginals_and_energies(fem, name, opt):
    inst, R, rb = make(name)
    pb = as_problem(inst)
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    extra = {} if opt == "adam" else dict(optimizer=2, lr=0.5, momentum=0.8, dampening=0.1)
    oopt = fo.Optimizer() if opt == "adam" else fo.Optimizer(kind=2, lr=0.5, momentum=0.8, dampening=0.1)
    h0 = fo.init_fields(3, R, inst.n, inst.q).astype(np.float32)
    st = fo.anneal_ex(fo.State(pb, h0.astype(np.float64)), beta, oopt, t_end=50)
    P_ref = fo.marginals(pb, st.h)
    for K, tol in ((50, WIDE_TOL), (8, MARGINAL_TOL)):
        eng = fem.Fem(inst, R)
        if rb:
            eng.set_option("replica_block", rb)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=K, **extra), R, stop_after=50)
        P = eng.get_marginals().astype(np.float64)
        assert P.shape[-1] == inst.q and np.max(np.abs(P - P_ref.reshape(P.shape))) < tol, (name, K)
        res = eng.result()
        cfg = eng.get_configs()
        assert np.array_equal(cfg, fo.round_configs(pb, eng.get_fields().astype(np.float64)))
        e_int, e_real, _ = fo.energies(pb, cfg)
        assert np.array_equal(res["energy_int"], e_int) and np.array_equal(res["energy"], e_real)
        assert res["best_replica"] == fo.argmin(e_real)
        # energies of caller-supplied configurations: the plain definition, bit-exact
        rnd = np.random.default_rng(1).integers(0, inst.q, (R, inst.n)).astype(np.int32)
        got = eng.energy_of(rnd)
        assert np.array_equal(got[0], fo.energies(pb, rnd)[0])
        eng.close()


def test_qsat_full_anneal_energy_distribution(fem):
    """north_star criterion 3: the whole anneal, seeded fields from the library's own generator, mean unsat count within
    0.5% of the oracle's (or within one clause over the replicas when the mean is that small)."""
    inst, R, _ = make("q3_k3_R8")
    R = 32
    pb = as_problem(inst)
    steps = 400
    beta = fem.linear_temperature_schedule(1.0, 0.01, steps)
    st = fo.anneal(fo.State(pb, fo.init_fields(7, R, inst.n, inst.q)), beta, fo.Adam(), openmp=True)
    e_ref = fo.energies(pb, fo.round_configs(pb, st.h))[1]
    eng = fem.Fem(inst, R)
    eng.anneal(fem.Schedule(beta=beta), R, seed=7)
    res = eng.result()
    assert np.array_equal(res["energy_int"], fo.energies(pb, eng.get_configs())[0])
    assert abs(res["energy"].mean() - e_ref.mean()) <= max(0.005 * abs(e_ref.mean()), 1.0 / R * 4)
    eng.close()


def test_bad_qsat_problems_are_rejected(fem):
    inst, R, _ = make("q3_k3_R8")
    for bad in ("state_out_of_range", "negative_literal", "q9", "on_maxcut", "boolean_q3"):
        lits, st, q, kind = inst.lits.copy(), inst.lit_state.copy(), inst.q, wl.MAXSAT
        if bad == "state_out_of_range":
            st[5] = 3
        elif bad == "negative_literal":
            lits[5] = -lits[5]
        elif bad == "q9":
            q = 9
        elif bad == "boolean_q3":
            st = None
        x = wl.Instance(kind, inst.n, q, m=inst.m, clause_ptr=inst.clause_ptr, lits=lits, lit_state=st)
        if bad == "on_maxcut":
            ring = wl.torus_maxcut(3, 1, W=4)
            x = wl.Instance(wl.MAXCUT, ring.n, 2, ring.row_ptr, ring.col_idx, ring.weight, lit_state=np.zeros(4, np.int32))
        with pytest.raises(fem.FemError):
            fem.Fem(x, 4)
