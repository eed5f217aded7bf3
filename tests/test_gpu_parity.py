"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Bars (north_star): integer energies bit-exact; marginals within 1e-4 absolute
after the first 50 steps from identical initial fields; mean final energy within 0.5%."""
import numpy as np
import pytest

from oracle import fem_oracle as fo
from paper_2412_09285_b200 import workloads as wl
from test_oracle_gradient import as_problem

pytestmark = pytest.mark.gpu

MARGINAL_TOL = 1e-4       # north_star: absolute, after 50 steps
WIDE_TOL = 2e-7          # fp64 state on both sides; the marginals come back as fp32


@pytest.fixture(scope="module")
def fem():
    from paper_2412_09285_b200 import fem as femlib
    return femlib


def small_instances():
    reg = wl.random_regular(1500, 10, 2002, wl.BMINCUT, 8, lam=0.05 / 1500)
    reg3 = wl.random_regular(999, 6, 2003, wl.BMINCUT, 3, lam=0.01)
    er = wl.erdos_renyi_maxcut(300, 0.1, 2004, pm1=False)
    potts_w = wl.Instance(wl.BMINCUT, er.n, 5, er.row_ptr, er.col_idx,
                          (np.random.default_rng(1).integers(1, 4, er.nnz // 2).astype(np.float32))[
                              edge_ids(er)], lam=0.02)
    return {
        "cfg0_maxcut_er800": (wl.CONFIGS["cfg0"].make(), 32),
        "maxcut_torus_30x34": (wl.torus_maxcut(30, 2001, W=34), 24),
        "maxcut_reg3_pm1": (wl.random_regular(5000, 3, 2005, wl.MAXCUT, pm1=True), 32),
        "maxcut_er_odd_R": (wl.erdos_renyi_maxcut(257, 0.08, 2006, pm1=True), 7),
        "ising_sparse": (wl.sparse_ising_from(wl.torus_maxcut(20, 2007), -0.5), 16),
        "ising_dense_sk": (wl.sk_dense(200, 2008), 40),            # R % 32 != 0: CUDA-core GEMM
        "ising_dense_sk_tc": (wl.sk_dense(328, 2011), 96),         # tcgen05 path: ragged row tile and k block, 3 column tiles
        "bmincut_q8_reg10": (reg, 16),
        "bmincut_q3_reg6_odd_R": (reg3, 10),
        "bmincut_q5_weighted": (potts_w, 12),
        "maxsat_k4": (wl.random_ksat(600, 6000, 4, 2009), 16),
        "maxsat_k3_odd_R": (wl.random_ksat(301, 1300, 3, 2010), 9),
    }


def edge_ids(inst):
    """Index of the undirected edge of every CSR entry (so both directions get the same weight)."""
    rows = np.repeat(np.arange(inst.n), np.diff(inst.row_ptr))
    a, b = np.minimum(rows, inst.col_idx), np.maximum(rows, inst.col_idx)
    _, inv = np.unique(a.astype(np.int64) * inst.n + b, return_inverse=True)
    return inv


INST = None


def get(name):
    global INST
    if INST is None:
        INST = small_instances()
    return INST[name]


NAMES = ["cfg0_maxcut_er800", "maxcut_torus_30x34", "maxcut_reg3_pm1", "maxcut_er_odd_R", "ising_sparse",
         "ising_dense_sk", "ising_dense_sk_tc", "bmincut_q8_reg10", "bmincut_q3_reg6_odd_R", "bmincut_q5_weighted", "maxsat_k4",
         "maxsat_k3_odd_R"]


def oracle_run(inst, h0, beta, steps, lam):
    pb = as_problem(inst)
    st = fo.State(pb, h0.astype(np.float64))
    fo.anneal(st, beta, fo.Adam(), lam, t_end=steps)
    return pb, st


@pytest.mark.parametrize("name", NAMES)
def test_marginals_after_50_steps(fem, name):
    inst, R = get(name)
    steps = 500
    beta = fem.linear_temperature_schedule(1.0, 0.01, steps)
    assert np.array_equal(beta, fo.schedule_inverse_proportional(1.0, 0.01, steps))
    h0 = fo.init_fields(0, R, inst.n, inst.fields_per_var).astype(np.float32)
    pb, st = oracle_run(inst, h0, beta, 50, inst.lam)
    P_ref = fo.marginals(pb, st.h)
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    assert np.array_equal(eng.get_fields(), h0)                      # layout round trip is exact
    # default launch configuration: wide (fp64) phase for the first 8 steps, fp32 afterwards
    eng.anneal(fem.Schedule(beta=beta, precise_steps=8), R, stop_after=50)
    P = eng.get_marginals().astype(np.float64)
    err = np.max(np.abs(P - P_ref.reshape(P.shape)))
    assert err < MARGINAL_TOL, err
    assert np.max(np.abs(eng.get_fields() - st.h.reshape(P.shape))) < 1e-3
    # wide phase over all 50 steps: the state is fp64 like the oracle's, only libm separates them
    eng.set_fields(h0)
    eng.anneal(fem.Schedule(beta=beta, precise_steps=50), R, stop_after=50)
    err64 = np.max(np.abs(eng.get_marginals().astype(np.float64) - P_ref.reshape(P.shape)))
    assert err64 < WIDE_TOL, err64
    # ... and the fp32 bulk kernel on its own: ten more steps from that state
    fo.anneal(st, beta, fo.Adam(), inst.lam, t_end=60)
    eng.anneal(fem.Schedule(beta=beta, precise_steps=50), R, stop_after=60)
    err60 = np.max(np.abs(eng.get_marginals().astype(np.float64) - fo.marginals(pb, st.h).reshape(P.shape)))
    assert err60 < 2e-5, err60
    eng.close()


@pytest.mark.parametrize("name", NAMES)
def test_first_steps_one_by_one(fem, name):
    """Steps 1, 2, 5, 10, 20 against the oracle (the first Adam steps normalise tiny gradients and are the
    sensitive ones), and resumability of fem_anneal."""
    inst, R = get(name)
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(3, R, inst.n, inst.fields_per_var).astype(np.float32)
    pb = as_problem(inst)
    st = fo.State(pb, h0.astype(np.float64))
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    sch = fem.Schedule(beta=beta, precise_steps=8)
    for stop in (1, 2, 5, 10, 20):
        fo.anneal(st, beta, fo.Adam(), inst.lam, t_end=stop)
        eng.anneal(sch, R, stop_after=stop)
        P = eng.get_marginals().astype(np.float64)
        err = np.max(np.abs(P - fo.marginals(pb, st.h).reshape(P.shape)))
        assert err < MARGINAL_TOL, (stop, err)
    m1, m2 = eng.get_moments()
    assert np.max(np.abs(m1 - st.m1.reshape(m1.shape))) < 1e-4 * max(1.0, np.max(np.abs(st.m1)))
    eng.close()


@pytest.mark.parametrize("name", NAMES)
def test_energies_bit_exact_on_random_configurations(fem, name):
    inst, R = get(name)
    pb = as_problem(inst)
    rng = np.random.default_rng(11)
    cfg = rng.integers(0, inst.q, size=(R, inst.n)).astype(np.int32)
    cfg[0] = 0                                                      # degenerate: everything in one state
    if R > 1:
        cfg[1] = np.arange(inst.n) % inst.q
    eng = fem.Fem(inst, R)
    e_int, e, part = eng.energy_of(cfg)
    r_int, r, rpart = fo.energies(pb, cfg, inst.lam)
    if inst.kind == wl.ISING:
        assert np.max(np.abs(e - r)) <= 1e-9 * max(1.0, np.max(np.abs(r)))
    else:
        assert np.array_equal(e_int, r_int)
        assert np.array_equal(e, r)                                 # fp64 energy bit-exact (integral weights)
    if inst.kind == wl.BMINCUT:
        assert np.array_equal(part, rpart)
    # fewer configurations than R_cap
    e1 = eng.energy_of(cfg[:1])
    assert e1[0][0] == e_int[0] and e1[1][0] == e[0]
    eng.close()


@pytest.mark.parametrize("name", ["cfg0_maxcut_er800", "bmincut_q8_reg10", "maxsat_k4", "ising_dense_sk"])
def test_readout_is_consistent_and_deterministic(fem, name):
    inst, R = get(name)
    pb = as_problem(inst)
    steps = 200
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, steps))
    outs = []
    for _ in range(2):
        eng = fem.Fem(inst, R)
        eng.anneal(sch, R, seed=5)
        res = eng.result()
        cfg = eng.get_configs()
        h = eng.get_fields()
        outs.append((res, cfg, h))
        eng.close()
    (res, cfg, h), (res2, cfg2, h2) = outs
    assert np.array_equal(h, h2) and np.array_equal(cfg, cfg2)       # bit-identical run to run
    assert np.array_equal(res["energy"], res2["energy"])
    # rounding rule on the final fields (reading R3) and energies of exactly those configurations
    assert np.array_equal(cfg, fo.round_configs(pb, h.astype(np.float64)))
    r_int, r, rpart = fo.energies(pb, cfg, inst.lam)
    if inst.kind == wl.ISING:
        assert np.max(np.abs(res["energy"] - r)) <= 1e-9 * np.max(np.abs(r))
    else:
        assert np.array_equal(res["energy_int"], r_int) and np.array_equal(res["energy"], r)
    assert res["best_replica"] == int(np.argmin(res["energy"]))     # first minimum = lowest index on ties
    assert np.array_equal(res["best_config"], cfg[res["best_replica"]])


def test_seeded_initial_fields_match_oracle_generator(fem):
    inst, R = get("maxcut_torus_30x34")
    eng = fem.Fem(inst, R)
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, 10))
    eng.anneal(sch, R, seed=42, stop_after=0)
    h = eng.get_fields()
    ref = fo.init_fields(42, R, inst.n, 1).astype(np.float32)
    ulp = np.abs(h.view(np.int32).astype(np.int64) - ref.view(np.int32).astype(np.int64))
    assert ulp.max() <= 1 and np.mean(ulp == 0) > 0.999
    # Potts layout and a replica subset: replica a does not depend on R
    pinst, _ = get("bmincut_q3_reg6_odd_R")
    e2 = fem.Fem(pinst, 10)
    e2.anneal(sch, 4, seed=7, stop_after=0)
    ref = fo.init_fields(7, 10, pinst.n, 3).astype(np.float32)[:4]
    ulp = np.abs(e2.get_fields().view(np.int32).astype(np.int64) - ref.view(np.int32).astype(np.int64))
    assert ulp.max() <= 1
    eng.close(); e2.close()


@pytest.mark.parametrize("name", ["maxcut_torus_30x34", "bmincut_q8_reg10", "maxsat_k4"])
def test_replica_blocking_changes_nothing(fem, name):
    """Replicas are independent, so running them in L2-sized blocks (any order of blocks and steps) must give
    bit-identical fields."""
    inst, R = get(name)
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, 60))
    ref = None
    for blk, spb in ((0, 0), (R // 2, 1), (R // 2, 0), (R // 4, 7)):
        eng = fem.Fem(inst, R)
        eng.set_option("replica_block", blk)
        eng.set_option("steps_per_block", spb)
        eng.anneal(sch, R, seed=9)
        h = eng.get_fields()
        res = eng.result()
        if ref is None:
            ref = (h, res)
        else:
            assert np.array_equal(h, ref[0])
            assert np.array_equal(res["energy"], ref[1]["energy"]) and res["best_replica"] == ref[1]["best_replica"]
        eng.close()


def test_full_anneal_energy_distribution_cfg0(fem):
    """Config 0 in full: R=32, 500 steps; mean final energy over replicas within 0.5% of the oracle's."""
    c = wl.CONFIGS["cfg0"]
    inst = c.make()
    pb = as_problem(inst)
    beta = fem.linear_temperature_schedule(c.T_max, c.T_min, c.steps)
    h0 = fo.init_fields(0, c.R, inst.n, 1).astype(np.float32)
    st = fo.anneal(fo.State(pb, h0.astype(np.float64)), beta, fo.Adam())
    ref = fo.energies(pb, fo.round_configs(pb, st.h))[0]
    eng = fem.Fem(inst, c.R)
    eng.anneal(fem.schedule_for(c), c.R, seed=0)
    res = eng.result()
    assert abs(res["energy_int"].mean() - ref.mean()) <= 0.005 * abs(ref.mean())
    assert res["energy_int"].min() <= 0.995 * ref.min()              # energies are negative cuts
    eng.close()


def test_dense_tensor_core_path_is_taken_and_agrees_with_cuda_cores(fem):
    """Dense Ising: the tcgen05 int8 digit step (default) and the 3xTF32 step against the CUDA-core GEMM step on the same
    fields, and against the oracle; the info counters prove which kernel ran."""
    inst, R = get("ising_dense_sk_tc")
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(5, R, inst.n, 1).astype(np.float32)
    pb, st = oracle_run(inst, h0, beta, 30, inst.lam)
    P_ref = fo.marginals(pb, st.h)
    out = {}
    for tc in (1, 2, 0):                                            # int8 digit step (default), 3xTF32 step, CUDA cores
        eng = fem.Fem(inst, R)
        eng.set_option("tensor_cores", tc)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=8), R, stop_after=30)
        out[tc] = eng.get_marginals().astype(np.float64)
        assert (eng.info("tc_launches") == 22) == (tc != 0)         # 30 steps - 8 wide ones
        assert (eng.info("tc8_launches") == 22) == (tc == 1)
        assert np.max(np.abs(out[tc] - P_ref.reshape(out[tc].shape))) < MARGINAL_TOL
        print("tensor_cores", tc, "max |dP| vs oracle", np.max(np.abs(out[tc] - P_ref.reshape(out[tc].shape))))
        eng.close()
    assert np.max(np.abs(out[1] - out[0])) < MARGINAL_TOL and np.max(np.abs(out[2] - out[0])) < MARGINAL_TOL


@pytest.mark.parametrize("bn", [32, 64, 128, 256])
def test_dense_tensor_core_every_tile_size(fem, bn):
    """Each replica-tile width of the tcgen05 step (tc_tile_n) against the oracle, and two tile sizes one after the
    other on ONE handle (the tensor maps bake in the box height: they are rebuilt when it changes)."""
    inst = wl.sk_dense(328, 2011)
    R = 256                                                        # divisible by every tile width
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(5, R, inst.n, 1).astype(np.float32)
    pb, st = oracle_run(inst, h0[:24], beta, 30, inst.lam)         # the oracle follows 24 of the replicas
    P_ref = fo.marginals(pb, st.h).reshape(24, inst.n)
    eng = fem.Fem(inst, R)
    for tile in (bn, 64 if bn != 64 else 128):
        eng.reset()
        eng.set_option("tc_tile_n", tile)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=8), R, stop_after=30)
        P = eng.get_marginals().astype(np.float64)[:24]
        assert np.max(np.abs(P - P_ref)) < MARGINAL_TOL, tile
    assert eng.info("tc_launches") == 44
    eng.close()


def test_dense_tensor_core_phase_resumes_anywhere(fem):
    """Resume points inside the tensor-core phase with the parity hooks called in between (the hooks use the spare
    gather buffer as scratch; the transposed gather layout of this phase must survive them)."""
    inst, R = get("ising_dense_sk_tc")
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(5, R, inst.n, 1).astype(np.float32)
    pb, st = oracle_run(inst, h0, beta, 30, inst.lam)
    eng = fem.Fem(inst, R)
    eng.set_fields(h0)
    sch = fem.Schedule(beta=beta, precise_steps=8)
    for stop in (12, 13, 21, 30):                                  # resume points inside the tensor-core phase
        eng.anneal(sch, R, stop_after=stop)
        eng.get_marginals()
    P = eng.get_marginals().astype(np.float64)
    assert np.max(np.abs(P - fo.marginals(pb, st.h).reshape(P.shape))) < MARGINAL_TOL
    assert eng.info("tc_launches") == 22
    eng.close()


def _persist_cases():
    return {
        "cfg0_maxcut_er800": lambda: get("cfg0_maxcut_er800"),                       # unit weights, 1 variable per thread
        "maxcut_er_odd_R": lambda: get("maxcut_er_odd_R"),                           # +-1 weights, odd R (scalar rows)
        "ising_sparse": lambda: get("ising_sparse"),                                 # real weights, Ising sign
        "maxcut_er_n1500": lambda: (wl.erdos_renyi_maxcut(1500, 0.01, 2012, pm1=True), 12),   # 2 variables per thread
        "maxcut_torus_61x50": lambda: (wl.torus_maxcut(61, 2013, W=50), 20),          # 3050 nodes: 4 variables per thread
        "maxsat_k4_n300": lambda: (wl.random_ksat(300, 2600, 4, 2014), 24),            # the paper's MaxSAT-2016 sizes (:179)
        "maxsat_k3_odd_R": lambda: get("maxsat_k3_odd_R"),
        "maxsat_k2_n1500": lambda: (wl.random_ksat(1500, 4000, 2, 2015), 10),          # 2 variables per thread
    }


@pytest.mark.parametrize("mode", ["adam_exact", "rmsprop_manipulated", "sgd_exact"])
@pytest.mark.parametrize("name", list(_persist_cases()))
def test_persistent_kernel_bit_identical_to_stepwise(fem, name, mode):
    """Small sparse two-state problems run in the replica-persistent kernel (one CTA per replica, state in
    registers, gathers from shared memory).  Its arithmetic is the stepwise kernel's, so fields, moments and
    energies must be bit-identical, including across a resume (stop_after) and the fp64 wide phase."""
    inst, R = _persist_cases()[name]()
    steps = 300                                                      # three launches of the fp32 kernel (persist_chunk below)
    extra = {"adam_exact": {}, "rmsprop_manipulated": dict(optimizer=1, lr=0.03, alpha=0.9, momentum=0.5,
                                                            manipulated=True, gamma_grad=0.9),
             "sgd_exact": dict(optimizer=2, lr=0.3, momentum=0.7, dampening=0.2)}[mode]
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, steps), precise_steps=8, **extra)
    out = {}
    for persistent in (0, 1, 2, 3, 5, 9):                             # off, automatic, clusters of 1, 2, 4, 8 CTAs per replica
        eng = fem.Fem(inst, R)
        eng.set_option("persistent", persistent)
        eng.set_option("persist_chunk", 128)
        eng.anneal(sch, R, seed=4, stop_after=5)                      # stops inside the wide phase
        h5 = eng.get_fields()
        eng.anneal(sch, R, seed=4, stop_after=37)
        h37 = eng.get_fields()
        eng.anneal(sch, R, seed=4, stop_after=steps)
        out[persistent] = (h5, h37, eng.get_fields(), eng.get_moments(), eng.result())
        if persistent <= 1:
            assert (eng.info("persist_launches") > 0) == (persistent == 1)
        elif eng.info("persist_launches") > 0:                        # a forced size that does not fit falls back to stepwise
            assert eng.info("persist_cluster") == persistent - 1
        eng.close()
    b = out[0]
    for persistent, a in out.items():
        for k in range(3):
            assert np.array_equal(a[k], b[k]), (persistent, k)
        assert np.array_equal(a[3][0], b[3][0]) and np.array_equal(a[3][1], b[3][1])
        assert np.array_equal(a[4]["energy"], b[4]["energy"]) and a[4]["best_replica"] == b[4]["best_replica"]


@pytest.mark.parametrize("case", ["q8_reg10_R16", "q8_reg10_R32_two_blocks", "q4_reg6_weighted_R32", "q32_reg16_R4", "q2_reg3_R64",
                                  "q8_er_csr_R16", "q4_er_csr_weighted_R32"])
@pytest.mark.parametrize("manipulated", [False, True])
def test_potts_tma_bit_identical_to_team_kernel(fem, case, manipulated):
    """The TMA-staged Potts step (rows fetched one variable ahead into a shared-memory ring) against the register
    path: same arithmetic, so fields, moments, energies must be bit-identical; the counter proves which one ran."""
    q, d, R, rb, weighted = {"q8_er_csr_R16": (8, 0, 16, 0, False), "q4_er_csr_weighted_R32": (4, 0, 32, 0, True), "q8_reg10_R16": (8, 10, 16, 0, False), "q8_reg10_R32_two_blocks": (8, 10, 32, 16, False),
                             "q4_reg6_weighted_R32": (4, 6, 32, 0, True), "q32_reg16_R4": (32, 16, 4, 0, False),
                             "q2_reg3_R64": (2, 3, 64, 0, False)}[case]
    if case.startswith(("q8_er", "q4_er")):                       # CSR rows of different lengths (0 .. 16), isolated nodes
        q, R, rb, weighted = (8, 16, 0, False) if case.startswith("q8") else (4, 32, 0, True)
        er = wl.erdos_renyi_maxcut(1203, 0.0045, 2040 + q, pm1=False)
        assert 0 < np.diff(er.row_ptr).max() <= 16 and np.diff(er.row_ptr).min() == 0
        inst = wl.Instance(wl.BMINCUT, er.n, q, er.row_ptr, er.col_idx, None, lam=0.03)
    else:
        inst = wl.random_regular(1201 if d % 2 == 0 else 1200, d, 2020 + q, wl.BMINCUT, q, lam=0.03)
    if weighted:
        w = np.random.default_rng(3).integers(1, 5, inst.nnz // 2).astype(np.float32)[edge_ids(inst)]
        inst = wl.Instance(wl.BMINCUT, inst.n, q, inst.row_ptr, inst.col_idx, w, lam=0.03)
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.05, 40), precise_steps=4, manipulated=manipulated,
                       gamma_grad=0.9, **(dict(optimizer=1, lr=0.03, alpha=0.9, momentum=0.5) if manipulated else {}))
    applies = not manipulated or q <= 8              # manipulated: the id rows must be whole 16-byte bulk copies
    out = {}
    for tma in (1, 0):
        eng = fem.Fem(inst, R)
        eng.set_option("potts_si", 0)                # (and the state-innermost kernel the q = 4 / 8 ones)
        eng.set_option("potts_tma", tma)
        if rb:
            eng.set_option("replica_block", rb)
        eng.anneal(sch, R, seed=8, stop_after=17)
        eng.anneal(sch, R, seed=8, stop_after=40)
        out[tma] = (eng.get_fields(), eng.get_moments(), eng.result())
        assert eng.info("tma_launches") == (36 * (R // rb if rb else 1) if tma and applies else 0)   # 40 steps - 4 wide, per block
        eng.close()
    assert np.array_equal(out[1][0], out[0][0])
    assert np.array_equal(out[1][1][0], out[0][1][0]) and np.array_equal(out[1][1][1], out[0][1][1])
    assert np.array_equal(out[1][2]["energy"], out[0][2]["energy"])


@pytest.mark.parametrize("opt", ["adam", "sgd_mom"])
@pytest.mark.parametrize("name", ["maxcut_torus_30x34", "maxcut_reg3_pm1", "ising_reg3"])
def test_gather_fields_mode_is_bit_identical(fem, name, opt):
    """Gather-the-fields mode of the sparse two-state step (regular degree 3 / 4): neighbours gathered from the field
    array with tanh recomputed, fields ping-ponging between two arrays, no gather array written.  Same arithmetic, so
    fields, moments, marginals and energies are bit-identical to the default path -- across resume points, replica
    blocks and the parity hooks called in between (which use the spare array as scratch)."""
    if name == "ising_reg3":
        inst, R = wl.sparse_ising_from(wl.random_regular(1000, 3, 2050, pm1=True), scale=0.37), 24
    else:
        inst, R = get(name)
    if R % 4:
        R = 4 * (R // 4 + 1)
    extra = {"adam": {}, "sgd_mom": dict(optimizer=2, lr=0.3, momentum=0.7, dampening=0.2)}[opt]
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.05, 60), precise_steps=4, **extra)
    out = {}
    for mode, rb in ((0, 0), (1, 0), (1, 4)):
        eng = fem.Fem(inst, R)
        eng.set_option("persistent", 0)
        eng.set_option("gather_fields", mode)
        if rb:
            eng.set_option("replica_block", rb)
        eng.anneal(sch, R, seed=9, stop_after=3)                      # inside the wide phase
        eng.anneal(sch, R, seed=9, stop_after=17)
        p17, h17 = eng.get_marginals(), eng.get_fields()
        eng.anneal(sch, R, seed=9, stop_after=18)                     # an odd number of fp32 steps later
        p18 = eng.get_marginals()
        eng.anneal(sch, R, seed=9)
        assert eng.info("gather_fields") == mode
        out[(mode, rb)] = (h17, p17, p18, eng.get_fields(), eng.get_moments(), eng.result(), eng.get_configs())
        eng.close()
    b = out[(0, 0)]
    for key, a in out.items():
        for k in range(4):
            assert np.array_equal(a[k], b[k]), (key, k)
        assert np.array_equal(a[4][0], b[4][0]) and np.array_equal(a[4][1], b[4][1]), key
        assert np.array_equal(a[5]["energy"], b[5]["energy"]) and a[5]["best_replica"] == b[5]["best_replica"], key
        assert np.array_equal(a[6], b[6]), key


SI_CASES = {
    # name: (q, degree (0 = Erdos-Renyi CSR with rows of 0..16 entries), n, R, replica_block, weighted)
    "q8_reg10_R16_rb8": (8, 10, 1200, 16, 8, False),           # cfg 2's shape: 4 variables per 32-cell group
    "q8_reg10_R32_rb16": (8, 10, 1200, 32, 16, False),         # 2 variables per group, two blocks
    "q8_reg10_R8_rb4": (8, 10, 1200, 8, 4, False),             # 8 variables per group
    "q8_reg3_R16_auto": (8, 3, 1200, 16, 0, False),
    "q4_reg6_weighted_R32": (4, 6, 1201, 32, 32, True),        # one variable per group, odd n
    "q4_reg4_R16_rb8": (4, 4, 1204, 16, 8, False),
    "q8_reg7_weighted_R16_rb16": (8, 7, 1202, 16, 16, True),   # a regular degree without an unrolled instantiation
    "q8_er_csr_R16_rb8": (8, 0, 1204, 16, 8, False),           # rows of different lengths, isolated nodes
    "q4_er_csr_weighted_R32_rb16": (4, 0, 1204, 32, 16, True),
    "q8_reg10_R16_rb8_n1201": (8, 10, 1201, 16, 8, False),     # n not a multiple of 32 / Rb: the kernel does not apply
}


@pytest.mark.parametrize("opt", ["adam", "sgd_mom", "rmsprop"])
@pytest.mark.parametrize("case", list(SI_CASES))
def test_potts_si_bit_identical_to_team_kernel(fem, case, opt):
    """The Potts step on state-innermost replica blocks (k_step_potts_si.cu: arrays re-laid out in place for the fp32
    steps of a fem_anneal call, a lane owns the q states of one (variable, replica) cell) against the register path:
    same arithmetic in the same order, so fields, moments, energies and part sizes must be bit-identical -- also across
    a resume point (two relayouts in, two out); the counter proves which kernel ran."""
    q, d, n, R, rb, weighted = SI_CASES[case]
    if d == 0:
        er = wl.erdos_renyi_maxcut(n, 0.0045, 2040 + q, pm1=False)
        assert 0 < np.diff(er.row_ptr).max() and np.diff(er.row_ptr).min() == 0
        inst = wl.Instance(wl.BMINCUT, er.n, q, er.row_ptr, er.col_idx, None, lam=0.03)
    else:
        inst = wl.random_regular(n if (n * d) % 2 == 0 else n + 1, d, 2020 + q, wl.BMINCUT, q, lam=0.03)
    if weighted:
        w = np.random.default_rng(3).integers(1, 5, inst.nnz // 2).astype(np.float32)[edge_ids(inst)]
        inst = wl.Instance(wl.BMINCUT, inst.n, q, inst.row_ptr, inst.col_idx, w, lam=0.03)
    extra = {"adam": {}, "sgd_mom": dict(optimizer=2, lr=0.3, momentum=0.7, dampening=0.2),
             "rmsprop": dict(optimizer=1, lr=0.03, alpha=0.9)}[opt]
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.05, 40), precise_steps=4, **extra)
    out = {}
    for si in (1, 0):
        eng = fem.Fem(inst, R)
        eng.set_option("potts_si", si)
        eng.set_option("potts_tma", 0)
        if rb:
            eng.set_option("replica_block", rb)
        eng.anneal(sch, R, seed=8, stop_after=17)
        mid = eng.get_fields()                        # a hook between the two calls sees the standard layout
        eng.anneal(sch, R, seed=8, stop_after=40)
        out[si] = (eng.get_fields(), eng.get_moments(), eng.result(), mid, eng.get_marginals())
        Rb = eng.info("replica_block")
        blocks = R // Rb
        applies = Rb in (4, 8, 16, 32) and inst.n % (32 // Rb) == 0
        assert eng.info("si_launches") == (36 * blocks if si and applies else 0), case   # 40 steps - 4 wide, per block
        if rb:
            assert Rb == rb
        eng.close()
    assert np.array_equal(out[1][0], out[0][0])
    assert np.array_equal(out[1][3], out[0][3])
    assert np.array_equal(out[1][4], out[0][4])
    assert np.array_equal(out[1][1][0], out[0][1][0]) and np.array_equal(out[1][1][1], out[0][1][1])
    assert np.array_equal(out[1][2]["energy"], out[0][2]["energy"])
    assert np.array_equal(out[1][2]["part_sizes"], out[0][2]["part_sizes"])


def test_potts_l2_persistence_changes_no_bit_and_gives_the_set_aside_back(fem):
    """State-innermost Potts steps keep the gather buffers of a replica block in a persisting L2 set-aside (option
    "l2_persist", default 1; fem_api.cu l2_persist_begin / l2_persist_end): a cache policy, so every bit of the result is
    the same with it off; the device-wide limit is raised while the steps run and is back at its old value after
    fem_result (and after fem_destroy when no result was asked for)."""
    try:
        from cuda.bindings import runtime as cudart
    except Exception:                                     # pragma: no cover - cuda-python is in the image
        cudart = None

    def limit():
        if cudart is None:
            return None
        err, val = cudart.cudaDeviceGetLimit(cudart.cudaLimit.cudaLimitPersistingL2CacheSize)
        assert int(err) == 0
        return int(val)

    q, d, n, R, rb, _ = SI_CASES["q8_reg10_R16_rb8"]
    inst = wl.random_regular(n, d, 2020 + q, wl.BMINCUT, q, lam=0.03)
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.05, 40), precise_steps=4)
    import torch
    torch.cuda.synchronize()
    before = limit()
    out = {}
    for persist in (1, 0):
        eng = fem.Fem(inst, R)
        eng.set_option("replica_block", rb)
        eng.set_option("l2_persist", persist)
        eng.anneal(sch, R, seed=8)
        bytes_on = eng.info("l2_persist_bytes")
        assert (bytes_on >= 2 * (inst.n * q + 1) * rb * 4) if persist else bytes_on == 0
        if persist and before is not None:
            assert limit() == bytes_on
        fields = eng.get_fields()
        res = eng.result()
        assert eng.info("l2_persist_bytes") == 0 and limit() == before
        assert eng.info("si_launches") == 36 * (R // rb)
        out[persist] = (fields, res)
        eng.close()
    assert np.array_equal(out[1][0], out[0][0])
    assert np.array_equal(out[1][1]["energy"], out[0][1]["energy"])
    eng = fem.Fem(inst, R)                                # no fem_result: fem_destroy gives the set-aside back
    eng.set_option("replica_block", rb)
    eng.anneal(sch, R, seed=8)
    assert eng.info("l2_persist_bytes") > 0
    eng.close()
    assert limit() == before


def test_two_handles_with_rank_seeds_match_single_runs(fem):
    """The N > 1 path on one device: two handles, seeded as ranks 0 and 1 (multigpu.replica_seed), advanced in turns on
    the same stream, give bit for bit what each seed gives alone -- handles share nothing -- and the Eq.5 pick over the
    two is the better of the two bests, rank 0 on ties (tests/test_multirank_cpu.py covers the exchange itself)."""
    from paper_2412_09285_b200 import multigpu
    inst, R = get("maxcut_reg3_pm1")
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, 120), precise_steps=8)
    alone = []
    for r in range(2):
        eng = fem.Fem(inst, R)
        eng.anneal(sch, R, seed=multigpu.replica_seed(4, r))
        alone.append(eng.result())
        eng.close()
    engs = [fem.Fem(inst, R) for _ in range(2)]
    for stop in (30, 31, 90, 120):                       # interleaved on one stream
        for r, eng in enumerate(engs):
            eng.anneal(sch, R, seed=multigpu.replica_seed(4, r), stop_after=stop)
    both = [eng.result() for eng in engs]
    for r in range(2):
        assert np.array_equal(both[r]["energy_int"], alone[r]["energy_int"])
        assert np.array_equal(both[r]["best_config"], alone[r]["best_config"])
        engs[r].close()
    assert not np.array_equal(alone[0]["energy_int"], alone[1]["energy_int"])   # different replicas on the two "ranks"
    bests = [float(x["energy"][x["best_replica"]]) for x in both]
    e, owner, cfg = multigpu.best_over_ranks(bests[int(np.argmin(bests))], both[int(np.argmin(bests))]["best_config"],
                                             __import__("torch").device("cpu"))
    assert e == min(bests) and np.array_equal(cfg, both[int(np.argmin(bests))]["best_config"])


@pytest.mark.parametrize("shape", [(512, 256, 0), (640, 128, 64), (384, 256, 0)])
def test_dense_int8_cluster_multicast_matches_single_cta(fem, shape):
    """The int8 digit step in 2 x 2 clusters with operand multicast (tc_cluster = 1, taken when the grid has an even number
    of row and column tiles) against the same step without clusters: integer accumulation is exact, so the two agree bit
    for bit; and against the oracle on a replica subset.  (384, 256): three row tiles -> no clusters either way."""
    n, R, tile = shape
    inst = wl.sk_dense(n, 2012)
    beta = fem.linear_temperature_schedule(1.0, 0.01, 500)
    h0 = fo.init_fields(6, R, inst.n, 1).astype(np.float32)
    pb, st = oracle_run(inst, h0[:16], beta, 30, inst.lam)
    P_ref = fo.marginals(pb, st.h).reshape(16, inst.n)
    out = []
    for cl in (1, 0):
        eng = fem.Fem(inst, R)
        eng.set_option("tc_cluster", cl)
        if tile:
            eng.set_option("tc_tile_n", tile)
        eng.set_fields(h0)
        eng.anneal(fem.Schedule(beta=beta, precise_steps=8), R, stop_after=30)
        out.append((eng.get_fields(), eng.get_marginals().astype(np.float64)))
        assert eng.info("tc8_launches") == 22
        eng.close()
    assert np.array_equal(out[0][0], out[1][0])
    assert np.max(np.abs(out[0][1][:16] - P_ref)) < MARGINAL_TOL
