"""Host-side checks that need no GPU: the C-ABI library loads, exports every symbol include/fem.h declares,
reports argument errors before touching a device, and fails loudly (no CPU fallback) without one."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2412_09285_b200 import build as fembuild
from paper_2412_09285_b200 import fem, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    fembuild.build()                      # nvcc cross-compiles for sm_100a without a GPU
    return fem.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "fem.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fem_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(fem.EXPORTS) == names
    assert lib.fem_abi_version() == 4


def cproblem(inst, keep):
    def p(a, dt):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=dt)
        keep.append(a)
        return a.ctypes.data_as(C.c_void_p)
    return fem.CProblem(inst.kind, inst.n, inst.q, p(inst.row_ptr, np.int64), p(inst.col_idx, np.int32),
                        p(inst.weight, np.float32), p(inst.dense_J, np.float32), inst.m, p(inst.clause_ptr, np.int64),
                        p(inst.lits, np.int32), float(inst.lam))


def create(lib, inst, R=4, ws=256 << 10):
    keep = []
    cp = cproblem(inst, keep)
    h = C.c_void_p()
    fake_ws = C.c_void_p(1 << 20)         # never dereferenced when validation fails first
    st = lib.fem_create(C.byref(cp), R, fake_ws, C.c_size_t(1 << 40), None, C.byref(h))
    return st, (lib.fem_last_error(None) or b"").decode()


def test_workspace_bytes_is_pure_host_arithmetic(lib):
    keep = []
    inst = wl.torus_maxcut(8, 1)
    a = lib.fem_workspace_bytes(C.byref(cproblem(inst, keep)), 16)
    b = lib.fem_workspace_bytes(C.byref(cproblem(inst, keep)), 32)
    assert 0 < a < b and a % 256 == 0
    assert lib.fem_workspace_bytes(C.byref(cproblem(inst, keep)), 0) == 0
    bad = wl.torus_maxcut(8, 1)
    bad.q = 3
    assert lib.fem_workspace_bytes(C.byref(cproblem(bad, keep)), 16) == 0


def test_argument_errors_come_before_the_device(lib):
    g = wl.erdos_renyi_maxcut(30, 0.3, 5, pm1=True)
    cases = {}
    a = wl.erdos_renyi_maxcut(30, 0.3, 5, pm1=True)
    a.col_idx = a.col_idx.copy()
    a.col_idx[0] = (a.col_idx[0] + 1) % 30 if (a.col_idx[0] + 1) % 30 not in a.col_idx[:a.row_ptr[1]] else a.col_idx[0]
    w = g.weight.copy()
    w[0] = -w[0]
    cases["weights are not symmetric"] = wl.Instance(wl.MAXCUT, 30, 2, g.row_ptr, g.col_idx, w)
    loop = g.col_idx.copy()
    loop[g.row_ptr[3]] = 3
    cases["self loop"] = wl.Instance(wl.MAXCUT, 30, 2, g.row_ptr, loop, g.weight)
    unsorted = g.col_idx.copy()
    r0, r1 = g.row_ptr[5], g.row_ptr[6]
    if r1 - r0 >= 2:
        unsorted[r0], unsorted[r0 + 1] = unsorted[r0 + 1], unsorted[r0]
        cases["columns must be strictly ascending"] = wl.Instance(wl.MAXCUT, 30, 2, g.row_ptr, unsorted, g.weight)
    asym_ptr = g.row_ptr.copy()
    asym_col = np.delete(g.col_idx, g.row_ptr[1] - 1)       # drop one direction of an edge of row 0
    asym_ptr[1:] -= 1
    cases["CSR is not symmetric"] = wl.Instance(wl.MAXCUT, 30, 2, asym_ptr, asym_col, np.delete(g.weight, g.row_ptr[1] - 1))
    cases["BMINCUT weights must be > 0"] = wl.Instance(wl.BMINCUT, 30, 4, g.row_ptr, g.col_idx, g.weight)
    cases["q must be in 2..32"] = wl.Instance(wl.BMINCUT, 30, 40, g.row_ptr, g.col_idx, None)
    sat = wl.random_ksat(20, 50, 3, 6)
    rep = sat.lits.copy()
    rep[1] = -rep[0]
    cases["a clause repeats a variable"] = wl.Instance(wl.MAXSAT, 20, 2, m=50, clause_ptr=sat.clause_ptr, lits=rep)
    oor = sat.lits.copy()
    oor[2] = 21
    cases["literal out of range"] = wl.Instance(wl.MAXSAT, 20, 2, m=50, clause_ptr=sat.clause_ptr, lits=oor)
    sk = wl.sk_dense(16, 7)
    J = sk.dense_J.copy()
    J[2, 3] += 1.0
    cases["dense_J must be symmetric"] = wl.Instance(wl.ISING, 16, 2, dense_J=J)
    for msg, inst in cases.items():
        st, err = create(lib, inst)
        assert st == fem.FEM_EINVAL and msg in err, (msg, st, err)
    # a misaligned or too-small workspace is an argument error too
    keep = []
    cp = cproblem(g, keep)
    h = C.c_void_p()
    assert lib.fem_create(C.byref(cp), 4, C.c_void_p((1 << 20) + 8), C.c_size_t(1 << 40), None, C.byref(h)) == fem.FEM_EINVAL
    assert lib.fem_create(C.byref(cp), 4, C.c_void_p(1 << 20), C.c_size_t(1024), None, C.byref(h)) == fem.FEM_EINVAL


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the loud-failure path is for boxes without one")
    with pytest.raises(fem.FemError) as e:
        fem.Fem(wl.torus_maxcut(8, 1), 4)
    assert e.value.status == fem.FEM_ECUDA


def test_schedule_helpers_match_the_paper_endpoints():
    b = fem.linear_temperature_schedule(1.0, 0.01, 500)
    assert b[0] == 1.0 and abs(b[-1] - 100.0) < 1e-9 and np.all(np.diff(b) > 0)
    e = fem.exponential_schedule(0.02, 750.0, 100)
    assert abs(e[0] - 0.02) < 1e-15 and abs(e[-1] - 750.0) < 1e-9


def test_schedules_behind_the_abi_equal_the_oracles(lib):
    """a5 lives behind the C ABI (fem_schedule_*): same arithmetic order as the paper's formulas, so
    the arrays are bit-identical to the oracle's; N = 1 gives beta(0); bad arguments are rejected."""
    from oracle import fem_oracle as fo
    for N in (1, 2, 7, 500, 2000):
        assert np.array_equal(fem.linear_temperature_schedule(1.0, 0.01, N), fo.schedule_inverse_proportional(1.0, 0.01, N))
        assert np.array_equal(fem.linear_temperature_schedule(2.5, 0.3, N), fo.schedule_inverse_proportional(2.5, 0.3, N))
        a, b = fem.exponential_schedule(0.02, 750.0, N), fo.schedule_exponential(0.02, 750.0, N)
        ulp = np.abs(a.view(np.int64) - b.view(np.int64))
        assert ulp.max() <= 1, ulp.max()                  # exp / log come from two different libm builds at most 1 ulp apart
    out = np.empty(4)
    ptr = out.ctypes.data_as(C.c_void_p)
    assert lib.fem_schedule_inverse_proportional(1.0, 0.01, 0, ptr) == fem.FEM_EINVAL
    assert lib.fem_schedule_inverse_proportional(1.0, -0.01, 4, ptr) == fem.FEM_EINVAL
    assert lib.fem_schedule_inverse_proportional(1.0, 0.01, 4, None) == fem.FEM_EINVAL
    assert lib.fem_schedule_exponential(0.0, 5.0, 4, ptr) == fem.FEM_EINVAL
    assert lib.fem_schedule_exponential(0.1, float("inf"), 4, ptr) == fem.FEM_EINVAL
    with pytest.raises(fem.FemError):
        fem.exponential_schedule(-1.0, 5.0, 10)


def test_schedule_struct_carries_its_size():
    sch = fem.Schedule(beta=np.ones(3)).c()
    assert sch.struct_bytes == C.sizeof(fem.CSchedule) and sch.steps == 3
