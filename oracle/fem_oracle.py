"""ctypes front-end of oracle/fem_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It marshals numpy arrays (logical layouts, float64) into the plain
C oracle and holds no arithmetic of the method itself.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fem_oracle.c")

MAXCUT, ISING, BMINCUT, MAXSAT = 0, 1, 2, 3


def build(openmp: bool = False, force: bool = False) -> str:
    """Compile fem_oracle.c with gcc (no FMA contraction so sums keep their written order)."""
    out = os.path.join(_HERE, "libfem_oracle_omp.so" if openmp else "libfem_oracle.so")
    if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
        return out
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c11"]
    if openmp:
        cmd.append("-fopenmp")
    tmp = out + f".tmp{os.getpid()}"
    cmd += [_SRC, "-o", tmp, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


class _Problem(C.Structure):
    _fields_ = [
        ("kind", C.c_int32), ("n", C.c_int32), ("q", C.c_int32),
        ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("weight", C.c_void_p),
        ("dense_J", C.c_void_p),
        ("m", C.c_int32), ("clause_ptr", C.c_void_p), ("lits", C.c_void_p),
        ("node_weight", C.c_void_p), ("lit_state", C.c_void_p),
    ]


class _Adam(C.Structure):
    _fields_ = [("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double),
                ("eps", C.c_double), ("weight_decay", C.c_double)]


class _Opt(C.Structure):
    _fields_ = [("kind", C.c_int32), ("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double),
                ("eps", C.c_double), ("weight_decay", C.c_double), ("alpha", C.c_double), ("momentum", C.c_double),
                ("dampening", C.c_double)]


ADAM, RMSPROP, SGD = 0, 1, 2

_libs: dict = {}


def _lib(openmp: bool = False):
    if openmp not in _libs:
        lib = C.CDLL(build(openmp))
        lib.femo_free_energy.restype = C.c_double
        lib.femo_internal_energy.restype = C.c_double
        lib.femo_entropy.restype = C.c_double
        lib.femo_argmin.restype = C.c_int32
        lib.femo_num_threads.restype = C.c_int32
        _libs[openmp] = lib
    return _libs[openmp]


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


@dataclass
class Problem:
    """Host-side problem description (numpy arrays; see fem_oracle.c femo_problem)."""
    kind: int
    n: int
    q: int = 2
    row_ptr: Optional[np.ndarray] = None   # int64 [n+1]
    col_idx: Optional[np.ndarray] = None   # int32 [nnz]
    weight: Optional[np.ndarray] = None    # float64 [nnz] or None (= all +1)
    dense_J: Optional[np.ndarray] = None   # float64 [n,n]
    m: int = 0
    clause_ptr: Optional[np.ndarray] = None  # int64 [m+1]
    lits: Optional[np.ndarray] = None        # int32, signed 1-based
    node_weight: Optional[np.ndarray] = None  # float64 [n], BMINCUT balance weights V_i (S33-S35) or None (= all 1)
    lit_state: Optional[np.ndarray] = None    # int32 [len(lits)], non-Boolean SAT: W_mi in 0..q-1 or None
    _keep: list = field(default_factory=list, repr=False)

    def __post_init__(self):
        def cast(a, dt):
            return None if a is None else np.ascontiguousarray(a, dtype=dt)
        self.row_ptr = cast(self.row_ptr, np.int64)
        self.col_idx = cast(self.col_idx, np.int32)
        self.weight = cast(self.weight, np.float64)
        self.dense_J = cast(self.dense_J, np.float64)
        self.clause_ptr = cast(self.clause_ptr, np.int64)
        self.lits = cast(self.lits, np.int32)
        self.node_weight = cast(self.node_weight, np.float64)
        self.lit_state = cast(self.lit_state, np.int32)

    @property
    def fields_per_var(self) -> int:
        return self.q if (self.kind == BMINCUT or (self.kind == MAXSAT and self.lit_state is not None)) else 1

    def c(self) -> _Problem:
        return _Problem(self.kind, self.n, self.q, _p(self.row_ptr), _p(self.col_idx), _p(self.weight),
                        _p(self.dense_J), self.m, _p(self.clause_ptr), _p(self.lits), _p(self.node_weight),
                        _p(self.lit_state))


@dataclass
class Adam:
    lr: float = 0.1
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8
    weight_decay: float = 0.0

    def c(self) -> _Adam:
        return _Adam(self.lr, self.beta1, self.beta2, self.eps, self.weight_decay)


@dataclass
class Optimizer:
    """Optimiser choice of SURVEY.md section 8(f) item 2 (PyTorch defaults for what the paper does not tune)."""
    kind: int = ADAM
    lr: float = 0.1
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8
    weight_decay: float = 0.0
    alpha: float = 0.99
    momentum: float = 0.0
    dampening: float = 0.0

    def c(self) -> _Opt:
        return _Opt(self.kind, self.lr, self.beta1, self.beta2, self.eps, self.weight_decay, self.alpha,
                    self.momentum, self.dampening)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def marginals(pb: Problem, h: np.ndarray) -> np.ndarray:
    """h[..., n, F] -> P of the same shape (two-state kinds: P(state 1))."""
    h = _f64(h)
    out = np.empty_like(h)
    per = pb.n * pb.fields_per_var
    hv, ov = h.reshape(-1, per), out.reshape(-1, per)
    cp = pb.c()
    for a in range(hv.shape[0]):
        _lib().femo_marginals(C.byref(cp), _p(hv[a]), _p(ov[a]))
    return out


def free_energy(pb: Problem, h: np.ndarray, beta: float, lam: float = 0.0) -> float:
    h = _f64(h)
    cp = pb.c()
    return float(_lib().femo_free_energy(C.byref(cp), _p(h), C.c_double(beta), C.c_double(lam)))


def internal_energy(pb: Problem, h: np.ndarray, lam: float = 0.0) -> float:
    h = _f64(h)
    cp = pb.c()
    return float(_lib().femo_internal_energy(C.byref(cp), _p(h), C.c_double(lam)))


def entropy(pb: Problem, h: np.ndarray) -> float:
    h = _f64(h)
    cp = pb.c()
    return float(_lib().femo_entropy(C.byref(cp), _p(h)))


def grad_h(pb: Problem, h: np.ndarray, beta: float, lam: float = 0.0) -> np.ndarray:
    """One replica: h[n*F] -> g^h[n*F]."""
    h = _f64(h)
    g = np.empty_like(h)
    cp = pb.c()
    _lib().femo_grad_h(C.byref(cp), _p(h), C.c_double(beta), C.c_double(lam), _p(g))
    return g


def grad_h_manipulated(pb: Problem, h: np.ndarray, beta: float, lam: float = 0.0, gamma: float = 1.0) -> np.ndarray:
    """One replica: manipulated gradient (S25/S27/S29/S30 with S20), h[n*F] -> g^h[n*F]."""
    h = _f64(h)
    g = np.empty_like(h)
    cp = pb.c()
    _lib().femo_grad_h_manipulated(C.byref(cp), _p(h), C.c_double(beta), C.c_double(lam), C.c_double(gamma), _p(g))
    return g


def rmsprop_update(opt: Optimizer, h: np.ndarray, m1: np.ndarray, m2: np.ndarray, g: np.ndarray) -> None:
    co = opt.c()
    _lib().femo_rmsprop(C.byref(co), C.c_int64(h.size), _p(h), _p(m1), _p(m2), _p(_f64(g)))


def sgd_update(opt: Optimizer, t: int, h: np.ndarray, m1: np.ndarray, g: np.ndarray) -> None:
    """t is the 1-based step count (the momentum buffer is initialised with the first gradient)."""
    co = opt.c()
    _lib().femo_sgd(C.byref(co), C.c_int32(t), C.c_int64(h.size), _p(h), _p(m1), _p(_f64(g)))


def adam_update(adam: Adam, t: int, h: np.ndarray, m1: np.ndarray, m2: np.ndarray, g: np.ndarray) -> None:
    """In place on float64 contiguous arrays; t is the 1-based step count."""
    ca = adam.c()
    _lib().femo_adam(C.byref(ca), C.c_int32(t), C.c_int64(h.size), _p(h), _p(m1), _p(m2), _p(_f64(g)))


def schedule_inverse_proportional(T_max: float, T_min: float, N: int) -> np.ndarray:
    beta = np.empty(N, dtype=np.float64)
    _lib().femo_schedule_inverse_proportional(C.c_double(T_max), C.c_double(T_min), C.c_int32(N), _p(beta))
    return beta


def schedule_exponential(beta_min: float, beta_max: float, N: int) -> np.ndarray:
    beta = np.empty(N, dtype=np.float64)
    _lib().femo_schedule_exponential(C.c_double(beta_min), C.c_double(beta_max), C.c_int32(N), _p(beta))
    return beta


def init_fields(seed: int, R: int, n: int, F: int, scale: float = 1e-3) -> np.ndarray:
    h = np.empty((R, n, F) if F > 1 else (R, n), dtype=np.float64)
    _lib().femo_init_fields(C.c_uint64(seed), C.c_int32(R), C.c_int32(n), C.c_int32(F), C.c_double(scale), _p(h))
    return h


class State:
    """Fields and Adam moments of R replicas, float64, logical layout [R][n][F]."""

    def __init__(self, pb: Problem, h0: np.ndarray):
        self.pb = pb
        self.h = _f64(h0).copy()
        self.R = self.h.size // (pb.n * pb.fields_per_var)
        self.m1 = np.zeros_like(self.h)
        self.m2 = np.zeros_like(self.h)
        self.t = 0


def anneal(st: State, beta: np.ndarray, adam: Adam, lam: float = 0.0, lam_t: Optional[np.ndarray] = None,
           t_end: Optional[int] = None, openmp: bool = False) -> State:
    """Run steps st.t .. t_end-1 of the schedule beta[0..N-1] in place."""
    beta = _f64(beta)
    t_end = len(beta) if t_end is None else t_end
    lam_t = None if lam_t is None else _f64(lam_t)
    cp, ca = st.pb.c(), adam.c()
    _lib(openmp).femo_anneal(C.byref(cp), C.c_int32(st.R), _p(st.h), _p(st.m1), _p(st.m2), _p(beta), _p(lam_t),
                             C.c_double(lam), C.c_int32(st.t), C.c_int32(t_end), C.byref(ca))
    st.t = t_end
    return st


def anneal_ex(st: State, beta: np.ndarray, opt: Optimizer, lam: float = 0.0, lam_t: Optional[np.ndarray] = None,
              t_end: Optional[int] = None, manipulated: bool = False, gamma: float = 1.0, openmp: bool = False) -> State:
    """anneal() with the optimiser / gradient choices of SURVEY.md section 8(f)."""
    beta = _f64(beta)
    t_end = len(beta) if t_end is None else t_end
    lam_t = None if lam_t is None else _f64(lam_t)
    cp, co = st.pb.c(), opt.c()
    _lib(openmp).femo_anneal_ex(C.byref(cp), C.c_int32(st.R), _p(st.h), _p(st.m1), _p(st.m2), _p(beta), _p(lam_t),
                                C.c_double(lam), C.c_int32(st.t), C.c_int32(t_end), C.byref(co),
                                C.c_int32(1 if manipulated else 0), C.c_double(gamma))
    st.t = t_end
    return st


def round_configs(pb: Problem, h: np.ndarray) -> np.ndarray:
    h = _f64(h)
    R = h.size // (pb.n * pb.fields_per_var)
    cfg = np.empty((R, pb.n), dtype=np.int32)
    cp = pb.c()
    _lib().femo_round(C.byref(cp), C.c_int32(R), _p(h), _p(cfg))
    return cfg


def energies(pb: Problem, cfg: np.ndarray, lam: float = 0.0):
    """cfg[R][n] int32 -> (e_int[R] int64, e_real[R] float64, part[R][q] int32)."""
    cfg = np.ascontiguousarray(cfg, dtype=np.int32).reshape(-1, pb.n)
    R = cfg.shape[0]
    e_int = np.empty(R, dtype=np.int64)
    e_real = np.empty(R, dtype=np.float64)
    part = np.zeros((R, pb.q), dtype=np.int32)
    cp = pb.c()
    _lib().femo_energies(C.byref(cp), C.c_int32(R), _p(cfg), C.c_double(lam), _p(e_int), _p(e_real), _p(part))
    return e_int, e_real, part


def argmin(e_real: np.ndarray) -> int:
    e_real = _f64(e_real)
    return int(_lib().femo_argmin(C.c_int32(e_real.size), _p(e_real)))


def num_threads(openmp: bool) -> int:
    return int(_lib(openmp).femo_num_threads())
