"""Python binding of include/fem.h: argument marshalling only.

Every step of the path (init, fused annealing steps, rounding, energies, argmin) runs in the CUDA
kernels of csrc/libfem_b200.so.  PyTorch provides the device workspace and the stream, nothing else.
If the library is missing or there is no CUDA device this module raises; there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import workloads as wl

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libfem_b200.so")

FEM_OK, FEM_EINVAL, FEM_ENOMEM, FEM_ECUDA, FEM_ESTATE = range(5)
STATUS_NAMES = {0: "FEM_OK", 1: "FEM_EINVAL", 2: "FEM_ENOMEM", 3: "FEM_ECUDA", 4: "FEM_ESTATE"}

EXPORTS = [
    "fem_abi_version", "fem_workspace_bytes", "fem_create", "fem_anneal", "fem_reset", "fem_readout", "fem_result",
    "fem_set_fields", "fem_get_fields", "fem_get_moments", "fem_get_marginals", "fem_get_configs", "fem_energy_of",
    "fem_set_option", "fem_get_info", "fem_last_error", "fem_destroy",
    "fem_schedule_inverse_proportional", "fem_schedule_exponential", "fem_probe_l2_read", "fem_probe_l2_gather",
    "fem_cut_static", "fem_cut_static_error",
]
CUT_STATIC_MAX_COUNT = 4096   # FEM_CUT_STATIC_MAX_COUNT of include/fem.h


class FemError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class CProblem(C.Structure):
    _fields_ = [
        ("kind", C.c_int32), ("n", C.c_int32), ("q", C.c_int32),
        ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("weight", C.c_void_p), ("dense_J", C.c_void_p),
        ("m", C.c_int32), ("clause_ptr", C.c_void_p), ("lits", C.c_void_p), ("lambda_", C.c_double),
        ("node_weight", C.c_void_p),   # ABI 4: BMINCUT node weights V_i (float32 [n]) or NULL
        ("lit_state", C.c_void_p),     # ABI 4: non-Boolean MAXSAT clause values W_mi (int32 [nlits]) or NULL
    ]


class CSchedule(C.Structure):
    _fields_ = [
        ("struct_bytes", C.c_uint32), ("steps", C.c_int32), ("beta", C.c_void_p), ("lambda_", C.c_void_p),
        ("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double), ("eps", C.c_double),
        ("weight_decay", C.c_double), ("init_scale", C.c_double), ("precise_steps", C.c_int32),
        ("optimizer", C.c_int32), ("alpha", C.c_double), ("momentum", C.c_double), ("dampening", C.c_double),
        ("manipulated", C.c_int32), ("gamma_grad", C.c_double),
    ]


ADAM, RMSPROP, SGD = 0, 1, 2   # fem_optimizer


_lib = None


def load_library():
    """dlopen csrc/libfem_b200.so (built by paper_2412_09285_b200.build); loud failure if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2412_09285_b200.build` "
                          "(there is no CPU fallback for the FEM path)")
    lib = C.CDLL(LIB_PATH)
    lib.fem_abi_version.restype = C.c_int32
    lib.fem_workspace_bytes.restype = C.c_size_t
    lib.fem_workspace_bytes.argtypes = [C.POINTER(CProblem), C.c_int32]
    lib.fem_create.argtypes = [C.POINTER(CProblem), C.c_int32, C.c_void_p, C.c_size_t, C.c_void_p,
                               C.POINTER(C.c_void_p)]
    lib.fem_anneal.argtypes = [C.c_void_p, C.POINTER(CSchedule), C.c_int32, C.c_uint64, C.c_int32]
    lib.fem_reset.argtypes = [C.c_void_p]
    lib.fem_readout.argtypes = [C.c_void_p]
    lib.fem_result.argtypes = [C.c_void_p] + [C.c_void_p] * 5
    lib.fem_set_fields.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    lib.fem_get_fields.argtypes = [C.c_void_p, C.c_void_p]
    lib.fem_get_moments.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.fem_get_marginals.argtypes = [C.c_void_p, C.c_void_p]
    lib.fem_get_configs.argtypes = [C.c_void_p, C.c_void_p]
    lib.fem_energy_of.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.fem_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
    lib.fem_get_info.restype = C.c_int64
    lib.fem_get_info.argtypes = [C.c_void_p, C.c_char_p]
    lib.fem_last_error.restype = C.c_char_p
    lib.fem_last_error.argtypes = [C.c_void_p]
    lib.fem_destroy.argtypes = [C.c_void_p]
    lib.fem_schedule_inverse_proportional.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_void_p]
    lib.fem_schedule_exponential.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_void_p]
    lib.fem_probe_l2_read.argtypes = [C.c_void_p, C.c_size_t, C.c_int32, C.c_void_p, C.POINTER(C.c_double)]
    lib.fem_probe_l2_gather.argtypes = [C.c_void_p, C.c_size_t, C.c_int32, C.c_int32, C.c_void_p, C.POINTER(C.c_double)]
    lib.fem_cut_static.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.fem_cut_static_error.restype = C.c_char_p
    _lib = lib
    return lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


@dataclass
class Schedule:
    """Host-side schedule: beta[t] (and optional lambda[t]), the optimiser and the gradient mode."""
    beta: np.ndarray
    lr: float = 0.1
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8
    weight_decay: float = 0.0
    init_scale: float = 1e-3
    precise_steps: int = 8
    lam: Optional[np.ndarray] = None
    optimizer: int = ADAM          # ADAM / RMSPROP / SGD, PyTorch semantics
    alpha: float = 0.99            # RMSprop smoothing constant
    momentum: float = 0.0          # RMSprop / SGD
    dampening: float = 0.0         # SGD
    manipulated: bool = False      # manipulated gradients S25/S27/S30
    gamma_grad: float = 1.0        # S20

    def c(self) -> CSchedule:
        self.beta = np.ascontiguousarray(self.beta, dtype=np.float64)
        if self.lam is not None:
            self.lam = np.ascontiguousarray(self.lam, dtype=np.float64)
        return CSchedule(C.sizeof(CSchedule), int(self.beta.size), _ptr(self.beta), _ptr(self.lam), self.lr, self.beta1, self.beta2, self.eps,
                         self.weight_decay, self.init_scale, self.precise_steps, int(self.optimizer), self.alpha,
                         self.momentum, self.dampening, 1 if self.manipulated else 0, self.gamma_grad)


def _schedule(fn_name: str, a: float, b: float, steps: int) -> np.ndarray:
    out = np.empty(int(steps), dtype=np.float64)
    st = getattr(load_library(), fn_name)(float(a), float(b), int(steps), _ptr(out))
    if st != FEM_OK:
        raise FemError(st, f"{fn_name}({a}, {b}, {steps})")
    return out


def linear_temperature_schedule(T_max: float, T_min: float, steps: int) -> np.ndarray:
    """fem_schedule_inverse_proportional: T linear from T_max to T_min; returns beta[t] = 1/T(t)."""
    return _schedule("fem_schedule_inverse_proportional", T_max, T_min, steps)


def exponential_schedule(beta_min: float, beta_max: float, steps: int) -> np.ndarray:
    """fem_schedule_exponential."""
    return _schedule("fem_schedule_exponential", beta_min, beta_max, steps)


class Fem:
    """One problem instance resident on a CUDA device (fem_create .. fem_destroy)."""

    def __init__(self, inst: wl.Instance, R_cap: int, device: str = "cuda:0", stream=None):
        import torch  # device memory and streams only

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise FemError(FEM_ECUDA, "no CUDA device: the FEM path has no CPU fallback")
        self.inst = inst
        self.R_cap = int(R_cap)
        self.device = torch.device(device)
        self._keep = []

        def host(a, dt):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=dt)
            self._keep.append(a)
            return a

        self._cp = CProblem(inst.kind, inst.n, inst.q, _ptr(host(inst.row_ptr, np.int64)),
                            _ptr(host(inst.col_idx, np.int32)), _ptr(host(inst.weight, np.float32)),
                            _ptr(host(inst.dense_J, np.float32)), inst.m, _ptr(host(inst.clause_ptr, np.int64)),
                            _ptr(host(inst.lits, np.int32)), float(inst.lam),
                            _ptr(host(getattr(inst, "node_weight", None), np.float32)),
                            _ptr(host(getattr(inst, "lit_state", None), np.int32)))
        nbytes = self._lib.fem_workspace_bytes(C.byref(self._cp), self.R_cap)
        if nbytes == 0:
            raise FemError(FEM_EINVAL, "fem_workspace_bytes rejected the problem")
        self.workspace_bytes = int(nbytes)
        with torch.cuda.device(self.device):
            # (guard bytes on both sides of the workspace, filled with a pattern: tests check that the library never writes
            # outside the bytes it asked for)
            self._guard = 1 << 16
            self._ws = torch.empty(nbytes + 256 + 2 * self._guard, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr() + self._guard
            self._ws_ptr = (base + 255) & ~255
            lo = self._ws_ptr - self._ws.data_ptr()
            self._ws[:lo].fill_(0xA5)               # only the guards are filled, not the workspace
            self._ws[lo + nbytes:].fill_(0xA5)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            st = self._lib.fem_create(C.byref(self._cp), self.R_cap, C.c_void_p(self._ws_ptr), C.c_size_t(nbytes),
                                      C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if st != FEM_OK:
            raise FemError(st, (self._lib.fem_last_error(None) or b"").decode())
        self._h = h
        self.R = 0

    def guards_intact(self) -> bool:
        """True when no byte outside the workspace handed to fem_create has been written (64 KiB checked on each side)."""
        lo = self._ws_ptr - self._ws.data_ptr()
        hi = lo + self.workspace_bytes
        return bool((self._ws[:lo] == 0xA5).all().item()) and bool((self._ws[hi:] == 0xA5).all().item())

    # -- plumbing
    def _check(self, st: int):
        if st != FEM_OK:
            raise FemError(st, (self._lib.fem_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.fem_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def F(self) -> int:
        return self.inst.fields_per_var

    def _shape(self, R: int):
        return (R, self.inst.n, self.F) if self.F > 1 else (R, self.inst.n)

    # -- the three calls of the path
    def anneal(self, schedule: Schedule, R: int, seed: int = 0, stop_after: Optional[int] = None) -> None:
        cs = schedule.c()
        stop = cs.steps if stop_after is None else int(stop_after)
        self._check(self._lib.fem_anneal(self._h, C.byref(cs), int(R), C.c_uint64(seed), stop))
        self.R = int(R)

    def readout(self) -> None:
        self._check(self._lib.fem_readout(self._h))

    def result(self):
        """-> dict(best_replica, best_config[n], energy_int[R], energy[R], part_sizes[R,q])"""
        R, n, q = self.R, self.inst.n, self.inst.q
        best = np.zeros(1, dtype=np.int32)
        cfg = np.empty(n, dtype=np.int32)
        e_int = np.empty(R, dtype=np.int64)
        e = np.empty(R, dtype=np.float64)
        part = np.empty((R, q), dtype=np.int32)
        self._check(self._lib.fem_result(self._h, _ptr(best), _ptr(cfg), _ptr(e_int), _ptr(e), _ptr(part)))
        return {"best_replica": int(best[0]), "best_config": cfg, "energy_int": e_int, "energy": e, "part_sizes": part}

    def reset(self) -> None:
        self._check(self._lib.fem_reset(self._h))

    # -- parity hooks
    def set_fields(self, h0: np.ndarray) -> None:
        h0 = np.ascontiguousarray(h0, dtype=np.float32)
        R = h0.size // (self.inst.n * self.F)
        self._check(self._lib.fem_set_fields(self._h, R, _ptr(h0)))
        self.R = R

    def get_fields(self) -> np.ndarray:
        out = np.empty(self._shape(self.R), dtype=np.float32)
        self._check(self._lib.fem_get_fields(self._h, _ptr(out)))
        return out

    def get_moments(self):
        m1 = np.empty(self._shape(self.R), dtype=np.float32)
        m2 = np.empty(self._shape(self.R), dtype=np.float32)
        self._check(self._lib.fem_get_moments(self._h, _ptr(m1), _ptr(m2)))
        return m1, m2

    def get_marginals(self) -> np.ndarray:
        out = np.empty(self._shape(self.R), dtype=np.float32)
        self._check(self._lib.fem_get_marginals(self._h, _ptr(out)))
        return out

    def get_configs(self) -> np.ndarray:
        out = np.empty((self.R, self.inst.n), dtype=np.int32)
        self._check(self._lib.fem_get_configs(self._h, _ptr(out)))
        return out

    def energy_of(self, cfg: np.ndarray):
        cfg = np.ascontiguousarray(cfg, dtype=np.int32).reshape(-1, self.inst.n)
        count = cfg.shape[0]
        e_int = np.empty(count, dtype=np.int64)
        e = np.empty(count, dtype=np.float64)
        part = np.empty((count, self.inst.q), dtype=np.int32)
        self._check(self._lib.fem_energy_of(self._h, _ptr(cfg), count, _ptr(e_int), _ptr(e), _ptr(part)))
        return e_int, e, part

    def set_option(self, key: str, value: int) -> None:
        self._check(self._lib.fem_set_option(self._h, key.encode(), int(value)))

    def info(self, key: str) -> int:
        return int(self._lib.fem_get_info(self._h, key.encode()))


def probe_l2_read(device: str = "cuda:0", mib: int = 32, repeats: int = 200) -> float:
    """fem_probe_l2_read on a torch-owned buffer: the L2 -> SM read rate in GB/s (measurement helper)."""
    import torch
    lib = load_library()
    with torch.cuda.device(torch.device(device)):
        buf = torch.empty(mib << 20, dtype=torch.uint8, device=device)
        out = C.c_double(0.0)
        st = lib.fem_probe_l2_read(C.c_void_p(buf.data_ptr()), C.c_size_t(buf.numel()), repeats,
                                   C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out))
    if st != FEM_OK:
        raise FemError(st, "fem_probe_l2_read")
    return float(out.value)


def probe_l2_gather(device: str = "cuda:0", mib: int = 32, row_bytes: int = 128, repeats: int = 300) -> float:
    """fem_probe_l2_gather on a torch-owned buffer: the rate in GB/s of random-row gathers out of a `mib` MiB working set."""
    import torch
    lib = load_library()
    with torch.cuda.device(torch.device(device)):
        buf = torch.empty(mib << 20, dtype=torch.uint8, device=device)
        out = C.c_double(0.0)
        st = lib.fem_probe_l2_gather(C.c_void_p(buf.data_ptr()), C.c_size_t(buf.numel()), int(row_bytes), int(repeats),
                                     C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out))
    if st != FEM_OK:
        raise FemError(st, "fem_probe_l2_gather")
    return float(out.value)


def cut_static(row_ptr, col_idx, weight, sigma, cut, stream=None) -> None:
    """fem_cut_static on torch CUDA tensors (all on one device): row_ptr int32 [n + 1], col_idx int32 [nnz], weight float32
    [nnz] or None, sigma int8 [n, count] (configuration innermost), cut int64 [count] (written).  Allocates nothing and does
    not synchronise; argument marshalling only."""
    import torch
    lib = load_library()
    want = ((row_ptr, torch.int32), (col_idx, torch.int32), (sigma, torch.int8), (cut, torch.int64)) + (((weight, torch.float32),) if weight is not None else ())
    for t, dt in want:
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.device == sigma.device):
            raise FemError(FEM_EINVAL, "cut_static: tensors must be contiguous CUDA tensors of the documented dtypes on one device")
    n, count = int(sigma.shape[0]), int(sigma.shape[1])
    if row_ptr.numel() != n + 1 or cut.numel() < min(count, CUT_STATIC_MAX_COUNT):
        raise FemError(FEM_EINVAL, "cut_static: row_ptr must have n + 1 entries and cut at least count")
    with torch.cuda.device(sigma.device):
        st_ = stream if stream is not None else torch.cuda.current_stream(sigma.device)
        st = lib.fem_cut_static(n, C.c_void_p(row_ptr.data_ptr()), C.c_void_p(col_idx.data_ptr()),
                                C.c_void_p(weight.data_ptr()) if weight is not None else None, C.c_void_p(sigma.data_ptr()),
                                count, C.c_void_p(cut.data_ptr()), C.c_void_p(st_.cuda_stream))
    if st != FEM_OK:
        raise FemError(st, (lib.fem_cut_static_error() or b"").decode())


def schedule_for(cfg: wl.Config, precise_steps: int = 8) -> Schedule:
    return Schedule(beta=linear_temperature_schedule(cfg.T_max, cfg.T_min, cfg.steps), lr=cfg.lr, beta1=cfg.beta1,
                    beta2=cfg.beta2, eps=cfg.eps, init_scale=cfg.init_scale, precise_steps=precise_steps)
