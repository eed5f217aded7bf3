"""Seeded synthetic inputs shaped like the paper's workloads (numpy only).

This module is the one thing the oracle-side tests and the CUDA-side binding share.  It holds
NONE of the method's arithmetic: no marginals, gradients, schedules, optimiser or energies --
only graphs, clause lists and coupling matrices, all from ``numpy.random.Generator(PCG64(seed))``.
The recipes are stated in DESIGN.md section 4; they stand in for the paper's datasets
(G-set, K2000, Walshaw graphs, MaxSAT-2016), none of which is reproduced here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

MAXCUT, ISING, BMINCUT, MAXSAT = 0, 1, 2, 3
KIND_NAMES = {MAXCUT: "maxcut", ISING: "ising", BMINCUT: "bmincut", MAXSAT: "maxsat"}


@dataclass
class Instance:
    """A problem instance on the host.  Graph kinds: symmetric CSR, both directions, no self loops."""
    kind: int
    n: int
    q: int = 2
    row_ptr: Optional[np.ndarray] = None     # int64 [n+1]
    col_idx: Optional[np.ndarray] = None     # int32 [nnz]
    weight: Optional[np.ndarray] = None      # float32 [nnz] or None (= all +1)
    dense_J: Optional[np.ndarray] = None     # float32 [n,n] (ISING only)
    m: int = 0
    clause_ptr: Optional[np.ndarray] = None  # int64 [m+1]
    lits: Optional[np.ndarray] = None        # int32 signed 1-based literals
    lam: float = 0.0                         # bMinCut balance weight
    name: str = ""
    meta: dict = field(default_factory=dict)
    node_weight: Optional[np.ndarray] = None  # float32 [n], bMinCut balance weights V_i (integral, > 0) or None (= all 1)
    lit_state: Optional[np.ndarray] = None    # int32 [len(lits)], non-Boolean SAT: the clause value W_mi in 0..q-1, or None

    @property
    def fields_per_var(self) -> int:
        return self.q if (self.kind == BMINCUT or (self.kind == MAXSAT and self.lit_state is not None)) else 1

    @property
    def nnz(self) -> int:
        return 0 if self.col_idx is None else int(self.col_idx.size)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def csr_from_edges(n: int, u: np.ndarray, v: np.ndarray, w: Optional[np.ndarray]):
    """Undirected edge list (each edge once) -> symmetric CSR sorted by (row, col)."""
    u = np.asarray(u, dtype=np.int64)
    v = np.asarray(v, dtype=np.int64)
    rows = np.concatenate([u, v])
    cols = np.concatenate([v, u])
    order = np.lexsort((cols, rows))
    rows, cols = rows[order], cols[order]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(row_ptr, rows + 1, 1)
    row_ptr = np.cumsum(row_ptr)
    weight = None
    if w is not None:
        ww = np.concatenate([w, w]).astype(np.float32)
        weight = ww[order]
    return row_ptr, cols.astype(np.int32), weight


def erdos_renyi_maxcut(n: int = 800, p: float = 0.06, seed: int = 1000, pm1: bool = False) -> Instance:
    """G(n,p), every pair i<j kept with probability p; weights +1 (or +-1 fair coin)."""
    rng = _rng(seed)
    iu, ju = np.triu_indices(n, k=1)
    keep = rng.random(iu.size) < p
    u, v = iu[keep], ju[keep]
    w = None
    if pm1:
        w = rng.integers(0, 2, size=u.size).astype(np.float32) * 2 - 1
    row_ptr, col, weight = csr_from_edges(n, u, v, w)
    return Instance(MAXCUT, n, 2, row_ptr, col, weight, name=f"maxcut_er_n{n}_p{p}", meta={"edges": int(u.size)})


def torus_maxcut(L: int = 200, seed: int = 1001, W: Optional[int] = None) -> Instance:
    """2D toroidal grid LxW, node (r,c) -> r*W+c, edges to (r,c+1) and (r+1,c) mod size, weights +-1."""
    W = L if W is None else W
    rng = _rng(seed)
    r, c = np.meshgrid(np.arange(L), np.arange(W), indexing="ij")
    me = (r * W + c).ravel()
    right = (r * W + (c + 1) % W).ravel()
    down = (((r + 1) % L) * W + c).ravel()
    u = np.concatenate([me, me])
    v = np.concatenate([right, down])
    # tiny tori (size 2) would create duplicate edges; drop duplicates and self loops
    a, b = np.minimum(u, v), np.maximum(u, v)
    key = np.unique(a * (L * W) + b)
    a, b = key // (L * W), key % (L * W)
    ok = a != b
    a, b = a[ok], b[ok]
    w = rng.integers(0, 2, size=a.size).astype(np.float32) * 2 - 1
    row_ptr, col, weight = csr_from_edges(L * W, a, b, w)
    return Instance(MAXCUT, L * W, 2, row_ptr, col, weight, name=f"maxcut_torus_{L}x{W}", meta={"edges": int(a.size)})


def preferential_attachment(n: int = 100000, m: int = 3, seed: int = 1007, pm1: bool = True) -> Instance:
    """Scale-free graph by preferential attachment (the shape of the G-set's scale-free family): nodes
    0..m form a clique; every later node attaches to m DISTINCT earlier nodes drawn with probability proportional to their
    degree (one draw = one entry of the list of all edge endpoints so far; repeats redrawn).  Weights +-1 fair coin or +1."""
    rng = _rng(seed)
    ends = np.empty(2 * (m * (m + 1) // 2 + (n - m - 1) * m), dtype=np.int64)
    u_list, v_list = [], []
    k = 0
    for a in range(m + 1):
        for b in range(a + 1, m + 1):
            u_list.append(a); v_list.append(b)
            ends[k] = a; ends[k + 1] = b
            k += 2
    draws = rng.random((n, 2 * m + 8))  # uniform numbers per node: enough for the redraws in all but freak cases
    for node in range(m + 1, n):
        chosen = []
        t = 0
        while len(chosen) < m:
            x = draws[node, t] if t < draws.shape[1] else rng.random()
            t += 1
            cand = int(ends[int(x * k)])
            if cand not in chosen:
                chosen.append(cand)
        for cnd in chosen:
            u_list.append(cnd); v_list.append(node)
            ends[k] = cnd; ends[k + 1] = node
            k += 2
    u = np.asarray(u_list, dtype=np.int64)
    v = np.asarray(v_list, dtype=np.int64)
    w = rng.integers(0, 2, size=u.size).astype(np.float32) * 2 - 1 if pm1 else None
    row_ptr, col, weight = csr_from_edges(n, u, v, w)
    return Instance(MAXCUT, n, 2, row_ptr, col, weight, name=f"maxcut_scalefree_n{n}_m{m}",
                    meta={"edges": int(u.size), "max_degree": int(np.diff(row_ptr).max())})


def _random_regular_edges(n: int, d: int, rng: np.random.Generator):
    """Pairing model with repair: shuffle the d*n stubs, pair consecutive stubs, then re-pair the stubs
    of bad pairs (self loops, repeated edges) together with as many random good pairs until none is left."""
    assert (n * d) % 2 == 0 and d < n
    stubs = np.repeat(np.arange(n, dtype=np.int64), d)
    rng.shuffle(stubs)
    u, v = stubs[0::2].copy(), stubs[1::2].copy()
    for _ in range(10000):
        a, b = np.minimum(u, v), np.maximum(u, v)
        key = a * n + b
        order = np.argsort(key, kind="stable")
        ks = key[order]
        dup = np.zeros(key.size, dtype=bool)
        dup[order[1:]] = ks[1:] == ks[:-1]
        bad = dup | (u == v)
        nb = int(bad.sum())
        if nb == 0:
            return a, b
        bad_idx = np.flatnonzero(bad)
        good_idx = np.flatnonzero(~bad)
        extra = rng.choice(good_idx, size=min(good_idx.size, max(nb, 8)), replace=False)
        sel = np.concatenate([bad_idx, extra])
        pool = np.concatenate([u[sel], v[sel]])
        rng.shuffle(pool)
        u[sel], v[sel] = pool[0::2], pool[1::2]
    raise RuntimeError("random regular graph repair did not converge")


def random_regular(n: int, d: int, seed: int, kind: int = MAXCUT, q: int = 2, pm1: bool = False,
                   lam: float = 0.0) -> Instance:
    rng = _rng(seed)
    a, b = _random_regular_edges(n, d, rng)
    w = None
    if pm1:
        w = rng.integers(0, 2, size=a.size).astype(np.float32) * 2 - 1
    row_ptr, col, weight = csr_from_edges(n, a, b, w)
    return Instance(kind, n, q, row_ptr, col, weight, lam=lam,
                    name=f"{KIND_NAMES[kind]}_reg{d}_n{n}" + (f"_q{q}" if kind == BMINCUT else ""),
                    meta={"edges": int(a.size), "degree": d})


def random_ksat(n: int = 20000, m: int = 200000, k: int = 4, seed: int = 1003) -> Instance:
    """Each clause: k distinct variables drawn uniformly (rejection), each literal negated with prob 1/2."""
    rng = _rng(seed)
    var = rng.integers(0, n, size=(m, k))
    while True:
        s = np.sort(var, axis=1)
        bad = (s[:, 1:] == s[:, :-1]).any(axis=1)
        nb = int(bad.sum())
        if nb == 0:
            break
        var[bad] = rng.integers(0, n, size=(nb, k))
    neg = rng.integers(0, 2, size=(m, k)).astype(bool)
    lits = (var + 1).astype(np.int32)
    lits[neg] = -lits[neg]
    clause_ptr = np.arange(m + 1, dtype=np.int64) * k
    return Instance(MAXSAT, n, 2, m=m, clause_ptr=clause_ptr, lits=lits.ravel().copy(),
                    name=f"max{k}sat_n{n}_m{m}", meta={"k": k})


def random_qsat(n: int, m: int, k: int, q: int, seed: int, kmin: Optional[int] = None) -> Instance:
    """Random non-Boolean SAT: m clauses of k (or kmin..k) distinct variables, each with a uniformly drawn
    clause value W_mi in 0..q-1; a clause is violated when no variable takes its clause value."""
    rng = _rng(seed)
    ptr, lits, states = [0], [], []
    for _ in range(m):
        kk = k if kmin is None else int(rng.integers(kmin, k + 1))
        vs = rng.choice(n, size=kk, replace=False)
        lits += [int(v) + 1 for v in vs]
        states += [int(x) for x in rng.integers(0, q, size=kk)]
        ptr.append(len(lits))
    return Instance(MAXSAT, n, q, m=m, clause_ptr=np.asarray(ptr, np.int64), lits=np.asarray(lits, np.int32),
                    lit_state=np.asarray(states, np.int32), name=f"qsat_q{q}_k{k}_n{n}_m{m}")


def sk_dense(n: int = 4096, seed: int = 1005) -> Instance:
    """Sherrington-Kirkpatrick couplings: J_ij = J_ji ~ N(0, 1/n) for i<j, J_ii = 0, fp32."""
    rng = _rng(seed)
    g = rng.standard_normal((n, n)).astype(np.float32) / np.float32(np.sqrt(n))
    J = np.triu(g, k=1)
    J = J + J.T
    return Instance(ISING, n, 2, dense_J=np.ascontiguousarray(J, dtype=np.float32), name=f"sk_dense_n{n}")


def sparse_ising_from(inst: Instance, scale: float = -0.5) -> Instance:
    """Same graph as a MaxCut instance, as an Ising instance with J = scale * W (J = -W/2 maps MaxCut to Ising)."""
    w = np.ones(inst.nnz, dtype=np.float32) if inst.weight is None else inst.weight
    return Instance(ISING, inst.n, 2, inst.row_ptr, inst.col_idx, (w * np.float32(scale)).astype(np.float32),
                    name="ising_of_" + inst.name)


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs.  Graph seed = 1000 + index; field seed = 0.
# Adam lr 0.1 / 0.9 / 0.999 / 1e-8, T from 1.0 to 0.01 linearly, h(0) = 0.001 N(0,1) for all.
# ------------------------------------------------------------------------------------------------
@dataclass
class Config:
    name: str
    make: callable
    R: int
    steps: int
    T_max: float = 1.0
    T_min: float = 0.01
    lr: float = 0.1
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8
    init_scale: float = 1e-3
    field_seed: int = 0


CONFIGS = {
    "cfg0": Config("cfg0 MaxCut ER(800,0.06) W=+1 R=32 N=500", lambda: erdos_renyi_maxcut(800, 0.06, 1000), 32, 500),
    "cfg1": Config("cfg1 MaxCut torus 200x200 W=+-1 R=256 N=2000", lambda: torus_maxcut(200, 1001), 256, 2000),
    "cfg2": Config("cfg2 bMinCut q=8 10-regular n=100000 lambda=0.05/n R=64 N=1000",
                   lambda: random_regular(100000, 10, 1002, BMINCUT, 8, lam=0.05 / 100000), 64, 1000),
    "cfg3": Config("cfg3 Max-4-SAT n=20000 m=200000 R=128 N=2000", lambda: random_ksat(20000, 200000, 4, 1003), 128, 2000),
    "cfg4a": Config("cfg4a MaxCut 3-regular n=1000000 W=+-1 R=32 N=1000",
                    lambda: random_regular(1000000, 3, 1004, MAXCUT, pm1=True), 32, 1000),
    # not a BASELINE.json config: the size of the paper's own MaxSAT-2016 instances (N 70-300, M 700-2600,
    # 50-800 replicas, 50-500 steps; mean 0.074 s per instance on the paper's GPU), for the replica-persistent Max-SAT kernel
    "sat2016": Config("sat2016 Max-4-SAT n=300 m=2600 R=128 N=500 (MaxSAT-2016-sized stand-in)",
                      lambda: random_ksat(300, 2600, 4, 1006), 128, 500),
    # not a BASELINE.json config: degree-skewed rows (north_star subsystem 2), shaped like the G-set's scale-free graphs
    # scaled up: preferential attachment, 3 edges per new node, weights +-1
    "skew": Config("skew MaxCut scale-free (preferential attachment m=3) n=100000 W=+-1 R=64 N=1000",
                   lambda: preferential_attachment(100000, 3, 1007, pm1=True), 64, 1000),
    "cfg4b": Config("cfg4b SK dense n=4096 J~N(0,1/n) R=1024 N=1000", lambda: sk_dense(4096, 1005), 1024, 1000),
}
