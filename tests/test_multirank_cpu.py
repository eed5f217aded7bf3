"""world_size-2 gloo test of the N > 1 host logic: replica sharding and the Eq.5 exchange across ranks."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_09285_b200 import multigpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank "anneals" its own replicas: stand-in energies, rank 1 holds the better one
        rng = np.random.default_rng(multigpu.replica_seed(0, rank))
        energies = np.array([-10.0, -12.0]) if rank == 0 else np.array([-15.0, -11.0])
        cfgs = rng.integers(0, 2, size=(2, 9)).astype(np.int32)
        a = int(np.argmin(energies))
        e, owner, cfg = multigpu.best_over_ranks(float(energies[a]), cfgs[a], torch.device("cpu"))
        assert e == -15.0 and owner == 1
        # a tie goes to the lowest rank
        e2, owner2, _ = multigpu.best_over_ranks(-7.0, cfgs[0], torch.device("cpu"))
        assert e2 == -7.0 and owner2 == 0
        out.put((rank, cfg.tolist(), cfgs[a].tolist()))
    finally:
        dist.destroy_process_group()


def test_best_replica_over_two_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = [out.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    got.sort()
    assert got[0][1] == got[1][1] == got[1][2]        # both ranks hold rank 1's configuration


def _anneal_worker(rank, world, port, out):
    """A rank's whole job as bench.py runs it, with the oracle standing in for the device: anneal its OWN replicas from
    replica_seed(base, rank), read out, then the Eq.5 exchange over the ranks."""
    from oracle import fem_oracle as fo
    from paper_2412_09285_b200 import workloads as wl
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inst = wl.torus_maxcut(6, 77, W=7)
        pb = fo.Problem(kind=inst.kind, n=inst.n, q=2, row_ptr=inst.row_ptr, col_idx=inst.col_idx, weight=inst.weight)
        R, N = 4, 80
        st = fo.State(pb, fo.init_fields(multigpu.replica_seed(3, rank), R, inst.n, 1))
        fo.anneal(st, fo.schedule_inverse_proportional(1.0, 0.01, N), fo.Adam())
        cfg = fo.round_configs(pb, st.h)
        _, e_real, _ = fo.energies(pb, cfg)
        a = fo.argmin(e_real)
        e, owner, best = multigpu.best_over_ranks(float(e_real[a]), cfg[a], torch.device("cpu"))
        out.put((rank, e, owner, best.tolist(), e_real.tolist(), cfg[a].tolist()))
    finally:
        dist.destroy_process_group()


def test_two_ranks_anneal_their_own_replicas_and_agree_on_the_best():
    """Replica sharding end to end on the host: rank r's energies are exactly what a single process gets from
    replica_seed(base, r) (no rank sees another's replicas), and every rank ends with the global argmin, lowest rank on ties."""
    from oracle import fem_oracle as fo
    from paper_2412_09285_b200 import workloads as wl
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_anneal_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    inst = wl.torus_maxcut(6, 77, W=7)
    pb = fo.Problem(kind=inst.kind, n=inst.n, q=2, row_ptr=inst.row_ptr, col_idx=inst.col_idx, weight=inst.weight)
    single = []
    for r in range(2):                                 # the same two anneals in ONE process
        st = fo.State(pb, fo.init_fields(multigpu.replica_seed(3, r), 4, inst.n, 1))
        fo.anneal(st, fo.schedule_inverse_proportional(1.0, 0.01, 80), fo.Adam())
        cfg = fo.round_configs(pb, st.h)
        _, e_real, _ = fo.energies(pb, cfg)
        single.append((e_real, cfg))
        assert got[r][4] == e_real.tolist()            # rank r annealed exactly its own seed's replicas
    best_e = [float(s[0].min()) for s in single]
    owner = int(np.argmin(best_e))
    for r in range(2):
        assert got[r][1] == best_e[owner] and got[r][2] == owner
        assert got[r][3] == single[owner][1][fo.argmin(single[owner][0])].tolist()


def test_replica_seeds_are_distinct():
    seeds = {multigpu.replica_seed(0, r) for r in range(64)} | {multigpu.replica_seed(1, r) for r in range(64)}
    assert len(seeds) == 128
