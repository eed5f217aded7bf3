#!/usr/bin/env python
"""bench.py -- throughput of the FEM annealing hot path on B200 (contract: see DESIGN.md section 9).

One "step" of this benchmark is one pass of the WHOLE hot path over one batch of synthetic input:
seeded initial fields, all annealing steps of the schedule (fused step kernel per step), rounding,
per-replica energies and the best-replica argmin.  The headline workload is BASELINE.json's LARGEST single-GPU
configuration, cfg2 (bMinCut, q = 8, random 10-regular graph, n = 100,000, R = 64, 1000 annealing steps: 51.2 M
fields); the same JSON line carries a `per_config` object with a short measured run (value, roofline, e2e, clocks) of
every other BASELINE.json workload (cfg0, cfg1, cfg3, cfg4a, cfg4b).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference] [--no-per-config]

`value`  : variable-replica updates/s with the problem already resident in HBM (CUDA events).
`e2e`    : the same metric through the public API from HOST buffers: fem_create (uploads the problem
           from pinned host memory) + fem_anneal + fem_result (downloads energies and the best config).
`roofline`: the fused fp32 step kernel, algorithmic bytes per launch / its mean launch duration measured
           with CUDA events inside the timed region, against the measured HBM copy bandwidth.
`cpu_baseline`: the oracle (oracle/fem_oracle.c, as it stands) on this box's host cores, bounded sample.
N > 1: replicas are independent, so every rank anneals its own R replicas (weak scaling, no data-path
collective); one tiny exchange at the end picks the best replica over all ranks (Eq.5).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "variable-replica updates/s"
UNIT = "updates/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def load_peak_file():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)
    return {}


def load_traffic(workload: str):
    """dram bytes per launch of the fused step kernel from the committed ncu capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f).get(workload)
    return None


class ClockSampler:
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self, t_begin=None, t_end=None):
        """Samples whose wall-clock timestamp falls in [t_begin, t_end] (the timed region); if the region was shorter
        than the sampling period, the samples nearest to it."""
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        import datetime
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = []
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(parts[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(parts[1]), float(parts[2]),
                             [nm for nm, val in zip(names, parts[4:8]) if val.lower().startswith("active")]))
            except ValueError:
                continue
        self.f.close()
        os.unlink(self.f.name)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        inside = [r for r in rows if t_begin is not None and t_begin <= r[0] <= t_end]
        where = "inside the timed region"
        if not inside:
            mid = 0.5 * ((t_begin or rows[-1][0]) + (t_end or rows[-1][0]))
            inside = sorted(rows, key=lambda r: abs(r[0] - mid))[:3]
            where = "nearest to the timed region (shorter than the 20 ms sampling period)"
        return {"sm_mhz": float(np.median([r[1] for r in inside])), "sm_max_mhz": max(r[2] for r in inside),
                "reasons": sorted({x for r in inside for x in r[3]}), "samples": len(inside), "sampled": where}


def oracle_sample(cfg, inst, seconds_target: float = 12.0):
    """Time the oracle on a bounded sample of the workload: a few annealing steps at full n and R."""
    from oracle import fem_oracle as fo
    pb = fo.Problem(kind=inst.kind, n=inst.n, q=inst.q, row_ptr=inst.row_ptr, col_idx=inst.col_idx, weight=inst.weight,
                    dense_J=inst.dense_J, m=inst.m, clause_ptr=inst.clause_ptr, lits=inst.lits)
    beta = fo.schedule_inverse_proportional(cfg.T_max, cfg.T_min, cfg.steps)
    h0 = fo.init_fields(cfg.field_seed, cfg.R, inst.n, inst.fields_per_var, cfg.init_scale)
    adam = fo.Adam(cfg.lr, cfg.beta1, cfg.beta2, cfg.eps)
    out = {}
    for openmp in (False, True):
        st = fo.State(pb, h0)
        t0 = time.perf_counter()
        fo.anneal(st, beta, adam, inst.lam, t_end=1, openmp=openmp)
        one = time.perf_counter() - t0
        nsteps = int(max(2, min(cfg.steps - 1, seconds_target / 2 / max(one, 1e-6))))
        t0 = time.perf_counter()
        fo.anneal(st, beta, adam, inst.lam, t_end=1 + nsteps, openmp=openmp)
        dt = time.perf_counter() - t0
        out[openmp] = (inst.n * cfg.R * nsteps / dt, nsteps, fo.num_threads(openmp))
    return out


def run_reference(args, cfg, inst):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample."""
    from oracle import fem_oracle as fo
    pb = fo.Problem(kind=inst.kind, n=inst.n, q=inst.q, row_ptr=inst.row_ptr, col_idx=inst.col_idx, weight=inst.weight,
                    dense_J=inst.dense_J, m=inst.m, clause_ptr=inst.clause_ptr, lits=inst.lits)
    beta = fo.schedule_inverse_proportional(cfg.T_max, cfg.T_min, cfg.steps)
    h0 = fo.init_fields(cfg.field_seed, cfg.R, inst.n, inst.fields_per_var, cfg.init_scale)
    adam = fo.Adam(cfg.lr, cfg.beta1, cfg.beta2, cfg.eps)
    st = fo.State(pb, h0)
    t0 = time.perf_counter()
    fo.anneal(st, beta, adam, inst.lam, t_end=1, openmp=True)
    one = time.perf_counter() - t0
    total = args.steps + args.warmup
    per = int(max(1, min((cfg.steps - 1) // max(total, 1), 120.0 / total / max(one, 1e-6))))
    t = 1
    for _ in range(args.warmup):
        fo.anneal(st, beta, adam, inst.lam, t_end=t + per, openmp=True)
        t += per
    t0 = time.perf_counter()
    for _ in range(args.steps):
        fo.anneal(st, beta, adam, inst.lam, t_end=t + per, openmp=True)
        t += per
    dt = time.perf_counter() - t0
    value = inst.n * cfg.R * per * args.steps / dt
    cores = fo.num_threads(True)
    sample = f"{per} annealing steps at full n={inst.n}, R={cfg.R} per bench step (of {cfg.steps})"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "note": "oracle/fem_oracle.c on host cores (OpenMP over replicas)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def measure_l2_peak(fem, local_rank):
    """L2 -> SM read bandwidth of this device, measured live by the library's probe kernel (fem_probe_l2_read: a 32 MiB
    buffer, resident in the 126 MB L2, read 200 times from all SMs with 16-byte loads that bypass L1)."""
    return max(fem.probe_l2_read(f"cuda:{local_rank}", 32, 200) for _ in range(3))


def run_workload(args, name, steps, warmup, ctx, with_e2e=True):
    """Time `steps` passes of the whole hot path of one workload (after `warmup` untimed ones); returns the fields of
    its JSON entry (rank 0) -- value, ms_per_step, roofline, e2e, clocks, ..."""
    torch, dist, fem, multigpu, wl = ctx["torch"], ctx["dist"], ctx["fem"], ctx["multigpu"], ctx["wl"]
    rank, local_rank, world, dev, use_dist = ctx["rank"], ctx["local_rank"], ctx["world"], ctx["dev"], ctx["use_dist"]
    cfg = wl.CONFIGS[name]
    if args.anneal_steps is not None:
        import dataclasses
        cfg = dataclasses.replace(cfg, steps=args.anneal_steps, name=cfg.name + f" [schedule cut to {args.anneal_steps} steps]")
    inst = cfg.make()
    R, N, n = cfg.R, cfg.steps, inst.n
    sched = fem.schedule_for(cfg, precise_steps=args.precise_steps)
    K = min(args.precise_steps, N)
    variant = None
    if args.optimizer != "adam" or args.manipulated:
        if args.optimizer == "rmsprop":
            sched.optimizer, sched.lr, sched.alpha, sched.momentum = fem.RMSPROP, 0.05, 0.9, 0.5
        elif args.optimizer == "sgd":
            sched.optimizer, sched.lr, sched.momentum = fem.SGD, 0.5, 0.8
        sched.manipulated = args.manipulated
        variant = f"{args.optimizer}{'+manipulated gradients' if args.manipulated else ''} (not the BASELINE.json configuration)"

    def apply_options(eng):
        if args.replica_block is not None:
            eng.set_option("replica_block", args.replica_block)
        if args.steps_per_block is not None:
            eng.set_option("steps_per_block", args.steps_per_block)
        for kv in args.opt:
            key, _, val = kv.partition("=")
            eng.set_option(key, int(val))

    eng = fem.Fem(inst, R, device=f"cuda:{local_rank}")
    apply_options(eng)
    flush = ctx["flush"]

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    def one_pass(seed, ev=None):
        """The whole hot path on resident inputs; `ev` collects (start, end) events around the fp32 bulk."""
        flush.zero_()
        eng.reset()
        if ev is not None:
            z = torch.cuda.Event(enable_timing=True)
            z.record()
        eng.anneal(sched, R, seed=seed, stop_after=K)          # init + wide phase
        if ev is not None:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = eng.info("launches")
            a.record()
        eng.anneal(sched, R, seed=seed, stop_after=N)          # launches of the fused fp32 step kernel (+1 narrowing)
        if ev is not None:
            b.record()
        eng.readout()                                          # rounding + energies + argmin
        if ev is not None:
            c = torch.cuda.Event(enable_timing=True)
            c.record()
            ev.append((a, b, eng.info("launches") - l0 - (1 if K > 0 else 0), z, c))

    sampler = ClockSampler(local_rank) if rank == 0 else None   # started before warm-up: nvidia-smi takes a while to start
    if sampler is not None and sampler.p is not None:           # ... so wait for its first line (short workloads: cfg 0)
        t_wait = time.time()
        while os.path.getsize(sampler.f.name) == 0 and time.time() - t_wait < 5.0:
            time.sleep(0.02)
    for w in range(warmup):
        one_pass(multigpu.replica_seed(1000 + w, rank))
    barrier()
    launches0 = eng.info("launches")
    wall_begin = time.time()
    bulk_events = []
    start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    start.record()
    for k in range(steps):
        one_pass(multigpu.replica_seed(k, rank), bulk_events)
    end.record()
    barrier()
    elapsed_ms = start.elapsed_time(end)
    wall_end = time.time()
    clocks = sampler.stop(wall_begin, wall_end) if sampler else None
    launches = eng.info("launches") - launches0
    l2_persist_bytes = eng.info("l2_persist_bytes")            # (read before fem_result gives the set-aside back)
    res = eng.result()
    bulk_ms = sum(e[0].elapsed_time(e[1]) for e in bulk_events)
    bulk_launches = sum(e[2] for e in bulk_events)
    init_wide_ms = sum(e[3].elapsed_time(e[0]) for e in bulk_events) / max(len(bulk_events), 1)
    readout_ms = sum(e[1].elapsed_time(e[4]) for e in bulk_events) / max(len(bulk_events), 1)
    # algorithmic bytes of one launch: the whole step's bytes spread over the launches that make up a step
    step_bytes = eng.info("step_bytes") * (N - K) * steps / max(bulk_launches, 1)
    info = {k: eng.info(k) for k in ("tc_launches", "tc8_launches", "persist_launches", "tma_launches", "si_launches", "replica_block", "nnz")}
    info["l2_persist_bytes"] = l2_persist_bytes
    eng.close()

    # ---- e2e through the public API from host buffers (pinned), host<->device copies inside the timed region
    e2e_ms, e2e_steps, h2d, d2h = 0.0, 0, 0, 0
    if with_e2e:
        def pin(a):
            return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        pinned = wl.Instance(inst.kind, inst.n, inst.q, pin(inst.row_ptr), pin(inst.col_idx), pin(inst.weight),
                             pin(inst.dense_J), inst.m, pin(inst.clause_ptr), pin(inst.lits), inst.lam, inst.name)
        h2d = sum(a.nbytes for a in (pinned.row_ptr, pinned.col_idx, pinned.weight, pinned.dense_J, pinned.clause_ptr,
                                     pinned.lits) if a is not None)
        d2h = 4 + 4 * n + 8 * R + 8 * R + 4 * R * inst.q

        def e2e_pass(seed):
            e = fem.Fem(pinned, R, device=f"cuda:{local_rank}")     # fem_create: validate + upload
            apply_options(e)
            e.anneal(sched, R, seed=seed)
            out = e.result()                                        # readout + download + synchronize
            e.close()
            return out

        e2e_pass(7)
        barrier()
        t0 = time.perf_counter()
        e2e_steps = max(1, min(steps, 3))
        for k in range(e2e_steps):
            e2e_pass(multigpu.replica_seed(k, rank))
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3

    # ---- max over ranks, best replica over ranks
    times = torch.tensor([elapsed_ms, e2e_ms, bulk_ms], dtype=torch.float64, device=dev)
    if use_dist:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    # Eq.5 across ranks: 8 bytes per rank, then the owner's configuration
    best_energy, best_owner, _ = multigpu.best_over_ranks(float(res["energy"][res["best_replica"]]),
                                                          res["best_config"], dev)
    elapsed_ms, e2e_ms, bulk_ms = [float(x) for x in times.tolist()]
    if rank != 0:
        return None, cfg, inst

    updates = float(n) * R * N
    value = updates * steps * world / (elapsed_ms * 1e-3)
    peak, peak_src = load_peaks()
    kernel_us = bulk_ms * 1e3 / bulk_launches
    peaks = load_peak_file()
    share = bulk_ms / elapsed_ms
    if inst.dense_J is not None and info["tc_launches"] > 0:
        # dense couplings: J.M is a GEMM (2 n^2 R flop per step) on tcgen05 kind::tf32.  The 3xTF32 split issues
        # three MMAs per algorithmic product; `achieved` counts the ALGORITHMIC flops only.
        flops = 2.0 * n * n * R
        achieved = flops / (kernel_us * 1e-6) / 1e12
        bf16 = float(peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops", 1671.0)))
        tf32_peak = 0.5 * bf16
        i8 = info["tc8_launches"] > 0
        roofline = {"bound": "tensor",
                    "kernel": ("dense_i8_step_kernel (tcgen05 kind::i8: both operands as three signed 8-bit digits of a 23-bit fixed point, six "
                               "MMAs per product into exact int32 accumulators; FEM update fused in the TMEM epilogue)" if i8 else
                               "dense_tc_step_kernel (tcgen05 3xTF32 GEMM, FEM update fused in the TMEM epilogue)"),
                    "achieved": achieved, "peak": tf32_peak, "unit": "TFLOP/s", "frac": achieved / tf32_peak,
                    "traffic": load_traffic(name),
                    "peak_source": "0.5 x measured sustained bf16 cuBLAS TFLOP/s (MEASURED_PEAKS.json; tf32:bf16 nominal ratio 1:2): the "
                                   "roof of an fp32-accurate product issued as ONE tf32 MMA per product; `achieved` counts the algorithmic "
                                   "2 n^2 R flop only",
                    "algorithmic_flops_per_launch": flops,
                    "mma_tflops_issued": (6.0 if i8 else 3.0) * achieved,
                    "issued_frac_of_own_dtype_peak": ((6.0 * achieved) / (2.0 * bf16)) if i8 else (3.0 * achieved / tf32_peak),
                    "own_dtype_peak_source": ("int8: 2 x measured sustained bf16 (nominal ratio 2:1)" if i8 else "tf32: 0.5 x measured sustained bf16"),
                    "kernel_us": kernel_us, "kernel_share_of_step": share}
    elif info["persist_launches"] > 0:
        # small sparse two-state problem: replica-persistent cluster kernel, state in registers, gathers from shared
        # memory, no HBM or L2 traffic during the anneal -- no bandwidth or flop roof applies.  What SURVEY 8(d) asks
        # for here is the time per annealing step; the ncu issue / LSU counters are in profiles/ (DESIGN.md section 6).
        roofline = {"bound": "latency", "kernel": "persist_q2_kernel<float> (one cluster per replica, all steps in one launch)",
                    "achieved": bulk_ms * 1e3 / ((N - K) * steps), "peak": None, "unit": "us per annealing step",
                    "frac": None, "traffic": load_traffic(name),
                    "note": "launch- and latency-bound by construction (614 KB of state, 500 dependent steps): an HBM "
                            "fraction is meaningless here (SURVEY 8(d)); see profiles/ for the issue-slot and shared-memory counters",
                    "kernel_us": kernel_us, "us_per_anneal_step": bulk_ms * 1e3 / ((N - K) * steps),
                    "kernel_share_of_step": share}
    elif inst.kind == wl.MAXSAT:
        # the state (41 MB at cfg 3) is L2-resident; the step gathers (k-1) rows of R floats per literal occurrence out
        # of L2: algorithmic L2 bytes per step = gathers + 28 B per field (h, m1, m2 in and out, m out) + occurrence table
        ks = int(np.diff(inst.clause_ptr).max()) - 1
        nocc = int(inst.lits.size)
        l2_bytes_step = 4.0 * nocc * ks * R + 28.0 * n * R + 4.0 * nocc * max(1, 1 << (ks - 1).bit_length())
        per_launch = l2_bytes_step * (N - K) * steps / max(bulk_launches, 1)
        achieved = per_launch / (kernel_us * 1e-6) / 1e9
        l2_peak = ctx["l2_peak"]()
        roofline = {"bound": "l2", "kernel": "step_q2_kernel<float, SAT> (fused clause products + entropy gradient + Adam)",
                    "achieved": achieved, "peak": l2_peak, "unit": "GB/s", "frac": achieved / l2_peak,
                    "traffic": load_traffic(name),
                    "peak_source": "L2 -> SM read bandwidth measured in this run (fem_probe_l2_read: 32 MiB resident buffer, 16-byte loads bypassing L1)",
                    "algorithmic_l2_bytes_per_launch": per_launch, "kernel_us": kernel_us, "kernel_share_of_step": share,
                    "hbm_frac_of_compulsory_bytes": step_bytes / (kernel_us * 1e-6) / 1e9 / peak,
                    "l2_gather_probe_gbs": {"32MiB": fem.probe_l2_gather(f"cuda:{local_rank}", 32, int(min(512, max(64, 4 * R)))),
                                            "row_bytes": int(min(512, max(64, 4 * R))),
                                            "what": "random-row reads of the same row length out of a 32 MiB working set (fem_probe_l2_gather): the "
                                                    "rate of the step's own access pattern; `peak` above is the sequential-read figure"},
                    "note": "state is L2-resident: the binding roof is L2 -> SM gather bandwidth, not HBM (DESIGN.md section 6); "
                            "rows gathered more than once by an SM can be served by its L1, so `achieved` (algorithmic gather bytes) is an upper bound on the L2 traffic"}
    else:
        achieved = step_bytes / (kernel_us * 1e-6) / 1e9
        kname = (("potts_si_kernel (state-innermost replica blocks: a lane owns the q states of a (variable, replica) cell; fused "
                  "softmax + gather + balance + chain rule + optimiser)" if info["si_launches"] > 0 else
                  "potts_tma_kernel (rows staged by cp.async.bulk one variable ahead; fused softmax + gather + balance + "
                  "chain rule + optimiser)" if info["tma_launches"] > 0 else
                  "potts_team_kernel<float> (fused softmax + gather + balance + chain rule + optimiser)")
                 if inst.kind == wl.BMINCUT else
                 "step_q2_kernel<float> (fused gather + entropy gradient + Adam)")
        roofline = {"bound": "hbm", "kernel": kname,
                    "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": load_traffic(name), "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": step_bytes, "kernel_us": kernel_us,
                    "kernel_share_of_step": share}
        if inst.kind == wl.BMINCUT:
            # what binds the Potts step: every neighbour row comes out of L2 (4 B per field and neighbour),
            # so the SM <-> L2 traffic per field is 12 B own rows + 4 deg B gathers + 16 B stores, and the streamed arrays pass
            # through L2 a second time on their way from / to DRAM.  The gather rate of this device out of a working set of
            # the block's footprint (five fp32 arrays of the block) is measured live beside the 32 MiB figure.
            deg_mean = float(info["nnz"]) / n
            l2_side = (12.0 + 4.0 * deg_mean + 16.0) * n * inst.q * info["replica_block"]
            foot_mib = int(min(1024, max(1, round(20.0 * n * inst.q * info["replica_block"] / 2 ** 20))))
            seg = int(min(512, max(64, 16 * info["replica_block"])))
            roofline["l2_side_bytes_per_launch"] = l2_side
            roofline["l2_side_gbs"] = l2_side / (kernel_us * 1e-6) / 1e9
            roofline["l2_gather_probe_gbs"] = {"32MiB": fem.probe_l2_gather(f"cuda:{local_rank}", 32, seg),
                                               f"{foot_mib}MiB (block footprint)": fem.probe_l2_gather(f"cuda:{local_rank}", foot_mib, seg),
                                               "row_bytes": seg}
            roofline["note"] = ("the step moves (12 + 4 deg + 16) B per field between SMs and L2 against 24 B of compulsory HBM traffic; "
                                "with a block footprint beyond one die's half of the L2 the measured SM <-> L2 rate, not HBM, is what "
                                "binds (l2_gather_probe_gbs: pure random-row reads, footprint-sized vs 32 MiB working set)")
            roofline["l2_persist_bytes"] = info["l2_persist_bytes"]   # persisting L2 set-aside holding the block's gather buffers
        if info["replica_block"] < R and 20.0 * n * inst.fields_per_var * info["replica_block"] < 0.5 * 126e6:
            roofline["note"] = ("replica block L2-resident for the whole anneal: `achieved` is the ALGORITHMIC-byte rate "
                                "(24 B per field per step / time) served out of L2, not DRAM utilisation; it is compared with "
                                "the HBM copy peak because that is what a streaming implementation would be bound by")
    entry = {
        "value": value, "ms_per_step": elapsed_ms / steps, "steps": steps, "warmup": warmup,
        "config": {"workload": cfg.name, "instance": inst.name, "n": n, "R_per_gpu": R, "anneal_steps": N,
                   "precise_steps": K, "replica_block": info["replica_block"],
                   "l2": "256 MiB buffer written between timed passes (L2 flush)",
                   "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                   **({"variant": variant} if variant else {})},
        "roofline": roofline,
        "gpu_launches": int(launches),
        "clocks": clocks,
        "breakdown_ms_per_pass": {"init_and_wide_phase": init_wide_ms, "fp32_steps": bulk_ms / max(len(bulk_events), 1),
                                  "readout": readout_ms, "note": "rank 0, CUDA events; the rest of ms_per_step is the L2 flush"},
        **({"field_updates_per_s": value * inst.q} if inst.kind == wl.BMINCUT else {}),
        "result": {"best_energy": best_energy, "best_rank": best_owner, "mean_energy": float(np.mean(res["energy"]))},
    }
    if with_e2e:
        entry["e2e"] = {"value": updates * e2e_steps * world / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h, "steps": e2e_steps}
    return entry, cfg, inst


PER_CONFIG = ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4a", "cfg4b", "skew"]   # skew: not a BASELINE.json config (degree-skewed rows)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2",
                    help="headline workload: cfg2 by default, the largest single-GPU configuration of BASELINE.json (51.2 M fields, "
                         "1.23 GB of compulsory traffic per annealing step)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true",
                    help="skip the per_config object (one short timed run of every other BASELINE.json workload)")
    ap.add_argument("--replica-block", type=int, default=None, help="override the replica_block option")
    ap.add_argument("--steps-per-block", type=int, default=None)
    ap.add_argument("--precise-steps", type=int, default=8)
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="library option passed to fem_set_option (e.g. tensor_cores=0); repeatable")
    ap.add_argument("--optimizer", default="adam", choices=["adam", "rmsprop", "sgd"],
                    help="SURVEY 8(f): adam is the BASELINE.json configuration; rmsprop (lr 0.05, alpha 0.9, momentum 0.5) and "
                         "sgd (lr 0.5, momentum 0.8) are variants, named in config")
    ap.add_argument("--manipulated", action="store_true", help="SURVEY 8(f): manipulated gradients S25/S27/S30 (variant)")
    ap.add_argument("--anneal-steps", type=int, default=None,
                    help="shorten the schedule (profiling under ncu only; such a run is not a bench value)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    from paper_2412_09285_b200 import workloads as wl
    if args.impl == "reference":
        if rank != 0:
            return
        cfg = wl.CONFIGS[args.workload]
        if args.anneal_steps is not None:
            import dataclasses
            cfg = dataclasses.replace(cfg, steps=args.anneal_steps, name=cfg.name + f" [schedule cut to {args.anneal_steps} steps]")
        run_reference(args, cfg, cfg.make())
        return

    import torch
    import torch.distributed as dist
    from paper_2412_09285_b200 import fem, multigpu

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the FEM path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    # under torchrun (even with one rank) the collectives of the N > 1 path are really run, over NCCL
    use_dist = world > 1 or ("RANK" in os.environ and "MASTER_ADDR" in os.environ)
    if use_dist:
        dist.init_process_group("nccl", device_id=dev)
    l2_cache = {}

    def l2_peak():
        if "v" not in l2_cache:
            l2_cache["v"] = measure_l2_peak(fem, local_rank)
        return l2_cache["v"]

    ctx = {"torch": torch, "dist": dist, "fem": fem, "multigpu": multigpu, "wl": wl, "rank": rank, "local_rank": local_rank,
           "world": world, "dev": dev, "use_dist": use_dist, "l2_peak": l2_peak,
           "flush": torch.empty(256 << 20, dtype=torch.uint8, device=dev)}   # > L2 (126 MB)

    head, cfg, inst = run_workload(args, args.workload, args.steps, args.warmup, ctx)
    per_config = {}
    plain = (args.anneal_steps is None and args.optimizer == "adam" and not args.manipulated and not args.opt
             and args.replica_block is None and args.steps_per_block is None)
    if not args.no_per_config and plain and args.workload == "cfg2":
        # every other BASELINE.json workload, a short run each (3 warm-up + up to 5 timed passes) so that the one line the
        # driver records carries a measured number, roofline and clock record for all six
        for name in PER_CONFIG:
            if name == args.workload:
                continue
            e, _, _ = run_workload(args, name, max(2, min(args.steps, 5)), 3, ctx)
            if rank == 0:
                per_config[name] = e
    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic"}
        for k in ("config", "roofline", "e2e", "gpu_launches", "clocks", "breakdown_ms_per_pass", "field_updates_per_s", "result"):
            if k in head:
                line[k] = head[k]
        if per_config:
            per_config[args.workload] = {k: head[k] for k in ("value", "ms_per_step", "roofline", "e2e", "clocks", "config")}
            line["per_config"] = {k: per_config[k] for k in PER_CONFIG if k in per_config}
            line["gpu_launches"] = int(sum(v.get("gpu_launches", 0) for k, v in per_config.items() if k != args.workload)
                                       + head["gpu_launches"])
            line["gpu_launches_headline"] = head["gpu_launches"]
        if not args.no_cpu_baseline and world == 1:
            o = oracle_sample(cfg, inst)
            v1, s1, c1 = o[False]
            vN, sN, cN = o[True]
            use_omp = vN > v1
            line["cpu_baseline"] = {"value": vN if use_omp else v1, "unit": UNIT, "cores": cN if use_omp else c1,
                                    "kind": "oracle",
                                    "sample": f"{sN if use_omp else s1} annealing steps at full n={inst.n}, R={cfg.R} of {cfg.name}",
                                    "single_thread_value": v1, "all_core_value": vN, "all_core_threads": cN}
        print(json.dumps(line))
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
