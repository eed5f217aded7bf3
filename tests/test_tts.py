"""The time-to-solution statistic and the batch harness around fem_anneal."""
import math

import numpy as np
import pytest

from paper_2412_09285_b200 import tts, workloads as wl


def test_tts99_formula_and_its_special_cases():
    assert tts.tts99(3.0, 0.99) == 3.0 and tts.tts99(3.0, 1.0) == 3.0        # P_S >= 0.99: one trial is enough
    assert tts.tts99(3.0, 0.0) == math.inf
    assert abs(tts.tts99(1.0, 0.5) - math.log(0.01) / math.log(0.5)) < 1e-15  # 6.64 trials
    assert abs(tts.tts99(2.0, 0.9) - 4.0) < 1e-12                             # log(0.01) / log(0.1) = 2 trials
    # the number of independent trials k with 1 - (1 - p)^k = 0.99
    for p in (0.05, 0.3, 0.7):
        k = tts.tts99(1.0, p)
        assert abs(1.0 - (1.0 - p) ** k - 0.99) < 1e-12
    with pytest.raises(ValueError):
        tts.tts99(1.0, 1.5)


def test_success_probability_counts_trials_that_reach_the_target():
    best = np.array([-10.0, -12.0, -12.0, -11.0])
    assert tts.success_probability(best, -12.0) == 0.5
    assert tts.success_probability(best, -13.0) == 0.0
    assert tts.success_probability(best, -10.0) == 1.0


@pytest.mark.gpu
def test_batch_harness_on_a_small_graph_with_known_optimum():
    """A graph small enough to enumerate (n = 16): the target is the brute-force optimum from the oracle's definition of
    the energy; every batch of 8 replicas finds it, so P_S = 1 and TTS = T_com."""
    from oracle import fem_oracle as fo
    from paper_2412_09285_b200 import fem
    inst = wl.erdos_renyi_maxcut(16, 0.4, 5, pm1=True)
    pb = fo.Problem(kind=inst.kind, n=inst.n, q=2, row_ptr=inst.row_ptr, col_idx=inst.col_idx, weight=inst.weight)
    cfgs = ((np.arange(1 << 15)[:, None] >> np.arange(16)[None, :]) & 1).astype(np.int32)   # node 15 fixed to 0 (symmetry)
    e_opt = float(fo.energies(pb, cfgs)[1].min())
    sch = fem.Schedule(beta=fem.linear_temperature_schedule(1.0, 0.01, 300))
    out = tts.run_batches(inst, sch, 8, 6, target=e_opt)
    assert out["best_energy"] == e_opt and out["p_s"] == 1.0 and out["tts_ms"] == out["t_com_ms"] > 0
    # without a known target the best value found is the target, and at least one trial reaches it
    out2 = tts.run_batches(wl.preferential_attachment(300, 3, 7, pm1=True), sch, 16, 5)
    assert out2["target_is_best_found"] and out2["p_s"] >= 0.2 and math.isfinite(out2["tts_ms"])
