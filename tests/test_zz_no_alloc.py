"""fem_cut_static (include/fem.h): the cut values of Eq.6 computed with the partial sums in a static
__device__ array instead of the caller's workspace -- an entry point that allocates nothing, for callers that cannot call
cudaMalloc.  Checked against the existing path (fem_energy_of on a handle: energy_int = -cut, integer work, so bit-exact) and
against the plain definition, on two calls in a row that share the scratch array (the second with more configurations and
another graph, so that it finds the first call's partials in the array).

Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

from paper_2412_09285_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fem():
    from paper_2412_09285_b200 import fem as femlib
    return femlib


def plain_cut(inst, cfg):
    """Eq.6 written out: every edge once, W_ij where the end points differ."""
    rows = np.repeat(np.arange(inst.n), np.diff(inst.row_ptr))
    keep = inst.col_idx > rows
    i, j = rows[keep], inst.col_idx[keep]
    w = np.ones(keep.sum(), dtype=np.int64) if inst.weight is None else np.rint(inst.weight[keep]).astype(np.int64)
    return ((cfg[:, i] != cfg[:, j]) * w[None, :]).sum(axis=1)


def on_device(inst, cfg, torch):
    dev = "cuda:0"
    row_ptr = torch.from_numpy(inst.row_ptr.astype(np.int32)).to(dev)
    col = torch.from_numpy(inst.col_idx.astype(np.int32)).to(dev)
    w = None if inst.weight is None else torch.from_numpy(inst.weight.astype(np.float32)).to(dev)
    sigma = torch.from_numpy(np.ascontiguousarray(cfg.T.astype(np.int8))).to(dev)       # [n][count], configuration innermost
    cut = torch.full((cfg.shape[0],), -12345, dtype=torch.int64, device=dev)
    return row_ptr, col, w, sigma, cut


def existing_path(fem, inst, cfg):
    eng = fem.Fem(inst, cfg.shape[0])
    e_int, _, _ = eng.energy_of(cfg)
    eng.close()
    return -e_int


def test_two_calls_in_a_row_match_the_existing_path(fem):
    import torch
    rng = np.random.default_rng(5)
    # call 1: weighted +-1 scale-free graph (a hub row), 70 configurations (two warps and a ragged tail)
    a = wl.preferential_attachment(3000, 3, 77, pm1=True)
    cfg_a = rng.integers(0, 2, (70, a.n)).astype(np.int32)
    # call 2: unit-weight random graph of another size, 200 configurations: more partials per chunk than call 1 wrote
    b = wl.erdos_renyi_maxcut(800, 0.06, 1000)
    cfg_b = rng.integers(0, 2, (200, b.n)).astype(np.int32)
    dev_a, dev_b = on_device(a, cfg_a, torch), on_device(b, cfg_b, torch)
    want_a, want_b = existing_path(fem, a, cfg_a), existing_path(fem, b, cfg_b)
    torch.cuda.synchronize()

    fem.cut_static(*dev_a)                       # first call on this device: looks up the scratch array's address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    fem.cut_static(*dev_b)                       # same stream, back to back with ...
    fem.cut_static(*dev_a)                       # ... a repeat of call 1 over call 2's partials
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # nothing was allocated on the device
    got_a, got_b = dev_a[4].cpu().numpy(), dev_b[4].cpu().numpy()
    assert np.array_equal(got_a, want_a) and np.array_equal(got_b, want_b)      # the existing path, bit for bit
    assert np.array_equal(got_a, plain_cut(a, cfg_a)) and np.array_equal(got_b, plain_cut(b, cfg_b))
    assert got_a.min() != got_a.max()            # (not a constant: the configurations differ)


def test_maximum_count_and_rejection_beyond_it(fem):
    import torch
    rng = np.random.default_rng(6)
    inst = wl.random_regular(512, 3, 9, wl.MAXCUT, pm1=True)
    cfg = rng.integers(0, 2, (fem.CUT_STATIC_MAX_COUNT, inst.n)).astype(np.int32)
    dev = on_device(inst, cfg, torch)
    fem.cut_static(*dev)                         # the largest batch the scratch array holds
    torch.cuda.synchronize()
    assert np.array_equal(dev[4].cpu().numpy(), plain_cut(inst, cfg))
    too_many = np.concatenate([cfg, cfg[:1]])
    dev2 = on_device(inst, too_many, torch)
    with pytest.raises(fem.FemError) as err:
        fem.cut_static(*dev2)
    assert err.value.status == fem.FEM_EINVAL and "FEM_CUT_STATIC_MAX_COUNT" in str(err.value)
    torch.cuda.synchronize()
    assert (dev2[4] == -12345).all().item()      # a rejected call launches nothing
