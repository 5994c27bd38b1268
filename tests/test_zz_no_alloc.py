"""mwf_monopoles_static: the monopole pass for callers that cannot allocate device memory.

Who needs it: code that runs inside somebody else's memory budget -- a plugin under an application whose pool owns the
GPU, a routine on a latency-bound path where cudaMalloc / cudaFree would stall the device, a job on a nearly full GPU --
and therefore cannot create an mwf_ctx (a ctx needs an arena that someone has to allocate).  The entry point keeps its
working memory in a fixed array inside the library image instead (limit: MWF_STATIC_MAX_CELL = 131072 tree cells), so the
things to check are (1) that it gives the records the ctx path gives, (2) that a call is not disturbed by what the
previous call left in the shared array -- hence calls in a row on trees of different sizes, without a synchronisation
in between --, (3) that it really takes no device memory, and (4) that a tree over the limit is refused in words.

The file is named test_zz_* so that pytest collects it last: under `pytest -x` a failure here hides no other test.  It
must pass alone in a fresh process (the first call does the per-device address look-up) and after the whole suite."""
import numpy as np
import pytest

import oracle
from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import CONFIGS, make_workload

pytestmark = pytest.mark.gpu


def ctx_monopoles(w):
    """The existing path: upload into a ctx, mwf_refresh_monopoles, read the records back."""
    f = binding.MultiWalkForce.for_workload(w)
    f.upload_workload(w)
    f.refresh_monopoles()
    got = f.get_monopoles(w.n_cell)
    f.close()
    return got


def assert_same_monopoles(got, ref, side, label):
    """The bounds tests/test_gpu_parity.py::test_monopole_refresh holds the ctx path to (reading S11 of DESIGN.md)."""
    got, ref = got.astype(np.float64), ref.astype(np.float64)
    assert np.all(np.isfinite(got)), label
    assert np.all(np.abs(got[:, 3] - ref[:, 3]) <= 1e-6 * ref[:, 3]), label
    dx = np.linalg.norm(got[:, :3] - ref[:, :3], axis=1)
    assert np.all(dx <= 2.0 ** -22 * np.maximum(np.linalg.norm(ref[:, :3], axis=1), side)), label


def test_static_scratch_monopoles_match_the_ctx_path():
    import torch
    dev = torch.device("cuda:0")
    big = make_workload(CONFIGS[2], 100000)        # disk + halo, 24 260 cells
    small = make_workload(CONFIGS[3], 30000)       # clumpy box, a smaller tree: it leaves part of the last call's scratch untouched
    assert small.n_cell < big.n_cell <= binding.STATIC_MAX_CELL
    ref = {id(w): ctx_monopoles(w) for w in (big, small)}

    def on_device(w):
        return (torch.from_numpy(np.ascontiguousarray(w.cells)).to(dev), torch.from_numpy(np.ascontiguousarray(w.posm)).to(dev),
                torch.full((w.n_cell, 4), float("nan"), dtype=torch.float32, device=dev))

    runs = [(big, on_device(big)), (small, on_device(small)), (big, on_device(big))]
    binding.monopoles_static(*runs[0][1])          # may be the first call in this process: it does the address look-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _, bufs in runs[1:]:                       # two more calls in a row on one stream, nothing between them
        binding.monopoles_static(*bufs)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the calls took device memory"
    for k, (w, (_, _, spj)) in enumerate(runs):
        got = spj.cpu().numpy()
        assert_same_monopoles(got, ref[id(w)], w.geom[:, 3], "call %d against the ctx path" % k)
        mom = oracle.monopoles(w.cells, w.posm)    # and against the definition
        assert_same_monopoles(got, mom, w.geom[:, 3], "call %d against the oracle" % k)
    assert np.array_equal(runs[0][1][2].cpu().numpy(), runs[2][1][2].cpu().numpy())   # same inputs, same bits, whatever ran in between


def test_static_scratch_refuses_a_tree_over_its_limit():
    import torch
    dev = torch.device("cuda:0")
    n_cell = binding.STATIC_MAX_CELL + 1
    cells = torch.zeros((n_cell, 4), dtype=torch.int32, device=dev)
    ptcl = torch.zeros((8, 4), dtype=torch.float32, device=dev)
    spj = torch.full((n_cell, 4), 7.0, dtype=torch.float32, device=dev)
    with pytest.raises(binding.MwfError) as err:
        binding.monopoles_static(cells, ptcl, spj)
    assert err.value.code == binding.ENOMEM
    assert str(binding.STATIC_MAX_CELL) in str(err.value) and "MWF_STATIC_MAX_CELL" in str(err.value)
    torch.cuda.synchronize()
    assert bool((spj == 7.0).all())                # nothing was launched
    with pytest.raises(binding.MwfError) as err:   # a misaligned record array is refused as well
        binding.monopoles_static(cells[:16], ptcl.reshape(-1)[1:29].reshape(7, 4), spj[:16])
    assert err.value.code == binding.EINVAL
