"""GPU test of ibm_sort_cells_noalloc, the entry point that allocates nothing (scratch in a file-scope device array).

Collected last on purpose (file name): the suite runs with pytest -x.  The existing path is the binning of the
time step: lbm_ibm_step sorts the markers by owning cell (single-block sort up to 32,768 markers, the three-kernel
passes above) and ibm_read_markers reports the cells and the permutation.  Integer work: the comparison is bit-exact
(R20: the stable permutation is unique)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available()
    from paper_1904_02108_b200 import api as _api
    return _api


def _cells_and_perm_of_the_step(api, wl, steps):
    """cell key per marker (caller order) and sort permutation of the last step, from the existing path"""
    import torch
    sim = api.from_workload(wl, stream=torch.cuda.Stream())
    sim.step(steps, wl.mdf_iters)
    sim.sync()
    mk = sim.read_markers(pos=False, force=False)
    sim.close()
    return mk["cell"].astype(np.int32), mk["perm"].astype(np.int32), wl.nx * wl.ny * wl.nz


def test_noalloc_sort_matches_the_binning_of_the_step_on_two_calls_in_a_row(api):
    import torch
    from paper_1904_02108_b200 import workloads
    # 147,456 markers (the step sorts them with the three-kernel passes), then 15,360 (single-block sort in the step):
    # the second call finds the first call's contents in the shared scratch array
    cases = [_cells_and_perm_of_the_step(api, workloads.w4(0, 8, n=128), 3),
             _cells_and_perm_of_the_step(api, workloads.get("W3"), 2)]
    assert cases[0][0].size > 32768 >= cases[1][0].size
    stream = torch.cuda.Stream()
    dev = [(torch.from_numpy(c).cuda(), torch.empty(c.size, dtype=torch.int32, device="cuda"),
            torch.empty(c.size, dtype=torch.int32, device="cuda")) for c, _, _ in cases]
    again = (torch.empty_like(dev[0][1]), torch.empty_like(dev[0][2]))
    # warm-up call (the first launch of a kernel loads its code), then nothing may change the free device memory
    api.sort_cells_noalloc(dev[1][0], cases[1][2], dev[1][1], dev[1][2], stream)
    stream.synchronize()
    dev[1][1].fill_(-1); dev[1][2].fill_(-1)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # two calls in a row on one stream, no synchronisation between them, then the first once more
    api.sort_cells_noalloc(dev[0][0], cases[0][2], dev[0][1], dev[0][2], stream)
    api.sort_cells_noalloc(dev[1][0], cases[1][2], dev[1][1], dev[1][2], stream)
    api.sort_cells_noalloc(dev[0][0], cases[0][2], again[0], again[1], stream)
    stream.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the free device memory"
    for (cell, perm, _), (d_cell, d_sorted, d_perm) in zip(cases, dev):
        got_perm, got_sorted = d_perm.cpu().numpy(), d_sorted.cpu().numpy()
        assert np.array_equal(got_perm, perm)                     # the existing path's permutation, bit for bit
        assert np.array_equal(got_sorted, cell[perm])
        assert np.array_equal(d_cell.cpu().numpy(), cell)         # the input is not modified
        assert np.array_equal(got_perm, np.argsort(cell, kind="stable").astype(np.int32))
    assert np.array_equal(again[1].cpu().numpy(), cases[0][1])
    assert np.array_equal(again[0].cpu().numpy(), cases[0][0][cases[0][1]])


def test_noalloc_sort_limits_and_errors(api):
    import torch
    big = torch.zeros(api.NOALLOC_MAX_MARKERS + 1, dtype=torch.int32, device="cuda")
    out = (torch.empty_like(big), torch.empty_like(big))
    with pytest.raises(api.LbmError) as e:
        api.sort_cells_noalloc(big, 1 << 20, out[0], out[1])
    assert e.value.code == -4 and str(api.NOALLOC_MAX_MARKERS) in str(e.value)      # LBM_ERANGE, names the limit
    # exactly the maximum, keys spread over 2^21 cells (three passes), against numpy
    rng = np.random.default_rng(3)
    keys = rng.integers(0, 1 << 21, api.NOALLOC_MAX_MARKERS, dtype=np.int32)
    d = torch.from_numpy(keys).cuda()
    api.sort_cells_noalloc(d, 1 << 21, out[0][:-1], out[1][:-1])
    torch.cuda.synchronize()
    want = np.argsort(keys, kind="stable").astype(np.int32)
    assert np.array_equal(out[1][:-1].cpu().numpy(), want)
    assert np.array_equal(out[0][:-1].cpu().numpy(), keys[want])
    # n = 0 is a no-op; host pointers and an output that aliases the input are rejected
    api.sort_cells_noalloc(d[:0], 1 << 21, out[0][:0], out[1][:0])
    with pytest.raises(api.LbmError):
        api.sort_cells_noalloc(torch.zeros(8, dtype=torch.int32), 64, out[0], out[1])
    with pytest.raises(api.LbmError):
        api.sort_cells_noalloc(d, 1 << 21, d, out[1])
