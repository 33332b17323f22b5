"""mps_cell_start_noalloc (the one entry point that allocates nothing: its scratch is a file-scope device
array) against the existing path, mps_bin + mps_get_cell_start, bit for bit -- the bar the bin parity tests
use for index work.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2105_01677_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2105_01677_b200 import binding
    return binding


def _existing_path(B, s, **over):
    """keys and cell-start table of the library's own bin (ctx buffers allocated at mps_init)"""
    g = B.Mps(s, **over)
    g.bin()
    key = g.get_dev("key", B.ORDER_SORTED)          # int32 words on the device, any order will do
    cs = g.cell_start()
    ncells = g.grid()[3]
    g.close()
    return key, cs, ncells


def test_no_alloc_cell_start_equals_the_bin_path_on_two_calls_in_a_row(B):
    import torch
    # two different scenes and grids, so that the second call finds the first call's counts in the shared array
    a = scenes.make_scene(1, shuffle=True)
    a.x[5] = 10.0                                   # two ghosts: the last counter is in use
    a.z[40] = -1.0
    b = scenes.small_tank(shuffle=True)
    cases = [_existing_path(B, a, cell_div=2), _existing_path(B, b), _existing_path(B, a, cell_div=2)]
    assert cases[0][2] != cases[1][2] and cases[0][2] > 2048   # several scan tiles and a ragged tail
    for key, cs, ncells in cases:                   # calls back to back on one stream
        out = torch.full((ncells + 1,), -1, dtype=torch.int32, device=key.device)
        B.cell_start_noalloc(key, ncells, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.array_equal(got, cs.astype(got.dtype))
        assert got[0] == 0 and got[-1] <= key.numel()
    # and twice on the same input without anything in between
    key, cs, ncells = cases[1]
    o1 = torch.empty(ncells + 1, dtype=torch.int32, device=key.device)
    o2 = torch.empty(ncells + 1, dtype=torch.int32, device=key.device)
    B.cell_start_noalloc(key, ncells, o1)
    B.cell_start_noalloc(key, ncells, o2)
    torch.cuda.synchronize()
    assert np.array_equal(o1.cpu().numpy(), cs.astype(np.int32)) and torch.equal(o1, o2)


def test_no_alloc_rejects_sizes_beyond_its_scratch(B):
    import torch
    lim = B.cell_start_noalloc_max_cells()
    assert lim == 262144
    key = torch.zeros(8, dtype=torch.int32, device="cuda:0")
    out = torch.empty(16, dtype=torch.int32, device="cuda:0")
    with pytest.raises(B.MpsError) as ei:
        B.cell_start_noalloc(key, lim + 1, out)
    assert ei.value.code == B.MPS_ERR_ARG and "exceeds the fixed scratch" in str(ei.value)
    with pytest.raises(B.MpsError):
        B.cell_start_noalloc(key, 0, out)
    # the limit itself is served (all keys in cell 3: cell_start is 0 up to 3, then 8)
    key.fill_(3)
    big = torch.empty(lim + 1, dtype=torch.int32, device="cuda:0")
    B.cell_start_noalloc(key, lim, big)
    torch.cuda.synchronize()
    h = big.cpu().numpy()
    assert (h[:4] == 0).all() and (h[4:] == 8).all()
