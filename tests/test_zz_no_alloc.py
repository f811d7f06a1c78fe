"""spray_cell_list_static -- the entry point that allocates nothing (its scratch is a static device array) -- against the
existing path spray_build_cells + spray_get_cell_table: keys, permutation and cell table are integer work, so the bar is
bit-exact equality (the bar of every cell-table test here).  Two calls in a row on different inputs, because every call
shares the array and finds the previous call's contents in it.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import workloads as W
from workloads import Grid

pytestmark = pytest.mark.gpu


def _cloud(n, seed, grid):
    """seeded positions: most inside the box, a few outside its open faces (clamped into the boundary cells)"""
    i = np.arange(n, dtype=np.int64)
    lo, hi = np.array(grid.lo, dtype=np.float64), np.array(grid.hi, dtype=np.float64)
    p = []
    for d in range(3):
        u = W.u01(seed, i, d)
        if not grid.periodic[d]:
            u = u * 1.04 - 0.02
        p.append(lo[d] + u * (hi[d] - lo[d]))
    return p


def _existing(grid, xyz):
    import torch
    import paper_2604_20124_b200 as P
    n = xyz[0].numel()
    sp = P.Spray(max(n, 1), grid.ncell_total)
    sp.set_path(0)                                    # cell list only: no tiles or lists needed for this comparison
    h = torch.full((n,), 0.5 * grid.h_max, dtype=torch.float64, device="cuda")
    sp.build_cells(grid, P.KERNEL_CUBIC_SPLINE, xyz[0], xyz[1], xyz[2], h)
    t = sp.get_cell_table()
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in t.items()}


# (n, grid): one, two and three radix passes, ragged sizes around the 4096-key sort tile, the maximum size, periodic and open
CASES = [
    (4096 + 37, Grid((0, 0, 0), (1, 1, 1), (6, 6, 6), (1, 1, 1), 0.05)),
    (200_001, Grid((-1, 0, 2), (1, 1, 2.5), (40, 41, 39), (0, 1, 0), 0.01)),
    (262_144, Grid((0, 0, 0), (1, 2, 1), (70, 140, 70), (0, 0, 0), 0.005)),
    (1, Grid((0, 0, 0), (1, 1, 1), (1, 1, 1), (0, 0, 0), 0.3)),
]


def test_static_matches_existing_path_two_calls_in_a_row():
    import torch
    import paper_2604_20124_b200 as P
    inputs = []
    for k, (n, grid) in enumerate(CASES):
        xyz = [torch.from_numpy(a).cuda() for a in _cloud(n, 2604201290 + k, grid)]
        inputs.append((grid, xyz, _existing(grid, xyz)))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    # back to back on one stream, each call finding the previous call's keys, indices and histograms in the scratch;
    # then the whole sequence once more in reverse order
    results = []
    order = list(range(len(inputs))) + list(reversed(range(len(inputs))))
    for k in order:
        grid, xyz, _ = inputs[k]
        results.append((k, P.cell_list_static(grid, xyz[0], xyz[1], xyz[2], dev_status=status)))
    torch.cuda.synchronize()
    for k, got in results:
        ref = inputs[k][2]
        for name in ("sorted_key", "perm", "cell_start", "cell_end"):
            assert np.array_equal(got[name].cpu().numpy(), ref[name]), (k, name)
    assert int(status.item()) == 0


def test_static_same_input_twice_and_status():
    import torch
    import paper_2604_20124_b200 as P
    grid = Grid((0, 0, 0), (1, 1, 1), (17, 16, 15), (1, 1, 1), 0.02)
    xyz = [torch.from_numpy(a).cuda() for a in _cloud(50_000, 2604201299, grid)]
    ref = _existing(grid, xyz)
    a = P.cell_list_static(grid, xyz[0], xyz[1], xyz[2])
    b = P.cell_list_static(grid, xyz[0], xyz[1], xyz[2])
    torch.cuda.synchronize()
    for name in ref:
        assert np.array_equal(a[name].cpu().numpy(), ref[name]), name
        assert np.array_equal(b[name].cpu().numpy(), ref[name]), name
    # a position outside a periodic box is reported in this call's status word and is gone in the next call's
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    bad = xyz[0].clone()
    bad[123] = 1.5
    P.cell_list_static(grid, bad, xyz[1], xyz[2], dev_status=status)
    assert int(status.item()) == P.DEV_OUTSIDE_BOX
    P.cell_list_static(grid, xyz[0], xyz[1], xyz[2], dev_status=status)
    assert int(status.item()) == 0


def test_static_limits_and_empty():
    import torch
    import paper_2604_20124_b200 as P
    grid = Grid((0, 0, 0), (1, 1, 1), (4, 4, 4), (0, 0, 0), 0.1)
    big = torch.zeros(P.STATIC_NMAX + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(P.SprayError, match=r"\(-4\).*SPRAY_STATIC_NMAX"):
        P.cell_list_static(grid, big, big, big)
    huge = Grid((0, 0, 0), (1, 1, 1), (512, 512, 65), (0, 0, 0), 0.1)
    z = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(P.SprayError, match=r"\(-3\)"):
        P.cell_list_static(huge, z, z, z)
    e = torch.zeros(0, dtype=torch.float64, device="cuda")
    t = P.cell_list_static(grid, e, e, e)
    torch.cuda.synchronize()
    assert not t["cell_start"].any() and not t["cell_end"].any()
