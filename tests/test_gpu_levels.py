"""The internal levels of the tiled path (spray_set_levels): particle sets whose smoothing lengths do not fit the caller's grid
(BASELINE.json configs 2 and 4: cell edge 2 mean(h)) are served by the tiled kernels on grids of the
library's own, with the same bit-exact neighbour sets and the same sums as the oracle."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import compare_isolated, gpu_isolated, make_ctx, oracle_isolated, u32, u64, upload

pytestmark = pytest.mark.gpu


def get(name):
    if name == "cloud":
        return W.random_cloud(6000, seed=21, periodic=(1, 0, 1), hvar=2.5)
    return W.make(name)


@pytest.mark.parametrize("name", ["c2_tiny", "c4_tiny", "c2_mid", "c4_mid", "cloud"])
@pytest.mark.parametrize("kmode", [0, 1])
def test_levels_parity(name, kmode):
    w = get(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.set_levels(w.grid, W.level_edges(w.h))
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    st = sp.path_stats_full()
    # the cell table is the caller's grid's, whatever the levels do
    ref = O.build_cells(w.grid, w.x, w.y, w.z)
    t = sp.get_cell_table()
    for k in ("sorted_key", "perm", "cell_start", "cell_end"):
        assert np.array_equal(u32(t[k]), ref[k]), k
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt, ds, dx = O.neighbor_digest(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(u32(sp.neighbor_counts(sym)), cnt), (name, sym)
        gs, gx = sp.neighbor_digest(sym)
        assert np.array_equal(u64(gs), ds) and np.array_equal(u64(gx), dx), (name, sym)
        off, nbr = sp.neighbor_lists(sym)
        ooff, onbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(off.cpu().numpy().astype(np.uint64), ooff) and np.array_equal(u32(nbr), onbr)
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    g = gpu_isolated(sp, d, w, mu_in=mu_full, kmode=kmode)
    o = oracle_isolated(w, sym_mode=(kmode == 0), mu_full=mu_full)
    errs = compare_isolated(g, o)
    assert sp.check() == 0
    print(name, "kmode", kmode, st, {k: f"{v:.1e}" for k, v in errs.items()})
    if name in ("c2_mid", "c4_mid"):
        assert st["n_fast"] >= 0.7 * w.n, st           # most of the set is on the tiled path now


@pytest.mark.parametrize("mk", [lambda: (W.config1(24), 4, 0.99), lambda: (W.config3(20), 4, 0.99),
                                # 8^3 cells of 216: more tile entries than the context has room for -- the groups cut off at
                                # the capacity must be left to the general kernels whole
                                lambda: (W.config1(48), 8, 0.3)])
@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 1, 0)])
def test_tiles_in_several_parts(mk, periodic):
    """Cells that hold ~200 particles each: the candidates of any column of a 2 x 2 bundle (48 cells) are several times what
    a tile stages, so EVERY tile is a group of parts (tiles.cuh) -- same targets, disjoint candidate rows, lists per part,
    sums carried from part to part.  Before the parts existed none of these particles could be tiled (n_fast = 0)."""
    import dataclasses
    from workloads import Grid
    w0, nc, served = mk()
    ncell = (nc, nc, nc)
    w = dataclasses.replace(w0, grid=Grid(w0.grid.lo, w0.grid.hi, ncell, periodic, w0.grid.h_max))
    assert 2.0 * w.grid.h_max <= (w.grid.hi[0] - w.grid.lo[0]) / ncell[0] and w.n / nc ** 3 > 100
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    st = sp.path_stats_full()
    assert st["n_fast"] >= served * w.n and st["tiles"] >= 2 * (w.n // 256), st
    if served < 0.9:
        assert st["n_fast"] < w.n, st                       # the capacity did bind
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt, ds, dx = O.neighbor_digest(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(u32(sp.neighbor_counts(sym)), cnt), sym
        gs, gx = sp.neighbor_digest(sym)
        assert np.array_equal(u64(gs), ds) and np.array_equal(u64(gx), dx), sym
        off, nbr = sp.neighbor_lists(sym)
        ooff, onbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(off.cpu().numpy().astype(np.uint64), ooff) and np.array_equal(u32(nbr), onbr)
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    g = gpu_isolated(sp, d, w, mu_in=mu_full)
    o = oracle_isolated(w, mu_full=mu_full)
    errs = compare_isolated(g, o)
    g2 = gpu_isolated(sp, d, w, mu_in=mu_full)          # bitwise the same from run to run
    for k in g:
        assert np.array_equal(g[k], g2[k]), k
    assert sp.check() == 0
    print(st, {k: f"{v:.1e}" for k, v in errs.items()})
    # the other calls that run on the same lists (rows N1-N4), against the general kernels of a second context
    import torch
    s0 = make_ctx(w, path=0)
    s0.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    tp = 2.0 * np.pi
    kk, T = 1.0 + 0.5 * torch.sin(tp * d["x"]), 1.0 + 0.3 * torch.cos(tp * d["y"])      # smooth fields of order one
    mu, En, one = 0.3 + 0.1 * torch.sin(tp * d["z"]), T ** 4, torch.ones_like(T)
    ca, cb = sp.conduction(d["m"], d["rho_nom"], kk, T), s0.conduction(d["m"], d["rho_nom"], kk, T)
    ka, kb = sp.kgc_continuity(d["m"], d["rho_nom"], d["vx"], d["vy"], d["vz"]), s0.kgc_continuity(d["m"], d["rho_nom"], d["vx"], d["vy"], d["vz"])
    i = np.arange(8, dtype=np.int64)
    rays = torch.from_numpy(np.vstack([0.9 - 0.05 * W.u01(5, i, 0), W.u01(5, i, 1), W.u01(5, i, 2), -np.ones(8), 0.1 * (W.u01(5, i, 3) - 0.5),
                                       0.1 * (W.u01(5, i, 4) - 0.5), 1.0 + W.u01(5, i, 5)])).cuda()
    fq = 0.8 * torch.exp(-2.0 * d["x"])
    kib = 4.0 * (0.2 + fq * fq)
    ra, rb = sp.ray_deposit(d["m"], d["rho_nom"], fq, kib, rays, 0.01, 30), s0.ray_deposit(d["m"], d["rho_nom"], fq, kib, rays, 0.01, 30)
    ja = sp.rad_jacobi(d["m"], d["rho_nom"], mu, one, En, T.clone(), T, one, 1e-3, niter=3)
    jb = s0.rad_jacobi(d["m"], d["rho_nom"], mu, one, En, T.clone(), T, one, 1e-3, niter=3)

    def close(a, b, what):
        sc = float(b.abs().max()) + 1e-300
        assert float((a - b).abs().max()) <= 1e-10 * sc, (what, float((a - b).abs().max()), sc)
    close(ca, cb, "conduction")
    close(ka["drhodt"], kb["drhodt"], "kgc drhodt")
    close(ka["L"], kb["L"], "kgc L")
    close(ra["gradn"], rb["gradn"], "ray gradn")
    close(ra["edep"], rb["edep"], "ray edep")
    close(ja["E"], jb["E"], "rad E")


def test_levels_are_optional_and_removable():
    w = W.make("c4_tiny")
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    r0 = sp.density(d["m"]).clone()
    f0 = sp.path_stats_full()["n_fast"]
    sp.set_levels(w.grid, W.level_edges(w.h))
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    r1 = sp.density(d["m"]).clone()
    f1 = sp.path_stats_full()["n_fast"]
    sp.set_levels(w.grid, [])
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    r2 = sp.density(d["m"])
    assert f1 > f0 and sp.path_stats_full()["n_fast"] == f0
    S = O.density(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)["S_rho"]
    assert np.all(np.abs((r1 - r0).cpu().numpy()) <= 1e-11 * S) and bool((r2 == r0).all())
