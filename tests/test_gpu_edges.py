"""GPU edge cases through the C-ABI: empty and one-particle inputs, ragged sizes around the sort tile, one-cell
grids, everything in one cell, error codes, sticky device status."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from workloads import Grid
from parity_util import compare_isolated, gpu_isolated, make_ctx, oracle_isolated, u32, upload

pytestmark = pytest.mark.gpu
PATHS = [0, 1]          # 0 = general kernels only, 1 = tiled kernels + general kernels for what they decline


def test_error_codes():
    import torch
    import paper_2604_20124_b200 as P
    sp = P.Spray(100, 64)
    z = torch.zeros(10, dtype=torch.float64, device="cuda")
    with pytest.raises(P.SprayError, match=r"\(-2\)"):          # NOT_BUILT
        sp.density(z)
    g = Grid((0, 0, 0), (1, 1, 1), (4, 4, 4), (1, 1, 1), 0.2)    # L < 6 h_max
    with pytest.raises(P.SprayError, match=r"\(-3\)"):
        sp.build_cells(g, 0, z, z, z, z)
    g = Grid((0, 0, 0), (1, 1, 1), (5, 5, 5), (0, 0, 0), 0.1)    # 125 cells > ncell_max
    with pytest.raises(P.SprayError, match=r"\(-3\)"):
        sp.build_cells(g, 0, z, z, z, z)
    g = Grid((0, 0, 0), (1, 1, 1), (4, 4, 4), (0, 0, 0), 0.1)
    big = torch.zeros(101, dtype=torch.float64, device="cuda")
    with pytest.raises(P.SprayError, match=r"\(-4\)"):          # CAPACITY
        sp.build_cells(g, 0, big, big, big, big)
    with pytest.raises(P.SprayError, match=r"\(-1\)"):
        sp.build_cells(g, 7, z, z, z, z)
    with pytest.raises(P.SprayError):
        sp.build_cells(g, 0, z.cpu(), z, z, z)                   # host tensor rejected by the binding
    # after failures the context is still usable
    h = torch.full((10,), 0.1, dtype=torch.float64, device="cuda")
    x = torch.linspace(0.05, 0.95, 10, dtype=torch.float64, device="cuda")
    sp.build_cells(g, 0, x, x, x, h)
    assert sp.density(h).shape[0] == 10
    with pytest.raises(P.SprayError, match=r"\(-1\)"):          # INVALID_ARG: NULL input of the fused call
        sp.hydro_rhs_limiter(h, h, h, h, h, h, h, h, None, h)
    assert sp.check() == 0


def test_sticky_device_status():
    import torch
    import paper_2604_20124_b200 as P
    sp = P.Spray(16, 64)
    g = Grid((0, 0, 0), (1, 1, 1), (4, 4, 4), (1, 1, 1), 0.1)
    x = torch.tensor([0.1, 0.5, 1.5], dtype=torch.float64, device="cuda")     # 1.5 outside the periodic box
    h = torch.tensor([0.1, 0.1, 0.3], dtype=torch.float64, device="cuda")     # 0.3 > declared h_max
    sp.build_cells(g, 1, x, x, x, h)
    st = sp.check()
    assert st & P.DEV_OUTSIDE_BOX and st & P.DEV_H_EXCEEDS_HMAX
    assert sp.check() == 0      # cleared


@pytest.mark.parametrize("path", PATHS)
def test_empty_and_single_particle(path):
    import torch
    import paper_2604_20124_b200 as P
    sp = P.Spray(8, 27)
    sp.set_path(path)
    g = Grid((0, 0, 0), (1, 1, 1), (3, 3, 3), (1, 1, 1), 0.1)
    e = torch.zeros(0, dtype=torch.float64, device="cuda")
    sp.build_cells(g, 0, e, e, e, e)
    assert sp.density(e).numel() == 0
    assert len(sp.hydro_rhs(e, e, e, e, e, e, e, e)) == 5
    assert sp.fld_apply(e, e, e, e)["y"].numel() == 0
    assert sp.hydro_rhs_limiter(e, e, e, e, e, e, e, e, e, e)[1].numel() == 0
    t = sp.get_cell_table()
    assert (u32(t["cell_start"]) == 0).all() and (u32(t["cell_end"]) == 0).all()
    one = torch.tensor([0.4], dtype=torch.float64, device="cuda")
    h = torch.tensor([0.1], dtype=torch.float64, device="cuda")
    m = torch.tensor([2.0], dtype=torch.float64, device="cuda")
    for k in (0, 1):
        sp.build_cells(g, k, one, one, one, h)
        rho, nn = sp.density(m, want_nnbr=True)
        assert float(rho[0]) == pytest.approx(2.0 * O.W(k, 0.0, 0.1), rel=1e-14)   # self term only (A11)
        assert int(nn[0]) == 0
        hy = sp.hydro_rhs(m, m, m, m, m, m, m, m)
        assert all(float(t[0]) == 0.0 for t in hy)
        fl = sp.fld_apply(m, m, m, m)
        assert float(fl["y"][0]) == 0.0 and float(fl["diag"][0]) == 0.0
        assert float(fl["mu"][0]) == pytest.approx(1.0 / 3.0 / 4.0, rel=1e-15)      # R = 0: lambda = 1/3, mu = c/(3 rho kappa)
        fy, fmu, _ = sp.hydro_rhs_limiter(m, m, m, m, m, m, m, m, m, m)
        assert all(float(t[0]) == 0.0 for t in fy) and float(fmu[0]) == float(fl["mu"][0])
        # next rows on one particle: no neighbour, so no conduction, L = I (A28) and no density change
        assert float(sp.conduction(m, m, m, m)[0]) == 0.0
        kg = sp.kgc_continuity(m, m, m, m, m)
        assert float(kg["drhodt"][0]) == 0.0 and float(kg["drhodt_raw"][0]) == 0.0
        assert kg["L"].flatten().tolist() == [1.0, 0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0]
    # ... and on the empty set
    sp.build_cells(g, 0, e, e, e, e)
    assert sp.conduction(e, e, e, e).numel() == 0
    assert sp.kgc_continuity(e, e, e, e, e)["drhodt"].numel() == 0
    assert sp.rad_jacobi(e, e, e, e, e, e, e, e, 0.1, niter=2)["E"].numel() == 0
    assert sp.check() == 0


def _cloud(n, **kw):
    return W.random_cloud(n, **kw)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("n", [2, 31, 33, 4095, 4096, 4097, 12345])
def test_ragged_sizes(path, n):
    """sizes around the warp, the radix-sort tile (4096) and the CTA tile; open box so tiny n is legal"""
    w = _cloud(n, seed=100 + n, periodic=(0, 0, 0), hvar=1.7)
    d = upload(w)
    sp = make_ctx(w, path, slack=5)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    ref = O.build_cells(w.grid, w.x, w.y, w.z)
    t = sp.get_cell_table()
    for k in ("sorted_key", "perm", "cell_start", "cell_end"):
        assert np.array_equal(u32(t[k]), ref[k]), k
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    compare_isolated(gpu_isolated(sp, d, w, mu_in=mu_full), oracle_isolated(w, mu_full=mu_full))
    assert sp.check() == 0


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("ncell,periodic", [((1, 1, 1), (0, 0, 0)), ((1, 1, 1), (1, 1, 1)), ((2, 1, 3), (1, 1, 1)),
                                            ((40, 1, 1), (0, 1, 0)), ((3, 3, 3), (1, 1, 1))])
def test_degenerate_grids(path, ncell, periodic):
    """one-cell grids, grids with fewer cells than the search stencil, very fine grids in one dimension"""
    w = _cloud(3000, seed=77, periodic=periodic, hvar=1.5, ncell=ncell)
    d = upload(w)
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt = u32(sp.neighbor_counts(sym))
        assert np.array_equal(cnt, O.neighbor_counts(w.grid, w.x, w.y, w.z, w.h, mode))
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    compare_isolated(gpu_isolated(sp, d, w, mu_in=mu_full), oracle_isolated(w, mu_full=mu_full))
    assert sp.check() == 0


@pytest.mark.parametrize("path", PATHS)
def test_all_particles_in_one_cell_and_coincident(path):
    """maximum cell occupancy + coincident distinct particles (r = 0: W(0) to density, nothing to gradients, A11)"""
    import copy
    w = _cloud(600, seed=5, periodic=(0, 0, 0), hvar=1.2, box=(0.05, 0.05, 0.05))
    w = copy.copy(w)
    w.grid = Grid((0, 0, 0), (1, 1, 1), (4, 4, 4), (0, 0, 0), w.grid.h_max)
    for f in ("x", "y", "z"):
        a = getattr(w, f).copy(); a[1] = a[0]; a[7] = a[3]; setattr(w, f, a)
    d = upload(w)
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    compare_isolated(gpu_isolated(sp, d, w, mu_in=mu_full), oracle_isolated(w, mu_full=mu_full))
    # row N3 with coincident particles: pairs at r = 0 add nothing to the moment sums on either side
    o = O.kgc_continuity(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.vx, w.vy, w.vz)
    r = sp.kgc_continuity(d["m"], d["rho_nom"], d["vx"], d["vy"], d["vz"])
    lo = np.linalg.norm(o["L"].reshape(-1, 9), axis=1)
    scale = w.rho_nom * lo * np.linalg.norm(o["S_N"].reshape(-1, 9), axis=1) * (1 + lo * np.linalg.norm(o["S_M"].reshape(-1, 9), axis=1))
    assert np.all(np.abs(r["drhodt"].cpu().numpy() - o["drhodt"]) <= 1e-11 * scale)
    assert sp.check() == 0


@pytest.mark.parametrize("path", PATHS)
def test_context_reuse_across_builds(path):
    """one ctx, several build_cells with different n / grids / kernels (scratch is sized for n_max)"""
    from paper_2604_20124_b200 import Spray
    sp = Spray(20000, 30000)
    sp.set_path(path)
    for name in ("c4_tiny", "c1_tiny", "c2_mid", "c3_tiny"):
        w = W.make(name)
        d = upload(w)
        sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
        rho = sp.density(d["m"]).cpu().numpy()
        o = O.density(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)
        assert np.abs(rho - o["rho"]).max() <= 1e-11 * o["S_rho"].max()
    assert sp.check() == 0


@pytest.mark.parametrize("name", ["hjit_w", "hjit_c"])
@pytest.mark.parametrize("kmode", [0, 1])
def test_every_tile_has_variable_h(name, kmode):
    """h jittered +-5 % on a grid with edge >= 2 max(h): the tiled path takes every particle, and every tile runs the
    VARIABLE-h pair bodies (clamped shapes, Fbar from the (1/h, Fn) record, N_gather a proper subset of N_sym).  The
    path statistics prove which kernels ran; both FLD kernel modes; neighbour sets and all sums against the oracle."""
    w = W.make(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    st = sp.path_stats_full()
    assert st["n_fast"] == w.n, st
    assert st["nonuniform_units"] > 0 and st["nonuniform_units"] >= st["tiles"], st
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt, ds, dx = O.neighbor_digest(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(u32(sp.neighbor_counts(sym)), cnt)
        gs, gx = sp.neighbor_digest(sym)
        assert np.array_equal(gs.cpu().numpy().view(np.uint64), ds) and np.array_equal(gx.cpu().numpy().view(np.uint64), dx)
    cg = O.neighbor_counts(w.grid, w.x, w.y, w.z, w.h, O.GATHER)
    cs = O.neighbor_counts(w.grid, w.x, w.y, w.z, w.h, O.SYM)
    assert (cs > cg).any()                         # the two set kinds differ: the clamps matter
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    g = gpu_isolated(sp, d, w, mu_in=mu_full, kmode=kmode)
    o = oracle_isolated(w, sym_mode=(kmode == 0), mu_full=mu_full)
    errs = compare_isolated(g, o)
    assert sp.check() == 0
    print(name, "kmode", kmode, st, {k: f"{v:.1e}" for k, v in errs.items()})


def test_particles_far_outside_an_open_box():
    """spray.h allows positions outside an open (non-periodic) box: they are clamped into the edge cells (A16).  Their distance to
    the cell block of a tile can then exceed the range the fp32 prefilter of the list builder is proven for: such half tiles must
    go to the general kernels (a declined unit), and the neighbour sets and sums must stay those of the oracle."""
    w = W.random_cloud(4000, seed=31, periodic=(0, 0, 0), hvar=1.0, ncell=(6, 6, 6))
    rng = np.random.default_rng(3)
    far = rng.choice(w.n, size=40, replace=False)
    w.x[far[:20]] += 7.3            # far outside the box in +x: clamped into the last column
    w.z[far[20:]] -= 5.1            # and in -z
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    st = sp.path_stats_full()
    assert st["tiles"] > 0 and st["n_fast"] < w.n and st["declined"][3] > 0, st
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt, ds, dx = O.neighbor_digest(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(u32(sp.neighbor_counts(sym)), cnt)
        gs, gx = sp.neighbor_digest(sym)
        assert np.array_equal(gs.cpu().numpy().view(np.uint64), ds) and np.array_equal(gx.cpu().numpy().view(np.uint64), dx)
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    errs = compare_isolated(gpu_isolated(sp, d, w, mu_in=mu_full), oracle_isolated(w, mu_full=mu_full))
    assert sp.check() == 0          # open box: nothing to flag
    print(st, {k: f"{v:.1e}" for k, v in errs.items()})


def test_levels_and_timing_arguments():
    import paper_2604_20124_b200 as P
    w = W.make("c1_tiny")
    d = upload(w)
    sp = make_ctx(w)
    with pytest.raises(P.SprayError, match=r"\(-2\)"):          # NOT_BUILT
        sp.build_timing()
    with pytest.raises(P.SprayError, match=r"\(-1\)"):          # edges must ascend
        sp.set_levels(w.grid, [0.3, 0.2])
    sp.set_levels(w.grid, [2.0 * float(w.h.max()) * 1.001])
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = sp.build_timing()
    assert len(t) == 3 and all(v >= 0.0 for v in t) and t[0] > 0.0
    assert sp.path_stats_full()["n_fast"] == w.n
