"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times: sampled outputs the oracle
computes one by one (its cell-list variant, restricted to the sampled targets), neighbour-set digests, the full cell
table, and conservation properties that hold at any size."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import compare_isolated, gpu_isolated, make_ctx, oracle_isolated, u32, u64, upload

pytestmark = pytest.mark.gpu
NSAMPLE = 768


def sample_targets(w, seed=0):
    rng = np.random.default_rng(seed)
    t = rng.choice(w.n, size=NSAMPLE - 8, replace=False)
    # always include the first/last particles and the extremes of h (the load-imbalance end of config 4)
    extra = np.array([0, 1, w.n - 1, w.n - 2, int(np.argmax(w.h)), int(np.argmin(w.h)), int(np.argmax(w.x)), int(np.argmin(w.x))])
    return np.unique(np.concatenate([t, extra])).astype(np.int64)


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5"])
def test_full_size_sampled(name):
    import torch
    w = W.make(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    # (1) the whole cell table, bit-exact
    ref = O.build_cells(w.grid, w.x, w.y, w.z)
    t = sp.get_cell_table()
    for k in ("sorted_key", "perm", "cell_start", "cell_end"):
        assert np.array_equal(u32(t[k]), ref[k]), k
    del t, ref
    # (2) neighbour sets of the sampled targets via counts + order-independent digests
    tg = sample_targets(w)
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        cnt = u32(sp.neighbor_counts(sym))[tg]
        ds, dx = sp.neighbor_digest(sym)
        ds, dx = u64(ds)[tg], u64(dx)[tg]
        off, nbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, mode, targets=tg)
        assert np.array_equal(cnt, np.diff(off).astype(np.uint32))
        hsh = W.splitmix64(nbr.astype(np.uint64))
        for i in range(tg.size):
            seg = hsh[int(off[i]):int(off[i + 1])]
            assert ds[i] == np.add.reduce(seg, dtype=np.uint64) and dx[i] == np.bitwise_xor.reduce(seg, initial=np.uint64(0))
    # (3) every sweep at the sampled targets, identical inputs on both sides.  mu for the frozen apply is needed at the
    # targets' neighbours too: take the oracle's mu on the closure (targets + their symmetric neighbours).
    off, nbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, O.SYM, targets=tg)
    closure = np.unique(np.concatenate([tg, nbr.astype(np.int64)]))
    mu_c = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light, targets=closure)["mu"]
    mu_full = np.ones(w.n)
    mu_full[closure] = mu_c
    g = gpu_isolated(sp, d, w, targets=tg, mu_in=mu_full)
    o = oracle_isolated(w, targets=tg, mu_full=mu_full)
    errs = compare_isolated(g, o)
    print(name, w.n, {k: f"{v:.1e}" for k, v in errs.items()})
    # (4) properties at full size on the chained pass
    rho = sp.density(d["m"])
    ax, ay, az, dudt, divv = sp.hydro_rhs(d["m"], rho, d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
    fl = sp.fld_apply(d["m"], rho, d["kappa"], d["E"], w.c_light)
    m = d["m"]
    for a in (ax, ay, az):
        assert abs(float((m * a).sum())) <= 1e-11 * float((m * a).abs().sum()) + 1e-300
    V = m / rho
    assert abs(float((V * fl["y"]).sum())) <= 1e-11 * float((V * fl["y"]).abs().sum()) + 1e-300
    assert bool((fl["diag"] <= 0).all()) and bool(torch.isfinite(fl["y"]).all())
    assert sp.check() == 0


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5"])
def test_full_population_neighbour_digests(name):
    """the neighbour sets of EVERY particle at full size, both set kinds, as (count, sum, xor) digests of the
    hashed caller ids -- the GPU's come from the lists the sweeps run on (and from the general kernels for what the tiled
    path declines), the oracle's from oracle_neighbor_digest (pinned in tests/test_oracle_pins.py)."""
    w = W.make(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    uniform = float(w.h.min()) == float(w.h.max())
    ref = {}
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        if sym and uniform:
            ref[mode] = ref[O.GATHER]          # one h: N_sym(a) = N_gather(a) minus a, nothing to transpose
        else:
            ref[mode] = O.neighbor_digest(w.grid, w.x, w.y, w.z, w.h, mode)
        cnt, ds, dx = ref[mode]
        assert np.array_equal(u32(sp.neighbor_counts(sym)), cnt), (name, sym, "counts")
        gs, gx = sp.neighbor_digest(sym)
        assert np.array_equal(u64(gs), ds), (name, sym, "sum digests")
        assert np.array_equal(u64(gx), dx), (name, sym, "xor digests")
    assert sp.check() == 0


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5", "c5_v"])
def test_full_size_outputs(name):
    """Every fp64 output of every sweep: ALL particles at c2 and c3, 200 000 sampled targets at c4, c5 and c5_v (the c5
    variant with v ~ N(0, 0.01^2): the viscous branch of eqs. (41)-(43) at full size on the tiled path).  The frozen apply
    takes mu = c / (3 rho kappa) (the diffusion limit, computed here from the inputs) on both sides, so no closure of the
    sample is needed; the limiter sweep (UPDATE mode) is compared on its own."""
    w = W.make(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    if name in ("c2", "c3"):
        tg = None
    else:
        rng = np.random.default_rng(5)
        tg = np.sort(rng.choice(w.n, size=200000, replace=False)).astype(np.int64)
    mu_full = w.c_light / (3.0 * w.rho_nom * w.kappa)
    g = gpu_isolated(sp, d, w, targets=tg, mu_in=mu_full)
    o = oracle_isolated(w, targets=tg, mu_full=mu_full)
    errs = compare_isolated(g, o)
    if name == "c5_v":
        assert np.abs(o["dudt"]).max() > 0 and (o["S_dudt"] > 0).all()
    assert sp.check() == 0
    print(name, w.n, "all" if tg is None else tg.size, {k: f"{v:.1e}" for k, v in errs.items()})
