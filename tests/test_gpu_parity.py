"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Integer outputs (cell table, neighbour sets) bit-exact; fp64 outputs within 1e-11 of the sum of absolute
pair contributions (BASELINE.json north_star).  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import (check, check_mu, compare_isolated, gpu_isolated, make_ctx, oracle_isolated, u32, u64, upload)

pytestmark = pytest.mark.gpu

SMALL = ["c1_tiny", "c2_tiny", "c3_tiny", "c4_tiny", "c5_tiny"]
MID = ["c2_mid", "c3_mid", "c4_mid", "c5_mid"]
PATHS = [0, 1]


def get_workload(name):
    if name == "cloud_open":
        return W.random_cloud(3000, seed=11, periodic=(0, 0, 0), hvar=3.0)
    if name == "cloud_periodic":
        return W.random_cloud(5000, seed=12, periodic=(1, 1, 1), hvar=2.0, kernel=W.KERNEL_CUBIC_SPLINE)
    if name == "cloud_mixed":
        return W.random_cloud(4000, seed=13, periodic=(1, 0, 1), hvar=2.2)
    return W.make(name)


@pytest.fixture(scope="module", params=SMALL + MID + ["cloud_open", "cloud_periodic", "cloud_mixed"])
def case(request):
    w = get_workload(request.param)
    d = upload(w)
    return w, d


@pytest.mark.parametrize("path", PATHS)
def test_cell_table_bit_exact(case, path):
    w, d = case
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = sp.get_cell_table()
    assert sp.check() == 0
    ref = O.build_cells(w.grid, w.x, w.y, w.z)
    for k in ("sorted_key", "perm", "cell_start", "cell_end"):
        assert np.array_equal(u32(t[k]), ref[k]), k


def test_neighbour_sets_bit_exact(case):
    w, d = case
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    for sym, mode in ((False, O.GATHER), (True, O.SYM)):
        off, nbr = sp.neighbor_lists(sym)
        ooff, onbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, mode)
        assert np.array_equal(off.cpu().numpy().astype(np.uint64), ooff)
        assert np.array_equal(u32(nbr), onbr)
        ds, dx = sp.neighbor_digest(sym)
        hsh = W.splitmix64(onbr.astype(np.uint64))
        cs = np.concatenate([[np.uint64(0)], np.cumsum(hsh, dtype=np.uint64)])
        want_sum = cs[ooff[1:].astype(np.int64)] - cs[ooff[:-1].astype(np.int64)]
        assert np.array_equal(u64(ds), want_sum)
        rows = np.repeat(np.arange(w.n), np.diff(ooff).astype(np.int64))
        want_xor = np.zeros(w.n, np.uint64)
        np.bitwise_xor.at(want_xor, rows, hsh)
        assert np.array_equal(u64(dx), want_xor)
    assert sp.check() == 0


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("kmode", [0, 1])
def test_sweeps_isolated(case, path, kmode):
    """Every sweep on its own, with identical inputs on both sides (rho = recipe density, mu = oracle mu)."""
    w, d = case
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    mu_full = O.limiter(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.kappa, w.E, w.c_light)["mu"]
    g = gpu_isolated(sp, d, w, mu_in=mu_full, kmode=kmode)
    o = oracle_isolated(w, sym_mode=(kmode == 0), mu_full=mu_full)
    errs = compare_isolated(g, o)
    assert sp.check() == 0
    print(w.name, "path", path, {k: f"{v:.1e}" for k, v in errs.items()})


@pytest.mark.parametrize("path", PATHS)
def test_chained_pass(case, path):
    """The pass as bench.py runs it: density -> hydro(rho) -> fld(rho), each side feeding its own rho and mu."""
    import torch
    w, d = case
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    rho = sp.density(d["m"])
    hy = sp.hydro_rhs(d["m"], rho, d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
    fl = sp.fld_apply(d["m"], rho, d["kappa"], d["E"], w.c_light)
    torch.cuda.synchronize()
    a = (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)
    od = O.density(*a)
    oh = O.hydro(*a, od["rho"], w.p, w.cs, w.vx, w.vy, w.vz, w.alpha, w.beta)
    ol = O.limiter(*a, od["rho"], w.kappa, w.E, w.c_light)
    oa = O.fld_apply(*a, od["rho"], ol["mu"], w.E, sym_mode=True)
    check("rho", rho.cpu().numpy(), od["rho"], od["S_rho"])
    # rho differs by ~1e-16 relative between the two sides; it enters each pair term linearly => same normalised bound
    for k, t in zip(("ax", "ay", "az", "dudt", "divv"), hy):
        check(k, t.cpu().numpy(), oh[k], oh["S_" + k])
    check_mu(fl["mu"].cpu().numpy(), ol)
    # y depends on mu_a, mu_b with the relative perturbation allowed for mu: widen by that factor
    # c_ab is homogeneous of degree one in (mu_a, mu_b), so its relative perturbation is at most the larger of the two
    # particles' allowed relative perturbation of mu: widen PER PARTICLE by the worst factor over a and its own
    # symmetric neighbours (not by the global worst).
    from parity_util import mu_tolerance
    tol_mu = mu_tolerance(ol)
    off, nbr = O.neighbor_lists(w.grid, w.x, w.y, w.z, w.h, O.SYM)
    worst = tol_mu.copy()
    if nbr.size:
        rows = np.repeat(np.arange(w.n), np.diff(off).astype(np.int64))
        np.maximum.at(worst, rows, tol_mu[nbr])
    gy, S = fl["y"].cpu().numpy(), oa["S_y"]
    bound = (1e-11 + 2.0 * worst) * S
    z = S == 0
    assert np.array_equal(gy[z], oa["y"][z]) and np.isfinite(gy).all()
    bad = np.abs(gy - oa["y"]) > bound
    assert not bad.any(), f"y: {bad.sum()} particles beyond the per-particle bound, worst {float((np.abs(gy - oa['y'])[~z] / bound[~z]).max()):.2e} x"
    assert sp.check() == 0


@pytest.mark.parametrize("path", PATHS)
def test_run_to_run_bitwise_identical(path):
    import torch
    w = W.make("c4_tiny")
    d = upload(w)
    outs = []
    for _ in range(2):
        sp = make_ctx(w, path)
        sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
        rho = sp.density(d["m"])
        hy = sp.hydro_rhs(d["m"], rho, d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
        fl = sp.fld_apply(d["m"], rho, d["kappa"], d["E"], w.c_light)
        torch.cuda.synchronize()
        outs.append([rho.cpu().numpy()] + [t.cpu().numpy() for t in hy] + [fl[k].cpu().numpy() for k in ("mu", "y", "diag", "offd")])
    for a, b in zip(*outs):
        assert np.array_equal(a, b)       # no floating-point atomics on the hot path


def test_conservation_on_gpu_outputs():
    """Properties that hold at any size (used again at full size): momentum, energy, FLD conservation."""
    import torch
    w = W.make("c4_mid")
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    rho = sp.density(d["m"])
    ax, ay, az, dudt, divv = sp.hydro_rhs(d["m"], rho, d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
    fl = sp.fld_apply(d["m"], rho, d["kappa"], d["E"], w.c_light)
    m = d["m"]
    for a in (ax, ay, az):
        assert abs(float((m * a).sum())) <= 1e-12 * float((m * a).abs().sum())
    e = m * (d["vx"] * ax + d["vy"] * ay + d["vz"] * az + dudt)
    pdv = (m * d["p"] / rho * divv).abs().sum()
    assert abs(float(e.sum())) <= 1e-12 * float(pdv + (m * (d["vx"] * ax).abs()).sum())
    V = m / rho
    assert abs(float((V * fl["y"]).sum())) <= 1e-12 * float((V * fl["y"]).abs().sum())
    assert bool((fl["diag"] <= 0).all())
