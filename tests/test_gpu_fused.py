"""GPU parity of spray_hydro_rhs_limiter (rows (a6) + (a7) in one sweep, include/spray.h): the hydro right-hand sides against
oracle.hydro and mu / gradE against oracle.limiter with the tolerances of the separate calls, and -- the stronger statement --
bitwise equality with spray_hydro_rhs followed by spray_fld_apply(UPDATE_LIMITER), which the fused kernel promises (same pair
terms, same summation order), on uniform-h tiles (fused kernel), variable-h tiles and general-path particles (separate kernels
inside the call), at the bench size too."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import check, check_mu, make_ctx, upload

pytestmark = pytest.mark.gpu


def workload(name):
    if name == "lattice_wendland":
        return W.config3(nside=24)
    if name == "cloud_periodic":
        return W.random_cloud(5000, seed=12, periodic=(1, 1, 1), hvar=2.0, kernel=W.KERNEL_CUBIC_SPLINE)
    if name == "cloud_mixed":
        return W.random_cloud(4000, seed=13, periodic=(1, 0, 1), hvar=2.2)
    return W.make(name)


def _both(sp, d, w):
    import torch
    hy = sp.hydro_rhs(d["m"], d["rho_nom"], d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
    fl = sp.fld_apply(d["m"], d["rho_nom"], d["kappa"], d["E"], w.c_light, want_gradE=True)
    fy, fmu, fg = sp.hydro_rhs_limiter(d["m"], d["rho_nom"], d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], d["E"], d["kappa"],
                                       beta=w.beta, c_light=w.c_light, want_gradE=True)
    # the (mu, E) records the fused call leaves behind serve a FROZEN apply exactly like those of the UPDATE call
    # (FROZEN_CHAINED reuses them without the per-call prologue: it must come right after the fused call, and equal FROZEN bit for bit)
    fc = sp.fld_apply(d["m"], d["rho_nom"], None, d["E"], w.c_light, lmode=2, mu=fmu)
    fc2 = sp.fld_apply(d["m"], d["rho_nom"], None, d["E"], w.c_light, lmode=2, mu=fmu)      # repeatable: the apply changes no record
    fr = sp.fld_apply(d["m"], d["rho_nom"], None, d["E"], w.c_light, lmode=1, mu=fmu)
    for k in ("y", "diag", "offd"):
        assert torch.equal(fc[k], fr[k]) and torch.equal(fc2[k], fr[k]), "chained " + k
    import paper_2604_20124_b200 as P
    with pytest.raises(P.SprayError, match=r"\(-1\)"):      # after any other call the chain is broken
        sp.fld_apply(d["m"], d["rho_nom"], None, d["E"], w.c_light, lmode=2, mu=fmu)
    torch.cuda.synchronize()
    return hy, fl, fy, fmu, fg, fr


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("name", ["c1", "lattice_wendland", "cloud_periodic", "cloud_mixed", "c2"])
def test_fused_equals_separate_calls_bitwise(name, path):
    w = workload(name)
    d = upload(w)
    sp = make_ctx(w, path)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    hy, fl, fy, fmu, fg, fr = _both(sp, d, w)
    for k, a, b in zip(("ax", "ay", "az", "dudt", "divv"), hy, fy):
        assert np.array_equal(a.cpu().numpy(), b.cpu().numpy()), k
    assert np.array_equal(fl["mu"].cpu().numpy(), fmu.cpu().numpy())
    assert np.array_equal(fl["gradE"].cpu().numpy(), fg.cpu().numpy())
    assert np.array_equal(fl["y"].cpu().numpy(), fr["y"].cpu().numpy())
    assert sp.check() == 0


@pytest.mark.parametrize("name", ["c1", "cloud_mixed"])
def test_fused_against_oracle(name):
    import torch
    w = workload(name)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    fy, fmu, fg = sp.hydro_rhs_limiter(d["m"], d["rho_nom"], d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], d["E"], d["kappa"],
                                       beta=w.beta, c_light=w.c_light, want_gradE=True)
    torch.cuda.synchronize()
    a = (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)
    oh = O.hydro(*a, w.rho_nom, w.p, w.cs, w.vx, w.vy, w.vz, w.alpha, w.beta)
    ol = O.limiter(*a, w.rho_nom, w.kappa, w.E, w.c_light)
    e = [check(k, t.cpu().numpy(), oh[k], oh["S_" + k]) for k, t in zip(("ax", "ay", "az", "dudt", "divv"), fy)]
    g = fg.cpu().numpy().reshape(3, w.n)
    e += [check("g" + c, g[i], ol["g" + c], ol["S_g" + c]) for i, c in enumerate("xyz")]
    e.append(check_mu(fmu.cpu().numpy(), ol))
    assert sp.check() == 0
    print(name, "max normalised errors", ["%.1e" % v for v in e])


def test_fused_full_size_bitwise():
    """Config 5 (16.7M particles), the launch configuration of bench.py: the fused call equals the two separate calls bit for bit
    (whose sampled parity against the oracle at this size is tests/test_gpu_fullsize.py), every particle on the tiled kernels."""
    w = W.make("c5")
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    hy, fl, fy, fmu, fg, fr = _both(sp, d, w)
    import torch
    for k, a, b in zip(("ax", "ay", "az", "dudt", "divv"), hy, fy):
        assert torch.equal(a, b), k
    assert torch.equal(fl["mu"], fmu) and torch.equal(fl["gradE"], fg) and torch.equal(fl["y"], fr["y"])
    assert sp.path_stats()[1] == w.n
    assert sp.check() == 0
