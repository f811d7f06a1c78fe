"""GPU parity of row N1 (spray_rad_jacobi, section 2.3) against oracle.rad_jacobi on the same seeded inputs.
Tolerance: every iteration passes Lambda and Gamma (accurate to 1e-11 of sum |c_ab E_b|, the bar of the apply) through
eq. (54), E = (E^n + dt Gamma + X a chi^4)/(1 - dt Lambda + X) with |dE/dGamma| <= dt and d(chi)/dGamma bounded the same
way, so after k iterations |E_gpu - E_oracle| <= k * 1e-11 * (|E| + dt * S_offd); u follows from eq. (55) scaled by
dt c kappa_P.  The measured error is two orders below that."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import make_ctx, upload

pytestmark = pytest.mark.gpu
GAMMA = 5.0 / 3.0
NITER = 5


def workload(name):
    if name == "c1":
        return W.make("c1")
    if name == "cloud_periodic":
        return W.random_cloud(5000, seed=12, periodic=(1, 1, 1), hvar=2.0, kernel=W.KERNEL_CUBIC_SPLINE)
    if name == "cloud_open":
        return W.random_cloud(3000, seed=11, periodic=(0, 0, 0), hvar=3.0)
    if name == "lattice_wendland":
        return W.config3(nside=20)
    raise KeyError(name)


@pytest.mark.parametrize("name", ["c1", "lattice_wendland", "cloud_periodic", "cloud_open"])
@pytest.mark.parametrize("kmode", [0, 1])
def test_rad_jacobi_parity(name, kmode):
    import torch
    w = workload(name)
    n = w.n
    u_n = w.p / ((GAMMA - 1.0) * w.rho_nom)
    T_n = (GAMMA - 1.0) * u_n
    dTdu = np.full(n, GAMMA - 1.0)
    kp = 0.5 + w.kappa / (1.0 + w.kappa)                      # a positive Planck opacity of order one
    mu = w.c_light / (3.0 * w.rho_nom * w.kappa)
    a_rad, dt = 1.0, 0.3 * float(np.min(w.h)) ** 2 / float(np.max(mu))      # a few diffusion times of the smallest h
    E_n = w.E * (0.5 + (w.x - w.x.min()) / (w.x.max() - w.x.min() + 1e-300))   # not in equilibrium with T
    o = O.rad_jacobi(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, mu, kp, E_n, u_n, T_n, dTdu, dt, w.c_light, a_rad,
                     NITER, sym_mode=(kmode == 0))
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.rad_jacobi(d["m"], d["rho_nom"], t(mu), t(kp), t(E_n), t(u_n), t(T_n), t(dTdu), dt, w.c_light, a_rad, niter=NITER,
                      kmode=kmode)
    torch.cuda.synchronize()
    E, u, resid = g["E"].cpu().numpy(), g["u"].cpu().numpy(), g["resid"].cpu().numpy()
    assert np.isfinite(E).all() and np.isfinite(u).all()
    tolE = NITER * 1e-11 * (np.abs(o["E"]) + dt * o["S_offd"])
    assert (np.abs(E - o["E"]) <= tolE).all(), f"E: worst {np.max(np.abs(E - o['E']) / tolE):.2e} x tol"
    K = dt * w.c_light * kp
    tolu = K * tolE + NITER * 1e-11 * np.abs(o["u"])
    assert (np.abs(u - o["u"]) <= tolu).all(), f"u: worst {np.max(np.abs(u - o['u']) / tolu):.2e} x tol"
    # the iteration actually moved the fields, and the residual of eq. (49) agrees with the oracle's
    assert np.max(np.abs(o["E"] - E_n) / E_n) > 1e-3
    assert resid[0] == 0.0
    assert np.allclose(resid[1:], o["resid"][1:], rtol=1e-6, atol=1e-13)
    assert sp.check() == 0
    print(name, kmode, "max dE/tol", float(np.max(np.abs(E - o["E"]) / tolE)), "resid", resid)


def test_rad_jacobi_full_size_sampled():
    """Config 5 (16.7M particles), the launch configuration of bench.py: the first Jacobi iteration at 2000 sampled targets
    (the oracle can follow a sample for one iteration: later ones need the iterate everywhere)."""
    import torch
    w = W.make("c5")
    i = np.arange(2000, dtype=np.uint64)
    sel = np.unique((W.splitmix64(i + np.uint64(57)) % np.uint64(w.n)).astype(np.int64))
    u_n = w.p / ((GAMMA - 1.0) * w.rho_nom)
    T_n = (GAMMA - 1.0) * u_n
    dTdu = np.full(w.n, GAMMA - 1.0)
    kp = 0.5 + w.kappa / (1.0 + w.kappa)
    mu = w.c_light / (3.0 * w.rho_nom * w.kappa)
    a_rad, dt = 1.0, 0.3 * float(np.min(w.h)) ** 2 / float(np.max(mu))
    E_n = w.E * (0.5 + (w.x - w.x.min()) / (w.x.max() - w.x.min()))
    o = O.rad_jacobi(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, mu, kp, E_n, u_n, T_n, dTdu, dt, w.c_light, a_rad,
                     1, targets=sel)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.rad_jacobi(d["m"], d["rho_nom"], t(mu), t(kp), t(E_n), t(u_n), t(T_n), t(dTdu), dt, w.c_light, a_rad, niter=1)
    torch.cuda.synchronize()
    E, u = g["E"].cpu().numpy()[sel], g["u"].cpu().numpy()[sel]
    # eq. (55), E = (u - u^n)/(dt c kappa_P) + a chi^4, divides the rounding error of chi (a few ulp, from the last Newton
    # step on either side) by dTdu dt c kappa_P, which is ~1e-5 at this workload's time step: that term is added to the bound
    K = dt * w.c_light * kp[sel]
    tolE = 1e-11 * (np.abs(o["E"]) + dt * o["S_offd"]) + 8.0 * np.finfo(np.float64).eps * np.abs(o["chi"]) / (dTdu[sel] * K)
    assert (np.abs(E - o["E"]) <= tolE).all(), f"E: worst {np.max(np.abs(E - o['E']) / tolE):.2e} x tol"
    tolu = K * tolE + 1e-11 * np.abs(o["u"])
    assert (np.abs(u - o["u"]) <= tolu).all()
    assert np.max(np.abs(o["E"] - E_n[sel]) / E_n[sel]) > 1e-4
    print("c5 sampled: max dE/tol", float(np.max(np.abs(E - o["E"]) / tolE)))
