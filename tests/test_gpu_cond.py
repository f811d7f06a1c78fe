"""GPU parity of row N2 (spray_conduction, eqs. (17)/(18) second term) against oracle.conduction: |gpu - oracle| <= 1e-11 S_a,
S_a = sum of the absolute pair contributions; exact zero for a uniform temperature."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import check, make_ctx, upload

pytestmark = pytest.mark.gpu


def workload(name):
    if name == "c1":
        return W.make("c1")
    if name == "lattice_wendland":
        return W.config3(nside=24)
    if name == "cloud_periodic":
        return W.random_cloud(5000, seed=12, periodic=(1, 1, 1), hvar=2.0, kernel=W.KERNEL_CUBIC_SPLINE)
    if name == "cloud_mixed":
        return W.random_cloud(4000, seed=13, periodic=(1, 0, 1), hvar=2.2)
    raise KeyError(name)


@pytest.mark.parametrize("name", ["c1", "lattice_wendland", "cloud_periodic", "cloud_mixed"])
def test_conduction_parity(name):
    import torch
    w = workload(name)
    k = 0.2 + w.kappa / (1.0 + w.kappa)
    T = 0.5 + w.E / np.max(w.E)
    o = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, k, T)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.conduction(d["m"], d["rho_nom"], t(k), t(T)).cpu().numpy()
    e = check("dudt", g, o["dudt"], o["S_dudt"])
    assert abs(np.sum(w.m * g)) <= 1e-11 * np.sum(w.m * o["S_dudt"])      # conservative on the GPU as well
    g0 = sp.conduction(d["m"], d["rho_nom"], t(k), t(np.full(w.n, 1.25))).cpu().numpy()
    assert np.all(g0 == 0.0)
    assert sp.check() == 0
    print(name, "max normalised error", e)


def test_conduction_full_size_sampled():
    """Config 5 (16.7M particles), the launch configuration of bench.py: 2000 sampled targets against the oracle."""
    import torch
    w = W.make("c5")
    i = np.arange(2000, dtype=np.uint64)
    sel = np.unique((W.splitmix64(i + np.uint64(91)) % np.uint64(w.n)).astype(np.int64))
    k = 0.2 + w.kappa / (1.0 + w.kappa)
    T = 0.5 + w.E / np.max(w.E) + 0.1 * np.sin(9.0 * w.x)
    o = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, k, T, targets=sel)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.conduction(d["m"], d["rho_nom"], t(k), t(T)).cpu().numpy()
    e = check("dudt", g[sel], o["dudt"], o["S_dudt"])
    assert sp.path_stats()[1] == w.n          # every particle was served by the tiled kernels
    print("c5 sampled: max normalised error", e)


# ---------------------------------------------------------------- implicit two-temperature system, eqs. (28)-(34)
def _state(w, seed=3):
    i = np.arange(w.n, dtype=np.int64)
    k_i = 0.05 + 0.2 * W.u01(seed, i, 0)
    k_e = 0.3 + w.kappa / (1.0 + w.kappa)
    kei = 0.5 + 2.0 * W.u01(seed, i, 1)
    tau_i = 0.6 + 0.3 * W.u01(seed, i, 2)
    tau_e = 1.2 + 0.5 * W.u01(seed, i, 3)
    u_i = 0.8 + 0.4 * W.u01(seed, i, 4)
    u_e = 1.5 + w.E / np.max(w.E)
    T_i = tau_i * u_i + 0.05 * W.u01(seed, i, 5)
    T_e = tau_e * u_e - 0.03 * W.u01(seed, i, 6)
    return k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e


@pytest.mark.parametrize("name", ["c1", "lattice_wendland", "cloud_periodic", "cloud_mixed"])
def test_conduction_implicit_parity(name):
    """Operator and right-hand side of eqs. (28)-(34) against oracle.cond_implicit (which assembles them from Lambda, chi, Gamma,
    b, c in the paper's notation): |gpu - oracle| <= 1e-11 S_a, S_a = the sum of the absolute contributions to the row."""
    import torch
    from paper_2604_20124_b200 import COND_OPERATOR, COND_RHS
    w = workload(name)
    st = _state(w)
    dt = 0.3 * float(w.h.min()) ** 2 / 0.5
    o = O.cond_implicit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, *st, dt)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ts = [t(a) for a in st]
    li, le = sp.conduction_implicit(d["m"], d["rho_nom"], *ts[:5], None, None, ts[7], ts[8], dt, COND_OPERATOR)
    ri, re = sp.conduction_implicit(d["m"], d["rho_nom"], *ts, dt, COND_RHS)
    torch.cuda.synchronize()
    e = max(check("lhs_i", li.cpu().numpy(), o["lhs_i"], o["S_i"]), check("lhs_e", le.cpu().numpy(), o["lhs_e"], o["S_e"]),
            check("rhs_i", ri.cpu().numpy(), o["rhs_i"], o["S_i"]), check("rhs_e", re.cpu().numpy(), o["rhs_e"], o["S_e"]))
    assert np.max(np.abs(o["lhs_i"] - st[7])) > 1e-6 * np.max(st[7])          # the step does something at this dt
    # energy conservation of the operator on the GPU result
    mm = w.m
    assert abs(np.sum(mm * (li.cpu().numpy() + le.cpu().numpy() - st[7] - st[8]))) <= 1e-11 * np.sum(mm * (o["S_i"] + o["S_e"]))
    assert sp.check() == 0
    print(name, "max normalised error", e)


def test_conduction_implicit_full_size_sampled():
    """Config 5 (16.7M particles), the launch configuration of bench.py: operator and right-hand side of eqs. (28)-(34) at 1500
    sampled rows against oracle.cond_implicit (which evaluates those rows only)."""
    import torch
    from paper_2604_20124_b200 import COND_OPERATOR, COND_RHS
    w = W.make("c5")
    i = np.arange(1500, dtype=np.uint64)
    sel = np.unique((W.splitmix64(i + np.uint64(177)) % np.uint64(w.n)).astype(np.int64))
    st = _state(w, seed=5)
    dt = 0.3 * float(w.h.min()) ** 2 / 0.5
    o = O.cond_implicit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, *st, dt, targets=sel)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ts = [t(a) for a in st]
    li, le = sp.conduction_implicit(d["m"], d["rho_nom"], *ts[:5], None, None, ts[7], ts[8], dt, COND_OPERATOR)
    ri, re = sp.conduction_implicit(d["m"], d["rho_nom"], *ts, dt, COND_RHS)
    torch.cuda.synchronize()
    g = lambda a: a.cpu().numpy()[sel]
    e = max(check("lhs_i", g(li), o["lhs_i"], o["S_i"]), check("lhs_e", g(le), o["lhs_e"], o["S_e"]),
            check("rhs_i", g(ri), o["rhs_i"], o["S_i"]), check("rhs_e", g(re), o["rhs_e"], o["S_e"]))
    assert np.max(np.abs(o["lhs_e"] - st[8][sel])) > 1e-6 * np.max(st[8])
    assert sp.path_stats()[1] == w.n          # every particle was served by the tiled kernels
    assert sp.check() == 0
    print("c5 sampled: max normalised error", e)


def test_conduction_implicit_jacobi_solve_converges_to_backward_euler():
    """The operator in use: a damped Jacobi iteration u <- u + (rhs - A u) / Lambda-bound on the GPU operator converges, and the
    fixed point satisfies eqs. (26)/(27) with the extrapolated temperature evaluated by the oracle's explicit conduction term."""
    import torch
    from paper_2604_20124_b200 import COND_OPERATOR, COND_RHS
    w = workload("c1")
    k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e = st = _state(w)
    dt = 0.1 * float(w.h.min()) ** 2 / 0.5
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ts = [t(a) for a in st]
    ri, re = sp.conduction_implicit(d["m"], d["rho_nom"], *ts, dt, COND_RHS)
    vi, ve = ts[7].clone(), ts[8].clone()
    for _ in range(200):
        ai, ae = sp.conduction_implicit(d["m"], d["rho_nom"], *ts[:5], None, None, vi, ve, dt, COND_OPERATOR)
        vi = vi + 0.5 * (ri - ai)
        ve = ve + 0.5 * (re - ae)
    ai, ae = sp.conduction_implicit(d["m"], d["rho_nom"], *ts[:5], None, None, vi, ve, dt, COND_OPERATOR)
    assert float((ri - ai).abs().max()) < 1e-10 and float((re - ae).abs().max()) < 1e-10
    v_i, v_e = vi.cpu().numpy(), ve.cpu().numpy()
    Tn_i = T_i + tau_i * (v_i - u_i); Tn_e = T_e + tau_e * (v_e - u_e)
    g = (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom)
    ci = O.conduction(*g, k_i, Tn_i)["dudt"]; ce = O.conduction(*g, k_e, Tn_e)["dudt"]
    assert np.allclose(v_i - u_i, dt * (ci + kei * (Tn_e - Tn_i)), rtol=0, atol=1e-9)
    assert np.allclose(v_e - u_e, dt * (ce - kei * (Tn_e - Tn_i)), rtol=0, atol=1e-9)
    assert abs(np.sum(w.m * (v_i + v_e - u_i - u_e))) <= 1e-10 * np.sum(w.m * (u_i + u_e))
