"""Pins of the N2 oracle (thermal-conduction term of eqs. (17)/(18)): oracle.conduction."""
import math

import numpy as np
import pytest

import oracle as O
import workloads as W
from test_oracle_pins import KID, golden, open_block_fields


def test_conduction_conserves_energy_under_variable_h():
    """the conduction terms conserve energy because they are symmetric in (a, b): sum_a m_a dudt_a = 0 to rounding,
    for unequal masses and variable h as well (m_a/rho_a V_b c_ab is symmetric)."""
    w = W.random_cloud(4000, seed=5, periodic=(1, 0, 1), hvar=2.2)
    k = 0.3 + w.kappa
    T = 0.5 + w.E
    r = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, k, T)
    assert abs(np.sum(w.m * r["dudt"])) <= 1e-14 * np.sum(w.m * r["S_dudt"])
    assert np.max(np.abs(r["dudt"])) > 0


def test_uniform_temperature_conducts_nothing():
    w = W.random_cloud(800, seed=6, periodic=(0, 0, 0), hvar=2.0)
    r = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, 0.3 + w.kappa, np.full(w.n, 1.7))
    assert np.all(r["dudt"] == 0.0)


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
def test_two_particles_heat_flows_from_hot_to_cold(kname):
    """Two equal particles one h apart, equal k: dudt_a = 4 m/rho^2 (k/2) (T_a - T_b) F(q=1)/h with the closed-form
    F(q=1) = -105/(128 pi h^4) (Wendland, eq. (3)) or -3/(4 pi h^4) (cubic spline): the hot one cools, the cold one heats."""
    h, m, rho, k0 = 0.1, 0.02, 1.5, 0.8
    x = np.array([0.3, 0.3 + h]); y = np.array([0.5, 0.5]); z = np.array([0.5, 0.5])
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (4, 4, 4), (0, 0, 0), h)
    T = np.array([2.0, 1.0])
    r = O.conduction(g, KID[kname], x, y, z, np.full(2, h), np.full(2, m), np.full(2, rho), np.full(2, k0), T)
    F1 = -105.0 / (128.0 * math.pi * h ** 4) if kname == "wendland" else -3.0 / (4.0 * math.pi * h ** 4)
    expect = 4.0 * m / rho ** 2 * (k0 / 2.0) * (T[0] - T[1]) * F1 / h
    assert expect < 0
    assert r["dudt"][0] == pytest.approx(expect, rel=1e-13)
    assert r["dudt"][1] == pytest.approx(-expect, rel=1e-13)


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
@pytest.mark.parametrize("hfac", [1.2, 1.3])
def test_quadratic_temperature_gives_the_laplacian(kname, hfac):
    """Constant k, T = T0 + g.x + x'Hx/2 on the unjittered lattice: dudt = k tr(H) S2 / rho, i.e. (1/rho) div(k grad T) of
    eq. (13) P:L110 times the lattice constant S2 of the kernel (tests/golden/lattice_constants.txt)."""
    _, s2 = golden()[(kname, hfac)]
    gvec = np.array([0.7, -1.3, 0.4])
    H = np.array([[1.0, 0.3, -0.2], [0.3, -0.5, 0.6], [-0.2, 0.6, 2.0]])
    x, y, z, h, g, m, rho, T, ctr = open_block_fields(kname, hfac, gvec, H)
    k0 = 0.37
    r = O.conduction(g, KID[kname], x, y, z, h, m, rho, np.full(x.size, k0), T, targets=ctr)
    assert r["dudt"][0] == pytest.approx(k0 * np.trace(H) * s2 / rho[ctr[0]], rel=1e-11)


# ---------------------------------------------------------------- implicit two-temperature system, eqs. (26)-(34) (oracle.cond_implicit)
def _two_temperature_state(w, seed=3):
    i = np.arange(w.n, dtype=np.int64)
    k_i = 0.05 + 0.2 * W.u01(seed, i, 0)
    k_e = 0.3 + w.kappa / (1.0 + w.kappa)
    kei = 0.5 + 2.0 * W.u01(seed, i, 1)
    tau_i = 0.6 + 0.3 * W.u01(seed, i, 2)
    tau_e = 1.2 + 0.5 * W.u01(seed, i, 3)
    u_i = 0.8 + 0.4 * W.u01(seed, i, 4)
    u_e = 1.5 + w.E / np.max(w.E)
    T_i = tau_i * u_i + 0.05 * W.u01(seed, i, 5)          # T need not be tau u (a general equation of state)
    T_e = tau_e * u_e - 0.03 * W.u01(seed, i, 6)
    return k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e


def _geom(w):
    return (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom)


def test_implicit_system_is_eqs_26_27_with_extrapolated_temperature():
    """Substitution: for ANY trial state u^{N+1}, lhs(u^{N+1}) - rhs(u^N, T^N) must equal the residual of the backward-Euler
    eqs. (26)/(27) with T^{N+1} = T^N + tau (u^{N+1} - u^N), evaluated independently with the pinned explicit
    conduction term (oracle.conduction) and the exchange term written out.  A wrong sign or a dropped term anywhere in
    eqs. (28)-(34) -- in particular the sign of Gamma in eq. (29) (A37) -- fails this."""
    w = W.random_cloud(2500, seed=31, periodic=(1, 0, 1), hvar=1.8)
    k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e = _two_temperature_state(w)
    i = np.arange(w.n, dtype=np.int64)
    v_i = u_i * (1.0 + 0.2 * (W.u01(8, i, 0) - 0.5))      # trial u^{N+1}
    v_e = u_e * (1.0 + 0.2 * (W.u01(8, i, 1) - 0.5))
    dt = 0.37
    g = _geom(w)
    rhs = O.cond_implicit(*g, k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e, dt)
    lhs = O.cond_implicit(*g, k_i, k_e, kei, tau_i, tau_e, T_i, T_e, v_i, v_e, dt)
    Tn_i = T_i + tau_i * (v_i - u_i)
    Tn_e = T_e + tau_e * (v_e - u_e)
    ci = O.conduction(*g, k_i, Tn_i); ce = O.conduction(*g, k_e, Tn_e)
    res_i = (v_i - u_i) - dt * (ci["dudt"] + kei * (Tn_e - Tn_i))          # eq. (26)
    res_e = (v_e - u_e) - dt * (ce["dudt"] - kei * (Tn_e - Tn_i))          # eq. (27)
    assert np.max(np.abs(res_i)) > 1e-3
    assert np.all(np.abs((lhs["lhs_i"] - rhs["rhs_i"]) - res_i) <= 1e-13 * (rhs["S_i"] + lhs["S_i"]))
    assert np.all(np.abs((lhs["lhs_e"] - rhs["rhs_e"]) - res_e) <= 1e-13 * (rhs["S_e"] + lhs["S_e"]))


def test_implicit_system_conserves_total_energy():
    """Conduction is symmetric in (a, b) and the exchange terms of the two species cancel, so for any u:
    sum_a m_a [lhs^i + lhs^e - u^i - u^e] = 0 and sum_a m_a [rhs^i + rhs^e - u^i - u^e] = 0: a solution of lhs = rhs has the
    total energy of the old state."""
    w = W.random_cloud(3000, seed=32, periodic=(1, 1, 1), hvar=2.0)
    st = _two_temperature_state(w)
    r = O.cond_implicit(*_geom(w), *st, 0.2)
    u_i, u_e = st[7], st[8]
    scale = np.sum(w.m * (r["S_i"] + r["S_e"]))
    assert abs(np.sum(w.m * (r["lhs_i"] + r["lhs_e"] - u_i - u_e))) <= 1e-13 * scale
    assert abs(np.sum(w.m * (r["rhs_i"] + r["rhs_e"] - u_i - u_e))) <= 1e-13 * scale
    assert np.max(np.abs(r["lhs_i"] - u_i)) > 1e-3 and np.max(np.abs(r["rhs_e"] - u_e)) > 1e-3


def test_implicit_system_equilibrium_and_identity_rows():
    """Uniform, equal temperatures with T = tau u: nothing conducts or is exchanged, so rhs = u^N; and with uniform tau the
    operator maps a uniform u (same for both species) to itself (row sums of A are 1)."""
    w = W.random_cloud(900, seed=33, periodic=(0, 0, 0), hvar=1.6)
    k_i, k_e, kei, *_ = _two_temperature_state(w)
    tau = np.full(w.n, 0.7)
    u = np.full(w.n, 2.0)
    r = O.cond_implicit(*_geom(w), k_i, k_e, kei, tau, tau, tau * u, tau * u, u, u, 0.5)
    for key in ("rhs_i", "rhs_e", "lhs_i", "lhs_e"):
        assert np.allclose(r[key], u, rtol=0, atol=1e-12 * np.max(r["S_i"] + r["S_e"])), key


def test_dense_solve_of_the_operator_satisfies_backward_euler():
    """40 particles: the 2n x 2n matrix of eqs. (28)/(29) assembled column by column from the matrix-free operator (it is
    linear: lhs(u) is applied to unit vectors), solved with numpy; the solution satisfies eqs. (26)/(27) with the extrapolated
    temperature (independent evaluation through oracle.conduction), conserves energy, and the matrix is strictly diagonally
    dominant by columns in the mass-weighted sense (Lambda >= 1)."""
    n = 40
    w = W.random_cloud(n, seed=34, periodic=(0, 0, 0), hvar=1.5)
    h = 1.6 * w.h
    grid = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (1, 1, 1), (0, 0, 0), float(h.max()))
    geom = (grid, w.kernel, w.x, w.y, w.z, h, w.m, w.rho_nom)
    k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e = _two_temperature_state(w)
    dt = 0.8
    args = (k_i, k_e, kei, tau_i, tau_e, T_i, T_e)
    base = O.cond_implicit(*geom, *args, u_i, u_e, dt)
    A = np.zeros((2 * n, 2 * n))
    z = np.zeros(n)
    for j in range(2 * n):
        e = np.zeros(2 * n); e[j] = 1.0
        r = O.cond_implicit(*geom, *args, e[:n], e[n:], dt)
        A[:n, j], A[n:, j] = r["lhs_i"], r["lhs_e"]
    assert np.all(np.diag(A) >= 1.0)
    sol = np.linalg.solve(A, np.concatenate([base["rhs_i"], base["rhs_e"]]))
    v_i, v_e = sol[:n], sol[n:]
    Tn_i = T_i + tau_i * (v_i - u_i); Tn_e = T_e + tau_e * (v_e - u_e)
    ci = O.conduction(*geom, k_i, Tn_i)["dudt"]; ce = O.conduction(*geom, k_e, Tn_e)["dudt"]
    assert np.allclose(v_i - u_i, dt * (ci + kei * (Tn_e - Tn_i)), rtol=1e-9, atol=1e-12)
    assert np.allclose(v_e - u_e, dt * (ce - kei * (Tn_e - Tn_i)), rtol=1e-9, atol=1e-12)
    assert abs(np.sum(w.m * (v_i + v_e - u_i - u_e))) <= 1e-12 * np.sum(w.m * (u_i + u_e))
    assert np.max(np.abs(v_e - u_e)) > 1e-2                                # something happened
    # relaxation: the species' temperatures move towards each other
    assert np.mean(np.abs(Tn_e - Tn_i)) < np.mean(np.abs(T_e - T_i))


def test_cond_implicit_targets_select_rows():
    """`targets` only selects the rows that are evaluated: the sampled rows are bitwise those of the full evaluation."""
    w = W.random_cloud(3000, seed=21, periodic=(1, 0, 1), hvar=1.8)
    i = np.arange(w.n, dtype=np.int64)
    f = lambda c, a, b: a + b * W.u01(9, i, c)
    st = (f(0, 0.05, 0.2), f(1, 0.3, 0.5), f(2, 0.5, 2.0), f(3, 0.6, 0.3), f(4, 1.2, 0.5), f(5, 0.7, 0.4), f(6, 1.9, 0.6),
          f(7, 0.8, 0.4), f(8, 1.5, 0.5))
    dt = 0.3 * float(w.h.min()) ** 2 / 0.5
    full = O.cond_implicit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, *st, dt)
    sel = np.array([0, 7, 2999, 123, 300], dtype=np.int64)
    part = O.cond_implicit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, *st, dt, targets=sel)
    for k in full:
        assert np.array_equal(part[k], full[k][sel]), k
