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
