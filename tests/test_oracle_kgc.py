"""Pins of the N3 oracle (continuity equation eq. (37) P:L213 with the kernel gradient correction of eqs. (39)-(40)
P:L222-L228): oracle.kgc_continuity."""
import math

import numpy as np
import pytest

import oracle as O
import workloads as W
from test_oracle_pins import KID, golden, open_block_fields

A_LIN = np.array([[0.7, -0.4, 0.25], [1.1, -0.3, 0.6], [-0.8, 0.15, 0.45]])     # not symmetric, trace 0.85
B_LIN = np.array([0.3, -1.2, 0.5])


def linear_velocity(w, A=A_LIN, b=B_LIN):
    X = np.stack([w.x, w.y, w.z], 1)
    V = X @ A.T + b
    return V[:, 0], V[:, 1], V[:, 2]


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
@pytest.mark.parametrize("hfac", [1.2, 1.3])
def test_moment_matrix_on_the_lattice_is_S2_times_identity(kname, hfac):
    """On the unjittered cubic lattice the moment matrix of eq. (40) is S2 I by symmetry, S2 the lattice constant of the
    kernel gradient (tests/golden/lattice_constants.txt, the constant of pins T6/T7), so L = I / S2."""
    _, s2 = golden()[(kname, hfac)]
    x, y, z, h, g, m, rho, E, ctr = open_block_fields(kname, hfac, np.zeros(3), np.zeros((3, 3)))
    v = np.zeros_like(x)
    r = O.kgc_continuity(g, KID[kname], x, y, z, h, m, rho, v, v, v, targets=ctr)
    assert np.allclose(r["M"][0], s2 * np.eye(3), rtol=0, atol=1e-13)
    assert np.allclose(r["L"][0], np.eye(3) / s2, rtol=0, atol=1e-12)
    assert abs(s2 - 1.0) < 0.03


@pytest.mark.parametrize("periodic", [(0, 0, 0), (1, 0, 1)])
def test_corrected_continuity_is_exact_for_linear_velocity_on_disordered_particles(periodic):
    """With L = M^-1, sum_b V_b (v_a - v_b) . L gradW = -tr(A) for v = A x + b whatever the particle positions, volumes and
    smoothing lengths are (L M = I), so eq. (37) with eq. (39) returns -rho div v of eq. (36) exactly, also at a free surface;
    the uncorrected sum does not.  (Periodic case: only particles whose support does not cross the box see one linear field.)"""
    w = W.random_cloud(4000, seed=11, periodic=periodic, hvar=2.2)
    vx, vy, vz = linear_velocity(w)
    r = O.kgc_continuity(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, vx, vy, vz)
    X = np.stack([w.x, w.y, w.z], 1)
    inside = np.ones(w.n, bool)
    for d in range(3):
        if periodic[d]:
            inside &= (X[:, d] > 2 * w.h) & (X[:, d] < 1.0 - 2 * w.h)
    lnorm = np.linalg.norm(r["L"].reshape(-1, 9), axis=1)
    snorm = np.linalg.norm(r["S_N"].reshape(-1, 9), axis=1)
    regular = np.abs(np.linalg.det(r["M"])) > 1e-6
    sel = inside & regular
    assert sel.sum() > 0.5 * inside.sum()
    err = np.abs(r["drhodt"] + w.rho_nom * np.trace(A_LIN))
    tol = 1e-12 * w.rho_nom * lnorm * snorm * (1.0 + lnorm * np.linalg.norm(r["S_M"].reshape(-1, 9), axis=1))
    assert np.all(err[sel] <= tol[sel])
    raw_err = np.abs(r["drhodt_raw"] + w.rho_nom * np.trace(A_LIN))
    assert np.median(raw_err[sel]) > 1e3 * np.median(err[sel])          # the filter is what makes it exact


def test_rigid_rotation_and_uniform_flow_do_not_change_density():
    """div v = 0: rigid rotation (antisymmetric A) gives 0 to rounding, uniform velocity gives exactly 0 (every v_ab = 0)."""
    w = W.random_cloud(1500, seed=12, periodic=(0, 0, 0), hvar=2.0)
    Om = np.array([[0.0, -0.9, 0.4], [0.9, 0.0, -0.2], [-0.4, 0.2, 0.0]])
    vx, vy, vz = linear_velocity(w, Om, np.array([0.1, 0.2, -0.3]))
    r = O.kgc_continuity(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, vx, vy, vz)
    reg = np.abs(np.linalg.det(r["M"])) > 1e-6
    lnorm = np.linalg.norm(r["L"].reshape(-1, 9), axis=1)
    scale = w.rho_nom * lnorm * np.linalg.norm(r["S_N"].reshape(-1, 9), axis=1) * (1 + lnorm * np.linalg.norm(r["S_M"].reshape(-1, 9), axis=1))
    assert np.all(np.abs(r["drhodt"][reg]) <= 1e-12 * scale[reg])
    u = np.full(w.n, 0.37)
    r0 = O.kgc_continuity(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, u, 2 * u, -u)
    assert np.all(r0["drhodt"] == 0.0) and np.all(r0["drhodt_raw"] == 0.0)


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
def test_brute_force_on_a_tiny_cloud(kname):
    """Eqs. (37), (39), (40) written out pair by pair in Python over ALL pairs (open box, W and F from the pinned scalar
    kernel functions), with numpy's inverse: catches a transposed operand or a wrong index for a velocity field that is not
    linear."""
    n = 70
    w = W.random_cloud(n, seed=13, kernel=KID[kname], periodic=(0, 0, 0), hvar=1.6)
    h = 1.6 * w.h                                                        # ~ 60 % of the cloud inside each support
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (1, 1, 1), (0, 0, 0), float(h.max()))
    r = O.kgc_continuity(g, KID[kname], w.x, w.y, w.z, h, w.m, w.rho_nom, w.vx, w.vy, w.vz)
    X = np.stack([w.x, w.y, w.z], 1)
    V = np.stack([w.vx, w.vy, w.vz], 1)
    for a in range(n):
        M = np.zeros((3, 3))
        grads = []
        for b in range(n):
            if b == a:
                continue
            xab = X[a] - X[b]
            rr = math.sqrt(xab @ xab)
            if not rr < 2.0 * h[a]:
                continue
            gw = O.F(KID[kname], rr, h[a]) * xab / rr                    # gradient of W at a (A4)
            Vb = w.m[b] / w.rho_nom[b]
            M += Vb * np.outer(gw, -xab)                                 # eq. (40): rows dW/dx_i, columns x_ba
            grads.append((b, Vb, gw))
        L = np.linalg.inv(M)
        s = sum(Vb * (V[a] - V[b]) @ (L @ gw) for b, Vb, gw in grads)    # eq. (37) with eq. (39)
        assert np.allclose(r["M"][a], M, rtol=1e-12, atol=1e-14)
        assert np.allclose(r["L"][a], L, rtol=1e-9, atol=1e-12 * np.abs(L).max())
        assert r["drhodt"][a] == pytest.approx(w.rho_nom[a] * s, rel=1e-9, abs=1e-12 * np.abs(L).max() ** 2)


def test_rotating_the_whole_problem_leaves_drhodt_unchanged():
    """Eq. (37) with eq. (39) is a scalar: rotate positions and velocities by Q (about the box centre, open box) and
    drho/dt is the same while M -> Q M Q^T."""
    w = W.random_cloud(1200, seed=14, periodic=(0, 0, 0), hvar=2.0, box=(0.5, 0.5, 0.5))
    th = 0.7
    Q = np.array([[math.cos(th), -math.sin(th), 0.0], [math.sin(th), math.cos(th), 0.0], [0.0, 0.0, 1.0]]) @ \
        np.array([[1.0, 0.0, 0.0], [0.0, math.cos(0.4), -math.sin(0.4)], [0.0, math.sin(0.4), math.cos(0.4)]])
    X = np.stack([w.x, w.y, w.z], 1) - 0.25
    V = np.stack([w.vx, w.vy, w.vz], 1)
    Xr, Vr = X @ Q.T + 0.5, V @ Q.T
    r0 = O.kgc_continuity(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, w.vx, w.vy, w.vz)
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (3, 3, 3), (0, 0, 0), w.grid.h_max)
    r1 = O.kgc_continuity(g, w.kernel, Xr[:, 0], Xr[:, 1], Xr[:, 2], w.h, w.m, w.rho_nom, Vr[:, 0], Vr[:, 1], Vr[:, 2])
    reg = np.abs(np.linalg.det(r0["M"])) > 1e-4
    lnorm = np.linalg.norm(r0["L"].reshape(-1, 9), axis=1)
    scale = w.rho_nom * lnorm * np.linalg.norm(r0["S_N"].reshape(-1, 9), axis=1) * (1 + lnorm * np.linalg.norm(r0["S_M"].reshape(-1, 9), axis=1))
    assert np.all(np.abs(r0["drhodt"] - r1["drhodt"])[reg] <= 1e-10 * scale[reg])
    assert np.allclose(np.einsum("ij,njk,lk->nil", Q, r0["M"], Q), r1["M"], rtol=0, atol=1e-12)


def test_singular_moment_matrix_leaves_the_gradient_uncorrected():
    """Reading A28: a particle without neighbours, or with collinear neighbours only (rank-1 M), gets L = I and the plain
    eq. (37)."""
    h = 0.1
    x = np.array([0.2, 0.2 + h, 0.8]); y = np.array([0.5, 0.5, 0.5]); z = np.array([0.5, 0.5, 0.5])
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (4, 4, 4), (0, 0, 0), h)
    m = np.full(3, 0.02); rho = np.full(3, 1.5)
    vx = np.array([1.0, -1.0, 0.3]); vz = np.zeros(3)
    r = O.kgc_continuity(g, O.WENDLAND_C2, x, y, z, np.full(3, h), m, rho, vx, vz, vz)
    assert np.all(r["L"] == np.eye(3))
    assert r["drhodt"][2] == 0.0 and np.all(r["M"][2] == 0.0)
    # two approaching particles: drho/dt = rho V (v_a - v_b) F(q=1) (x_ab/r) > 0 (compression), closed form F(q=1)
    F1 = -105.0 / (128.0 * math.pi * h ** 4)
    assert r["drhodt"][0] == pytest.approx(1.5 * (0.02 / 1.5) * 2.0 * F1 * (-1.0), rel=1e-13)
    assert r["drhodt"][0] > 0 and r["drhodt"][0] == r["drhodt_raw"][0]
