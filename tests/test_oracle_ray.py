"""Pins of the N4 oracle (mesh-free laser ray tracing and deposition, section 2.5):
oracle.ray_deposit.  f = n_e/n_c, kib = absorption coefficient per particle (inputs)."""
import math

import numpy as np
import pytest

import oracle as O
import workloads as W
from test_oracle_pins import KID, golden, lattice_block


def rays_of(x0, v0, P0):
    x0 = np.atleast_2d(x0); v0 = np.atleast_2d(v0)
    return np.vstack([x0.T, v0.T, np.atleast_1d(P0)[None, :]])


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
@pytest.mark.parametrize("hfac", [1.2, 1.3])
def test_uniform_medium_straight_ray_and_exponential_attenuation(kname, hfac):
    """Periodic lattice, uniform f and kib: the gradient of P:L420 vanishes by symmetry, so the ray is straight; with steps of
    one lattice spacing from a lattice point the interpolated absorption coefficient is kib S0 at every step (S0 = lattice
    constant of the kernel, tests/golden/lattice_constants.txt), so eq. (71) gives P_K = P_0 exp(-kib S0 K ds) exactly."""
    s0, _ = golden()[(kname, hfac)]
    n, dx = 10, 0.1
    x, y, z, h, g = lattice_block(n, dx, True, hfac)
    rho = np.full(x.size, 2.0); m = rho * dx ** 3
    f = np.full(x.size, 0.3); kib = np.full(x.size, 1.7)
    c, K = 1.0, 6
    dt = dx / c
    r = O.ray_deposit(g, KID[kname], x, y, z, h, m, rho, f, kib, rays_of([0.25, 0.35, 0.45], [c, 0.0, 0.0], 2.5), dt, K, c)
    assert np.max(np.abs(r["gradn"])) < 1e-12
    assert np.allclose(r["rays"][3:6, 0], [c, 0.0, 0.0], atol=1e-13)
    assert r["rays"][0, 0] == pytest.approx(0.25 + K * dx, abs=1e-12)
    assert r["rays"][6, 0] == pytest.approx(2.5 * math.exp(-1.7 * s0 * K * dx), rel=1e-12)
    assert np.sum(r["edep"]) + r["rays"][6, 0] == pytest.approx(2.5, rel=1e-14)
    assert r["steps"][0] == K


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
def test_linear_density_gradient_bends_the_ray_by_eq_72(kname):
    """f = f0 + g.x on an open lattice block: interior particles get G_a = S2 g (the lattice constant of pins T6/T7, sum of the
    printed form, whose constant part cancels by symmetry), interpolated at a lattice point G = S0 S2 g, so after one step
    v_1 = v_0 - (c^2/2) S0 S2 g dt and x_1 = x_0 + v_1 dt exactly; over several steps the ray follows the parabola of a
    constant acceleration -(c^2/2) g within the lattice error of the kernel."""
    hfac = 1.2
    s0, s2 = golden()[(kname, hfac)]
    n, dx = 17, 0.1
    x, y, z, h, g = lattice_block(n, dx, False, hfac)
    gvec = np.array([0.0, 0.8, -0.3])
    f = 0.2 + np.stack([x, y, z], 1) @ gvec
    rho = np.full(x.size, 2.0); m = rho * dx ** 3
    kib = np.zeros(x.size)
    c = 1.0
    x0 = np.array([6.5, 8.5, 8.5]) * dx                                   # a lattice point, > 5.2 dx from every face
    dt = 0.05 * dx / c
    r1 = O.ray_deposit(g, KID[kname], x, y, z, h, m, rho, f, kib, rays_of(x0, [c, 0.0, 0.0], 1.0), dt, 1, c)
    centre = int(6 + 8 * n + 8 * n * n)
    assert np.allclose(r1["gradn"][:, centre], s2 * gvec, rtol=1e-12, atol=1e-13)
    v1 = np.array([c, 0.0, 0.0]) - 0.5 * c * c * s0 * s2 * gvec * dt
    assert np.allclose(r1["rays"][3:6, 0], v1, rtol=1e-12, atol=1e-15)
    assert np.allclose(r1["rays"][0:3, 0], x0 + v1 * dt, rtol=1e-13)
    K = 40                                                                # 2 lattice spacings along x
    rK = O.ray_deposit(g, KID[kname], x, y, z, h, m, rho, f, kib, rays_of(x0, [c, 0.0, 0.0], 1.0), dt, K, c)
    a = -0.5 * c * c * gvec
    xK = x0 + np.array([c, 0.0, 0.0]) * K * dt + a * dt * dt * K * (K + 1) / 2.0     # semi-implicit Euler, constant acceleration
    dev = rK["rays"][0:3, 0] - (x0 + np.array([c, 0, 0]) * K * dt)
    assert np.allclose(dev[1:], (xK - x0)[1:], rtol=0.03)
    assert dev[1] < 0 < dev[2]                                            # bends away from increasing electron density
    assert rK["rays"][6, 0] == 1.0 and np.all(rK["edep"] == 0.0)          # no absorber


def test_energy_is_conserved_and_rays_stop():
    """Whatever the rays do, sum(edep) + sum(P_final) = sum(P_0) (the weights are normalised, A33); a ray leaving the open box
    stops there, a ray below pmin stops, a ray through empty space loses nothing."""
    w = W.random_cloud(1500, seed=21, periodic=(0, 1, 1), hvar=1.5)
    f = 0.5 * w.x + 0.05 * w.E
    kib = 20.0 * (0.2 + w.kappa / np.max(w.kappa))
    i = np.arange(12)
    x0 = np.stack([np.full(12, 0.02), 0.1 + 0.07 * i, 0.9 - 0.06 * i], 1)
    v0 = np.stack([np.ones(12), 0.1 * np.sin(i), 0.1 * np.cos(i)], 1)
    P0 = 1.0 + 0.1 * i
    r = O.ray_deposit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, f, kib, rays_of(x0, v0, P0), 0.01, 400, 1.0)
    assert np.sum(r["edep"]) + np.sum(r["rays"][6]) == pytest.approx(np.sum(P0), rel=1e-13)
    assert np.all(r["edep"] >= 0.0) and np.sum(r["edep"]) > 0.5 * np.sum(P0)
    assert np.all(r["steps"] < 400)                                       # every ray left through an x face
    out = (r["rays"][0] < 0.0) | (r["rays"][0] >= 1.0)
    assert out.all()
    assert np.all((r["rays"][1] >= 0) & (r["rays"][1] < 1) & (r["rays"][2] >= 0) & (r["rays"][2] < 1))   # periodic y, z wrap
    rp = O.ray_deposit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, f, kib, rays_of(x0, v0, P0), 0.01, 400, 1.0, pmin=0.5)
    assert np.all(rp["rays"][6] <= np.maximum(0.5, r["rays"][6]) + 1e-15) and np.all(rp["steps"] <= r["steps"])
    # empty space: particles only in x < 0.5, ray far from them
    keep = w.x < 0.3
    re = O.ray_deposit(w.grid, w.kernel, w.x[keep], w.y[keep], w.z[keep], w.h[keep], w.m[keep], w.rho_nom[keep], f[keep], kib[keep],
                       rays_of([0.6, 0.5, 0.5], [1.0, 0.0, 0.0], 3.0), 0.01, 100, 1.0)
    assert re["rays"][6, 0] == 3.0 and np.all(re["edep"] == 0.0) and re["steps"][0] == 40


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
def test_single_particle_closed_form(kname):
    """One particle, one step starting at distance h from it: kappa(x) = V kib W(h; h), all of dE = P (1 - exp(-kappa ds)) goes to
    that particle; W(q = 1) = 1/(4 pi h^3) (cubic spline) or 63/(256 pi h^3) (Wendland C2, eq. (3): 21/(16 pi) (1/2)^4 3)."""
    h, m, rho, kib = 0.1, 0.02, 1.5, 40.0
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (4, 4, 4), (0, 0, 0), h)
    one = lambda v: np.array([v])
    r = O.ray_deposit(g, KID[kname], one(0.5), one(0.5), one(0.5), one(h), one(m), one(rho), one(0.3), one(kib),
                      rays_of([0.5 - h, 0.5, 0.5], [2.0, 0.0, 0.0], 7.0), 0.01, 1, 2.0)
    W1 = 1.0 / (4.0 * math.pi * h ** 3) if kname == "cubic" else 63.0 / (256.0 * math.pi * h ** 3)
    dE = 7.0 * (1.0 - math.exp(-(m / rho) * kib * W1 * 2.0 * 0.01))
    assert r["edep"][0] == pytest.approx(dE, rel=1e-13)
    assert r["rays"][6, 0] == pytest.approx(7.0 - dE, rel=1e-14)
    assert np.all(r["gradn"] == 0.0) and np.allclose(r["rays"][3:6, 0], [2.0, 0.0, 0.0])


@pytest.mark.parametrize("kname", ["cubic", "wendland"])
def test_brute_force_on_a_tiny_cloud(kname):
    """The scheme of P:L418-L422 written out in Python over all particles (W and F from the pinned scalar kernel functions):
    gradient at the particles, interpolation at the ray, eq. (72), eq. (71), kernel-weighted deposition."""
    n = 60
    w = W.random_cloud(n, seed=23, kernel=KID[kname], periodic=(0, 0, 0), hvar=1.5)
    h = 1.5 * w.h
    g = W.Grid((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (1, 1, 1), (0, 0, 0), float(h.max()))
    f = 0.3 + 0.4 * w.x * w.y + 0.2 * w.z
    kib = 5.0 + 10.0 * w.kappa / np.max(w.kappa)
    V = w.m / w.rho_nom
    X = np.stack([w.x, w.y, w.z], 1)
    rays = rays_of([[0.1, 0.4, 0.5], [0.9, 0.6, 0.3]], [[1.0, 0.1, 0.0], [-0.8, 0.0, 0.3]], [1.0, 2.0])
    dt, K, c = 0.02, 12, 1.3
    r = O.ray_deposit(g, KID[kname], w.x, w.y, w.z, h, w.m, w.rho_nom, f, kib, rays, dt, K, c)
    G = np.zeros((n, 3))
    for a in range(n):
        for b in range(n):
            d = X[a] - X[b]; rr = math.sqrt(d @ d)
            if b != a and rr < 2 * h[a]:
                G[a] += V[b] * f[b] * O.F(KID[kname], rr, h[a]) * d / rr
    assert np.allclose(r["gradn"].T, G, rtol=1e-12, atol=1e-13)
    edep = np.zeros(n)
    for q in range(2):
        p, v, P = rays[0:3, q].copy(), rays[3:6, q].copy(), rays[6, q]
        for _ in range(K):
            wgt = np.array([V[a] * O.W(KID[kname], math.sqrt((p - X[a]) @ (p - X[a])), h[a])
                            if (p - X[a]) @ (p - X[a]) < 4 * h[a] ** 2 else 0.0 for a in range(n)])
            v = v - 0.5 * c * c * (wgt @ G) * dt
            ds = math.sqrt(v @ v) * dt
            if wgt.sum() > 0:
                dE = P * (1.0 - math.exp(-(wgt @ kib) * ds))
                P -= dE
                edep += dE * wgt / wgt.sum()
            p = p + v * dt
            if np.any(p < 0) or np.any(p >= 1):
                break
        assert np.allclose(r["rays"][0:3, q], p, rtol=1e-12) and np.allclose(r["rays"][3:6, q], v, rtol=1e-12)
        assert r["rays"][6, q] == pytest.approx(P, rel=1e-12)
    assert np.allclose(r["edep"], edep, rtol=1e-11, atol=1e-16)
    assert np.sum(edep) > 0.01


def test_periodic_wrap_equals_translated_problem():
    """A ray crossing a periodic face continues on the other side: shifting particles and ray by half a box along the periodic
    direction (mod L) changes nothing but the coordinates."""
    w = W.random_cloud(1200, seed=25, periodic=(1, 1, 1), hvar=1.4)
    f = 0.3 + 0.2 * np.sin(2 * np.pi * w.x) * np.cos(2 * np.pi * w.z)
    kib = np.full(w.n, 3.0)
    rays = rays_of([[0.9, 0.5, 0.2]], [[1.0, 0.2, 0.1]], [1.0])
    a = O.ray_deposit(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, f, kib, rays, 0.01, 50, 1.0)
    xs = (w.x + 0.5) % 1.0
    rays2 = rays.copy(); rays2[0] = (rays2[0] + 0.5) % 1.0
    b = O.ray_deposit(w.grid, w.kernel, xs, w.y, w.z, w.h, w.m, w.rho_nom, f, kib, rays2, 0.01, 50, 1.0)
    assert np.allclose(a["edep"], b["edep"], rtol=1e-9, atol=1e-15)
    assert (a["rays"][0, 0] + 0.5) % 1.0 == pytest.approx(b["rays"][0, 0], abs=1e-10)
    assert np.allclose(a["rays"][1:, 0], b["rays"][1:, 0], rtol=1e-9, atol=1e-12)
    assert a["steps"][0] == 50 and 0.0 <= a["rays"][0, 0] < 1.0
