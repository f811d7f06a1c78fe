"""Pins of the N1 oracle (implicit radiation step, section 2.3, eqs. (47)-(60)): oracle.quartic_positive_root,
oracle.quartic_roots, oracle.rad_jacobi.  Every pin is something the paper or the mathematics fixes, not a re-typing of
the oracle's own formula."""
import numpy as np

import oracle as O
import workloads as W

GAMMA = 5.0 / 3.0


def small(nside=8):
    w = W.config1(nside=nside)
    T = (GAMMA - 1.0) * (w.p / ((GAMMA - 1.0) * w.rho_nom))      # T = (gamma - 1) u
    return w, T


def setup(w, T, dt=0.05, c=1.0, a=1.0, kp=None):
    u = T / (GAMMA - 1.0)
    mu = c / (3.0 * w.rho_nom * w.kappa)                          # lambda = 1/3 (optically thick limit)
    kp = np.full(w.n, 2.0) if kp is None else kp
    dTdu = np.full(w.n, GAMMA - 1.0)
    return dict(mu=mu, kappa_p=kp, u_n=u, T_n=T, dTdu=dTdu, dt=dt, c_light=c, a_rad=a)


def run(w, E_n, s, niter, **kw):
    return O.rad_jacobi(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, s["mu"], s["kappa_p"], E_n, s["u_n"], s["T_n"],
                        s["dTdu"], s["dt"], s["c_light"], s["a_rad"], niter, **kw)


def test_quartic_root_substitution():
    """eq. (57) as x^4 + b x + c = 0: the root substituted back vanishes to rounding over 14 decades of (b, c)."""
    rng = np.random.default_rng(7)
    b = 10.0 ** rng.uniform(-6, 8, 200000)
    c = -(10.0 ** rng.uniform(-8, 8, 200000))
    x = O.quartic_positive_root(b, c)
    assert (x > 0).all()
    res = np.abs(x ** 4 + b * x + c) / (x ** 4 + b * x - c)
    assert res.max() < 1e-15 * 8


def test_quartic_limits():
    """b -> 0: x = (-c)^(1/4); c -> 0-: x = -c/b (textbook limits of the depressed quartic)."""
    x = O.quartic_positive_root(np.array([1e-30]), np.array([-16.0]))
    assert abs(x[0] - 2.0) < 1e-14
    x = O.quartic_positive_root(np.array([5.0]), np.array([-1e-12]))
    assert abs(x[0] - 2e-13) < 1e-27


def test_closed_form_agrees_where_well_conditioned():
    """eqs. (58)-(60) with the sign pairing (-, +) give the same positive root; the pairing (-, -) gives the negative one."""
    rng = np.random.default_rng(11)
    b = rng.uniform(0.5, 2.0, 5000)
    c = -rng.uniform(0.5, 2.0, 5000)
    xp, xm = O.quartic_roots(b, c)
    x = O.quartic_positive_root(b, c)
    assert np.max(np.abs(xp - x) / x) < 1e-12
    assert (xm < 0).all()
    assert np.max(np.abs(xm ** 4 + b * xm + c)) < 1e-12           # also a root
    # Vieta: the four roots sum to 0 and the two complex ones have real part s/2 = -(xp + xm)/2; product of all = c
    s = -(xp + xm)
    y = 0.5 * s * s
    quad2_const = y + b / (2.0 * s)                               # x^2 - s x + (y + b/(2s)): product of the complex pair
    assert np.max(np.abs(xp * xm * quad2_const - c) / np.abs(c)) < 1e-11


def test_equilibrium_is_stationary():
    """E = a T^4 uniform and T uniform: diffusion and exchange both vanish, chi = T^n solves eq. (57) exactly."""
    w, _ = small()
    T = np.full(w.n, 0.8)
    s = setup(w, T, a=1.3)
    E_n = 1.3 * T ** 4
    r = run(w, E_n, s, 3)
    assert np.max(np.abs(r["E"] - E_n) / E_n) < 1e-12
    assert np.max(np.abs(r["u"] - s["u_n"]) / s["u_n"]) < 1e-12


def test_pure_exchange_conserves_energy_per_particle():
    """mu -> 0 switches the diffusion off: eqs. (49)+(50) give E' + rho u' = E + rho u for every particle, for ANY iterate."""
    w, T = small()
    s = setup(w, T)
    s["mu"] = np.full(w.n, 1e-300)
    r = run(w, w.E, s, 2)
    lhs = r["E"] + w.rho_nom * r["u"]
    rhs = w.E + w.rho_nom * s["u_n"]
    assert np.max(np.abs(lhs - rhs) / rhs) < 1e-13
    # and the fixed point of eq. (50): u' - u = dt c kappa (E' - a T'^4), T' = T + dT/du (u' - u)
    Tp = s["T_n"] + s["dTdu"] * (r["u"] - s["u_n"])
    assert np.max(np.abs((r["u"] - s["u_n"]) - s["dt"] * s["c_light"] * s["kappa_p"] * (r["E"] - s["a_rad"] * Tp ** 4))) < 1e-13


def test_small_dt_limit():
    """dt -> 0: the step changes nothing to first order in dt."""
    w, T = small()
    s = setup(w, T, dt=1e-9)
    r = run(w, w.E, s, 3)
    assert np.max(np.abs(r["E"] - w.E) / w.E) < 1e-6
    assert np.max(np.abs(r["u"] - s["u_n"]) / s["u_n"]) < 1e-6


def test_converged_step_satisfies_eqs_49_50_and_conserves_total_energy():
    """Iterate to convergence; then eq. (49) holds with an INDEPENDENT evaluation of the operator on E^{n+1} (fld_apply's
    difference-form y), eq. (50) holds, and sum_a [V_a dE_a + m_a du_a] = dt sum_a V_a y_a = 0 (conservative operator, T11)."""
    w, T = small()
    s = setup(w, T, dt=0.02)
    r = run(w, w.E, s, 60)
    assert r["resid"][-1] < 1e-12 and r["resid"][1] > r["resid"][-1]
    ap = O.fld_apply(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, s["mu"], r["E"], sym_mode=True)
    Tp = s["T_n"] + s["dTdu"] * (r["u"] - s["u_n"])
    UP = s["a_rad"] * Tp ** 4
    X = s["dt"] * w.rho_nom * s["c_light"] * s["kappa_p"]
    r49 = r["E"] - (w.E + s["dt"] * ap["y"] + X * (UP - r["E"]))
    assert np.max(np.abs(r49) / r["E"]) < 1e-11
    r50 = (r["u"] - s["u_n"]) - s["dt"] * s["c_light"] * s["kappa_p"] * (r["E"] - UP)
    assert np.max(np.abs(r50) / s["u_n"]) < 1e-12
    V = w.m / w.rho_nom
    tot = np.sum(V * (r["E"] - w.E) + w.m * (r["u"] - s["u_n"]))
    scale = np.sum(np.abs(V * (r["E"] - w.E)) + np.abs(w.m * (r["u"] - s["u_n"])))
    assert abs(tot) / scale < 1e-10
