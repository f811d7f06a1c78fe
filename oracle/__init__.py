"""CPU oracle for the SPRAY pair-summation pass -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over ``oracle/spray_oracle.c`` (plain C, fp64, long-double accumulation,
written from PAPER.md; see the header of that file for citations and the pin list).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2604_20124_b200`` and shares no
code with it.

Parity unpinned: the A6 reading (viscosity only for w < 0) -- see ``spray_oracle.c`` header.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "spray_oracle.c"
_LIB = _HERE / "liboracle.so"

GATHER, SYM = 0, 1
CUBIC_SPLINE, WENDLAND_C2 = 0, 1


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2 -ffp-contract=off -fopenmp).  Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3), ("ncell", C.c_int32 * 3),
                ("periodic", C.c_int32 * 3), ("h_max", C.c_double)]


def _grid(g) -> _Grid:
    return _Grid((C.c_double * 3)(*g.lo), (C.c_double * 3)(*g.hi), (C.c_int32 * 3)(*g.ncell),
                 (C.c_int32 * 3)(*g.periodic), float(g.h_max))


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.oracle_W.restype = C.c_double
        _lib.oracle_W.argtypes = [C.c_int, C.c_double, C.c_double]
        _lib.oracle_F.restype = C.c_double
        _lib.oracle_F.argtypes = [C.c_int, C.c_double, C.c_double]
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(n: int) -> None:
    """OpenMP threads of the calls that follow (timing harness: single-thread and all-core oracle timings)."""
    lib().oracle_set_threads(int(n))


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.c_void_p)


def _targets(targets, n):
    if targets is None:
        return None, C.c_void_p(None), n
    t = np.ascontiguousarray(targets, dtype=np.int64)
    return t, t.ctypes.data_as(C.c_void_p), t.size


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def W(kernel: int, r: float, h: float) -> float:
    return lib().oracle_W(int(kernel), float(r), float(h))


def F(kernel: int, r: float, h: float) -> float:
    return lib().oracle_F(int(kernel), float(r), float(h))


def build_cells(grid, x, y, z):
    """O1.  Returns dict(key, sorted_key, perm, cell_start, cell_end), all uint32."""
    n = len(x)
    (x, px), (y, py), (z, pz) = _d(x), _d(y), _d(z)
    nc = grid.ncell_total
    key = np.zeros(n, np.uint32); sk = np.zeros(n, np.uint32); perm = np.zeros(n, np.uint32)
    cs = np.zeros(nc, np.uint32); ce = np.zeros(nc, np.uint32)
    g = _grid(grid)
    rc = lib().oracle_build_cells(C.byref(g), C.c_int64(n), px, py, pz, _p(key), _p(sk), _p(perm), _p(cs), _p(ce))
    assert rc == 0
    return dict(key=key, sorted_key=sk, perm=perm, cell_start=cs, cell_end=ce)


def neighbor_counts(grid, x, y, z, h, mode, use_cells=True, targets=None):
    n = len(x)
    (x, px), (y, py), (z, pz), (h, ph) = _d(x), _d(y), _d(z), _d(h)
    t, pt, nt = _targets(targets, n)
    cnt = np.zeros(nt, np.uint32)
    g = _grid(grid)
    rc = lib().oracle_neighbor_counts(C.byref(g), C.c_int64(n), px, py, pz, ph, int(use_cells), int(mode), pt,
                                      C.c_int64(nt), _p(cnt))
    assert rc == 0
    return cnt


def neighbor_lists(grid, x, y, z, h, mode, use_cells=True, targets=None):
    """Returns (offsets[nt+1] uint64, nbr uint32): ascending caller ids per target, self excluded."""
    n = len(x)
    cnt = neighbor_counts(grid, x, y, z, h, mode, use_cells, targets)
    off = np.zeros(cnt.size + 1, np.uint64)
    np.cumsum(cnt, out=off[1:])
    (x, px), (y, py), (z, pz), (h, ph) = _d(x), _d(y), _d(z), _d(h)
    t, pt, nt = _targets(targets, n)
    nbr = np.zeros(max(int(off[-1]), 1), np.uint32)
    g = _grid(grid)
    rc = lib().oracle_neighbor_lists(C.byref(g), C.c_int64(n), px, py, pz, ph, int(use_cells), int(mode), pt,
                                     C.c_int64(nt), _p(off), _p(nbr))
    assert rc == 0
    return off, nbr[: int(off[-1])]


def neighbor_digest(grid, x, y, z, h, mode, use_cells=True):
    """Full-population (count uint32, sum uint64, xor uint64) of splitmix64(caller id) over each particle's neighbour set
    (self excluded); SYM is built from the gather sets by transposition (see oracle_neighbor_digest)."""
    n = len(x)
    (x, px), (y, py), (z, pz), (h, ph) = _d(x), _d(y), _d(z), _d(h)
    cnt = np.zeros(n, np.uint32); ds = np.zeros(n, np.uint64); dx = np.zeros(n, np.uint64)
    g = _grid(grid)
    rc = lib().oracle_neighbor_digest(C.byref(g), C.c_int64(n), px, py, pz, ph, int(use_cells), int(mode), _p(cnt), _p(ds), _p(dx))
    assert rc == 0
    return cnt, ds, dx


def density(grid, kernel, x, y, z, h, m, use_cells=True, targets=None):
    """O4, eq. (35).  Returns dict(rho, nnbr, S_rho) at the targets."""
    n = len(x)
    (x, px), (y, py), (z, pz), (h, ph), (m, pm) = _d(x), _d(y), _d(z), _d(h), _d(m)
    t, pt, nt = _targets(targets, n)
    rho = np.zeros(nt); nn = np.zeros(nt, np.uint32); S = np.zeros(nt)
    g = _grid(grid)
    rc = lib().oracle_density(C.byref(g), int(kernel), C.c_int64(n), px, py, pz, ph, pm, int(use_cells), pt,
                              C.c_int64(nt), _p(rho), _p(nn), _p(S))
    assert rc == 0
    return dict(rho=rho, nnbr=nn, S_rho=S)


def hydro(grid, kernel, x, y, z, h, m, rho, p, cs, vx, vy, vz, alpha, beta=2.0, use_cells=True, targets=None):
    """O5.  Returns dict(ax, ay, az, dudt, divv, S_ax, S_ay, S_az, S_dudt, S_divv) at the targets."""
    n = len(x)
    arrs = [_d(a) for a in (x, y, z, h, m, rho, p, cs, vx, vy, vz, alpha)]
    t, pt, nt = _targets(targets, n)
    out = {k: np.zeros(nt) for k in ("ax", "ay", "az", "dudt", "divv", "S_ax", "S_ay", "S_az", "S_dudt", "S_divv")}
    g = _grid(grid)
    rc = lib().oracle_hydro(C.byref(g), int(kernel), C.c_int64(n), *[a[1] for a in arrs], C.c_double(beta),
                            int(use_cells), pt, C.c_int64(nt), *[_p(out[k]) for k in
                            ("ax", "ay", "az", "dudt", "divv", "S_ax", "S_ay", "S_az", "S_dudt", "S_divv")])
    assert rc == 0
    return out


def limiter(grid, kernel, x, y, z, h, m, rho, kappa, E, c_light=1.0, use_cells=True, targets=None):
    """O6.  Returns dict(gx, gy, gz, R, lam, mu, S_gx, S_gy, S_gz) at the targets."""
    n = len(x)
    arrs = [_d(a) for a in (x, y, z, h, m, rho, kappa, E)]
    t, pt, nt = _targets(targets, n)
    keys = ("gx", "gy", "gz", "R", "lam", "mu", "S_gx", "S_gy", "S_gz")
    out = {k: np.zeros(nt) for k in keys}
    g = _grid(grid)
    rc = lib().oracle_limiter(C.byref(g), int(kernel), C.c_int64(n), *[a[1] for a in arrs], C.c_double(c_light),
                              int(use_cells), pt, C.c_int64(nt), *[_p(out[k]) for k in keys])
    assert rc == 0
    return out


def fld_apply(grid, kernel, x, y, z, h, m, rho, mu, E, sym_mode=True, use_cells=True, targets=None):
    """O7.  Returns dict(y, diag, offd, S_y, S_diag, S_offd) at the targets."""
    n = len(x)
    arrs = [_d(a) for a in (x, y, z, h, m, rho, mu, E)]
    t, pt, nt = _targets(targets, n)
    keys = ("y", "diag", "offd", "S_y", "S_diag", "S_offd")
    out = {k: np.zeros(nt) for k in keys}
    g = _grid(grid)
    rc = lib().oracle_fld_apply(C.byref(g), int(kernel), C.c_int64(n), *[a[1] for a in arrs], int(bool(sym_mode)),
                                int(use_cells), pt, C.c_int64(nt), *[_p(out[k]) for k in keys])
    assert rc == 0
    return out


# ---------------------------------------------------------------------------------------------------------------
# Row N1 of SURVEY.md section 8(f): the implicit radiation step (section 2.3).
# Backward-Euler energy exchange + diffusion, eqs. (49)-(50), solved by Jacobi iteration: every iteration applies the
# FLD operator to the current iterate (eqs. (51)-(52): Lambda, Gamma), then solves the per-particle quartic eq. (57)
# for chi (eq. (56)) in closed form (eqs. (58)-(60)) and updates E by eq. (55) and u by eq. (56).
# TEST INFRASTRUCTURE like the rest of oracle/: plain numpy fp64 on top of fld_apply, no code shared with the CUDA path.
# Readings (A25 ff.): the limiter is frozen during the iteration (mu is an input, A18); the resolvent
# cubic of x^4 + b x + c = 0 is y^3 + p y + q = 0 with p = -c, q = -b^2/8, the factorisation is
# (x^2 + s x + y - b/(2s)) (x^2 - s x + y + b/(2s)), s = sqrt(2y), so the two real roots for b > 0, c < 0 are
# x = (-s +- sqrt(-2y + 2b/s)) / 2 (the sign pairing eq. (58) leaves open); "the root that yields a real value of u closest
# to u^n" is then the one closest to T^n, i.e. the positive one.  That root is computed by safeguarded Newton
# (quartic_positive_root) because the closed form is numerically unusable over part of the parameter range.

def quartic_roots(b, c):
    """Real roots of x^4 + b x + c = 0 for b > 0, c < 0 by eqs. (58)-(60): returns (x_plus, x_minus)."""
    b = np.asarray(b, dtype=np.float64); c = np.asarray(c, dtype=np.float64)
    p = -c
    q = -b * b / 8.0
    w = np.cbrt(-q / 2.0 + np.sqrt(q * q / 4.0 + p ** 3 / 27.0))          # eq. (60)
    y = w - p / (3.0 * w)                                                  # eq. (59)
    s = np.sqrt(2.0 * y)
    d = np.sqrt(-2.0 * y + 2.0 * b / s)
    return 0.5 * (-s + d), 0.5 * (-s - d)                                  # eq. (58)


def quartic_positive_root(b, c):
    """The unique positive root of x^4 + b x + c = 0 (b > 0, c < 0) to rounding: Newton's method from the upper bound
    min((-c)^(1/4), -c/b) (f is convex and increasing on x > 0, so the iterates decrease monotonically to the root).
    The closed form of eqs. (58)-(60) is the same number algebraically but cancels catastrophically when the root is
    small (relative residuals up to 0.4, even inf/nan, on a log-uniform sweep of (b, c)); it is kept as quartic_roots
    and pinned against this routine where it is well conditioned (tests/test_oracle_rad.py)."""
    b = np.asarray(b, dtype=np.float64); c = np.asarray(c, dtype=np.float64)
    x = np.minimum((-c) ** 0.25, -c / b)
    for _ in range(100):
        dx = (x ** 4 + b * x + c) / (4.0 * x ** 3 + b)
        x = x - dx
        if np.all(np.abs(dx) <= 4.0 * np.finfo(np.float64).eps * np.abs(x)):
            break
    return x


def rad_jacobi(grid, kernel, x, y, z, h, m, rho, mu, kappa_p, E_n, u_n, T_n, dTdu, dt, c_light, a_rad, niter,
               sym_mode=True, E0=None, targets=None):
    """niter Jacobi iterations of eqs. (49)-(50) from the iterate E0 (default E_n).  Returns dict(E, u, chi, resid[niter],
    S_offd): resid[k] = max_a |lhs - rhs| / |lhs| of eq. (49) for the iterate that ENTERS iteration k, 0 for k = 0.
    targets (niter = 1 only: the first iteration needs the operator at the targets alone) restricts the outputs to a sample."""
    E_full = np.asarray(E_n, np.float64) if E0 is None else np.asarray(E0, np.float64)
    rho_full = np.asarray(rho, np.float64)
    sel = slice(None)
    if targets is not None:
        assert niter == 1, "a sample of targets can only be followed for one iteration"
        sel = np.asarray(targets, np.int64)
    E_n = np.asarray(E_n, np.float64)[sel]; u_n = np.asarray(u_n, np.float64)[sel]; T_n = np.asarray(T_n, np.float64)[sel]
    rho = rho_full[sel]; kp = np.asarray(kappa_p, np.float64)[sel]; dTdu = np.asarray(dTdu, np.float64)[sel]
    E = E_full.copy() if targets is None else E_full
    u = u_n.copy()
    chi = T_n.copy()
    resid = np.zeros(niter)
    S_offd = None
    K = dt * c_light * kp                                                  # denominator of eq. (55)
    X = dt * rho * c_light * kp
    for k in range(niter):
        ap = fld_apply(grid, kernel, x, y, z, h, m, rho_full, mu, E, sym_mode=sym_mode, targets=targets)
        lam, gam, S_offd = ap["diag"], ap["offd"], ap["S_offd"]
        if k > 0:                                                          # both sides of eq. (49) for the current iterate
            rhs = E_n + dt * (lam * E + gam) + X * (a_rad * chi ** 4 - E)
            resid[k] = np.max(np.abs(E - rhs) / np.abs(E))
        D = 1.0 - dt * lam
        Bq = (D + X) / K / dTdu                                            # coefficient of chi in eq. (57)
        Aq = D * a_rad
        Cq = E_n + dt * gam + Bq * T_n
        # of the two real roots the positive one is the closer to T^n > 0: the other is negative
        chi = quartic_positive_root(Bq / Aq, -Cq / Aq)
        u = u_n + (chi - T_n) / dTdu                                       # eq. (56)
        E = (u - u_n) / K + a_rad * chi ** 4                               # eq. (55)
    return dict(E=E, u=u, chi=chi, resid=resid, S_offd=S_offd)


# ---------------------------------------------------------------------------------------------------------------
# Row N2: thermal-conduction term of eqs. (17)/(18) for one species:
#   dudt_a = sum_b 4 m_b/(rho_a rho_b) k_a k_b/(k_a+k_b) (T_a - T_b) x_ab . gradWbar / |x_ab|^2
# i.e. eq. (16) with c = k, f = T and the kernel gradient averaged over h_a, h_b, divided by rho_a.  The pair sum is
# the one oracle_fld_apply evaluates in its symmetric mode (same formula with mu = k, E = T), so it is called, not retyped.
def conduction(grid, kernel, x, y, z, h, m, rho, k, T, targets=None):
    """Returns dict(dudt, S_dudt) at the targets."""
    ap = fld_apply(grid, kernel, x, y, z, h, m, rho, k, T, sym_mode=True, targets=targets)
    r = np.asarray(rho, np.float64)
    r = r if targets is None else r[np.asarray(targets)]
    return dict(dudt=ap["y"] / r, S_dudt=ap["S_y"] / r)


# ---------------------------------------------------------------------------------------------------------------
# Row N2, second half: the implicit (backward-Euler) two-temperature heat-transport system of eqs. (26)-(34), P:L166-L192,
# as a MATRIX-FREE operator: cond_implicit returns the left-hand sides of eqs. (28)/(29) applied to a given (u^i, u^e) and the
# right-hand sides b^i + c, b^e - c of eqs. (33)/(34), assembled term by term in the paper's notation from the pair sums of
# oracle_fld_apply in its symmetric mode with mu = k^s (called, not retyped: with E = g it returns diag_a = sum_b c_ab and
# offd_a = -sum_b c_ab g_b, c_ab = (m_b/rho_b) 4 k_a k_b/(k_a+k_b) x_ab.gradWbar/|x_ab|^2, so that sum_b [4 m_b/(rho_a rho_b) ...] g_b =
# -offd_a/rho_a).  tau^s = dT^s/du^s.
#   Lambda^s_a = 1 - dt tau_a D_a + dt kei_a tau_a,  D_a = diag_a/rho_a                                  eq. (30)
#   sum_b chi^s_ab u_b = dt sum_b [..]_ab tau_b u_b = -dt offd_a[g = tau u]/rho_a                        eq. (31)
#   Gamma^s_a u_a = dt kei_a tau_a u_a                                                                  eq. (32)
#   b^s_a = u_a + dt sum_b [..]_ab [T_a - T_b - tau_a u_a + tau_b u_b] = u_a + dt y_a[g = T - tau u]/rho_a   eq. (33)
#   c_a = dt kei_a [T^e_a - T^i_a - tau^e_a u^e_a + tau^i_a u^i_a]                                       eq. (34)
#   lhs^i = Lambda^i u^i + sum_b chi^i_ab u^i_b - Gamma^e u^e                                            eq. (28)
#   lhs^e = Lambda^e u^e + sum_b chi^e_ab u^e_b - Gamma^i u^i                                            eq. (29), reading A37
# Reading A37: eq. (29) prints "+ Gamma^i u^i"; substituting T^{N+1} = T^N + tau (u^{N+1} - u^N) into eq. (27), whose
# exchange term is -k^ei (T^e - T^i), gives -Gamma^i u^i (the mirror image of eq. (28)); with the printed sign the exchange
# would not conserve energy.  Pinned by substitution into eqs. (26)/(27) and by energy conservation (tests/test_oracle_cond.py).
# Sign note: the paper's sums carry x_ab.gradWbar/|x_ab|^2 <= 0, and eqs. (26)/(27) are used exactly as printed (the same
# expression oracle.conduction evaluates for eqs. (17)/(18)).
def cond_implicit(grid, kernel, x, y, z, h, m, rho, k_i, k_e, kei, tau_i, tau_e, T_i, T_e, u_i, u_e, dt, targets=None):
    """Returns dict(lhs_i, lhs_e, rhs_i, rhs_e, S_i, S_e): lhs = operator of eqs. (28)/(29) applied to (u_i, u_e); rhs = b^i + c,
    b^e - c of eqs. (33)/(34) for (u, T) taken as the time-level-N state; S = sums of absolute contributions (parity normaliser).  `targets` (indices)
    restricts the rows that are evaluated (full-size sampled parity); the arithmetic of a row does not depend on it."""
    rho_all = np.asarray(rho, np.float64)
    sel = slice(None) if targets is None else np.asarray(targets, np.int64)
    rho = rho_all[sel]; kei = np.asarray(kei, np.float64)[sel]
    T_i, T_e, tau_i, tau_e, u_i, u_e = (np.asarray(a, np.float64) for a in (T_i, T_e, tau_i, tau_e, u_i, u_e))
    out = {}
    gam = {}
    S = {}
    for s, k, tau, T, u in (("i", k_i, tau_i, T_i, u_i), ("e", k_e, tau_e, T_e, u_e)):
        k = np.asarray(k, np.float64)
        a1 = fld_apply(grid, kernel, x, y, z, h, m, rho_all, k, tau * u, sym_mode=True, targets=targets)
        g2 = T - tau * u
        tau = tau[sel]; T = T[sel]; u = u[sel]
        D = a1["diag"] / rho
        Lam = 1.0 - dt * tau * D + dt * kei * tau                         # eq. (30)
        chi = -dt * a1["offd"] / rho                                      # eq. (31)
        gam[s] = dt * kei * tau * u                                       # eq. (32)
        a2 = fld_apply(grid, kernel, x, y, z, h, m, rho_all, k, g2, sym_mode=True, targets=targets)
        out["b_" + s] = u + dt * a2["y"] / rho                            # eq. (33)
        out["lu_" + s] = Lam * u + chi
        S[s] = np.abs(u) + dt * (a1["S_y"] + a2["S_y"] + a1["S_offd"]) / rho + dt * kei * (np.abs(tau * u) + np.abs(T))
    T_i, T_e, tau_i, tau_e, u_i, u_e = T_i[sel], T_e[sel], tau_i[sel], tau_e[sel], u_i[sel], u_e[sel]
    c = dt * kei * (T_e - T_i - tau_e * u_e + tau_i * u_i)   # eq. (34)
    Sx = dt * kei * (np.abs(T_e) + np.abs(T_i) + np.abs(tau_e * u_e) + np.abs(tau_i * u_i))
    return dict(lhs_i=out["lu_i"] - gam["e"], lhs_e=out["lu_e"] - gam["i"],          # eqs. (28), (29) (A37)
                rhs_i=out["b_i"] + c, rhs_e=out["b_e"] - c, S_i=S["i"] + Sx, S_e=S["e"] + Sx)


# ---------------------------------------------------------------------------------------------------------------
# Row N3: continuity equation eq. (37) with the kernel-gradient-correction filter of eqs. (39)-(40),
# oracle_kgc_continuity in spray_oracle.c.  Reading A28: where the moment matrix is singular (|det| <= 1e-12) L = I.
def kgc_continuity(grid, kernel, x, y, z, h, m, rho, vx, vy, vz, use_cells=True, targets=None):
    """Returns dict(drhodt, drhodt_raw, M, L, S_M, S_N) at the targets; M, L, S_M, S_N have shape (nt, 3, 3)."""
    n = len(x)
    (x, px), (y, py), (z, pz), (h, ph), (m, pm), (rho, pr) = _d(x), _d(y), _d(z), _d(h), _d(m), _d(rho)
    (vx, pvx), (vy, pvy), (vz, pvz) = _d(vx), _d(vy), _d(vz)
    t, pt, nt = _targets(targets, n)
    out = {k: np.zeros(nt) for k in ("drhodt", "drhodt_raw")}
    mats = {k: np.zeros((nt, 3, 3)) for k in ("M", "L", "S_M", "S_N")}
    g = _grid(grid)
    rc = lib().oracle_kgc_continuity(C.byref(g), int(kernel), C.c_int64(n), px, py, pz, ph, pm, pr, pvx, pvy, pvz,
                                     int(use_cells), pt, C.c_int64(nt), _p(out["drhodt"]), _p(out["drhodt_raw"]),
                                     _p(mats["M"]), _p(mats["L"]), _p(mats["S_M"]), _p(mats["S_N"]))
    assert rc == 0
    out.update(mats)
    return out


# ---------------------------------------------------------------------------------------------------------------
# Row N4: mesh-free laser ray tracing and inverse-bremsstrahlung deposition, section 2.5:
# oracle_ray_deposit in spray_oracle.c (readings A29-A35 of DESIGN.md in its header).
def ray_deposit(grid, kernel, x, y, z, h, m, rho, f, kib, rays, dt, nsteps, c_light=1.0, pmin=0.0, use_cells=True):
    """rays: array (7, nrays) with rows x, y, z, vx, vy, vz, P.  Returns dict(gradn (3, n), edep (n), rays (7, nrays), steps,
    S_gradn (3, n): sums of the absolute pair contributions to gradn, the parity normaliser)."""
    n = len(x)
    (x, px), (y, py), (z, pz), (h, ph), (m, pm), (rho, pr), (f, pf), (kib, pk) = (_d(a) for a in (x, y, z, h, m, rho, f, kib))
    rays = np.ascontiguousarray(rays, dtype=np.float64)
    assert rays.ndim == 2 and rays.shape[0] == 7
    nr = rays.shape[1]
    gradn = np.zeros((3, n)); edep = np.zeros(n); rout = np.zeros((7, nr)); steps = np.zeros(nr, np.int64); S = np.zeros((3, n))
    g = _grid(grid)
    rc = lib().oracle_ray_deposit(C.byref(g), int(kernel), C.c_int64(n), px, py, pz, ph, pm, pr, pf, pk, int(use_cells),
                                  C.c_int64(nr), _p(rays), C.c_double(dt), C.c_int64(nsteps), C.c_double(c_light),
                                  C.c_double(pmin), _p(gradn), _p(edep), _p(rout), _p(steps), _p(S))
    assert rc == 0
    return dict(gradn=gradn, edep=edep, rays=rout, steps=steps, S_gradn=S)
