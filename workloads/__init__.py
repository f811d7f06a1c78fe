"""Seeded synthetic SPH particle sets shaped like the paper's workloads.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2604_20124_b200/``).  It holds none of the method's arithmetic: no
kernel function, no neighbour search, no SPH sum.  It only lays particles out and
fills per-particle input fields (positions, h, m, u, v, and the caller-side
EOS/opacity fields p, c_s, E, kappa that the pass takes as *inputs*,
SURVEY.md §8(c2) A9/A10/A22).

Recipes follow BASELINE.json ``configs`` as concretised in SURVEY.md §8(d); the
workload shapes stand in for the paper's cases (Sod Table 1, PAPER.md L488-L493;
laser-irradiated slab with exponential corona, L335/L369; Rayleigh-Taylor
interface, L527-L531).  None of the paper's data sets exist here.

RNG: counter-based, ``u01(seed, i, ch) = (splitmix64(seed ^ (i*K1 + ch*K2)) >> 11) * 2**-53``
so any particle/channel can be regenerated independently and reproducibly.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

K1 = np.uint64(0x9E3779B97F4A7C15)
K2 = np.uint64(0xD1B54A32D192ED03)
SEEDS = {1: 2604201241, 2: 2604201242, 3: 2604201243, 4: 2604201244, 5: 2604201245}

KERNEL_CUBIC_SPLINE = 0
KERNEL_WENDLAND_C2 = 1


def splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def u01(seed: int, i: np.ndarray, ch: int) -> np.ndarray:
    """Uniform [0,1) fp64 for particle counter(s) ``i`` and channel ``ch``."""
    i = np.asarray(i, dtype=np.uint64)
    with np.errstate(over="ignore"):
        ctr = np.uint64(seed) ^ (i * K1 + np.uint64(ch) * K2)
    return (splitmix64(ctr) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def normal(seed: int, i: np.ndarray, ch: int) -> np.ndarray:
    """Standard normal by Box-Muller from channels ``ch`` and ``ch+1``."""
    u1 = u01(seed, i, ch)
    u2 = u01(seed, i, ch + 1)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


@dataclass
class Grid:
    """Uniform cell grid handed to ``spray_build_cells`` / the oracle (an INPUT, A14)."""
    lo: tuple
    hi: tuple
    ncell: tuple
    periodic: tuple
    h_max: float

    @property
    def ncell_total(self) -> int:
        return int(self.ncell[0]) * int(self.ncell[1]) * int(self.ncell[2])


@dataclass
class Workload:
    name: str
    kernel: int
    grid: Grid
    gamma: float
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    h: np.ndarray
    m: np.ndarray
    rho_nom: np.ndarray   # the recipe's nominal density (input to isolated-sweep tests)
    u: np.ndarray
    p: np.ndarray         # (gamma-1) rho_nom u   -- caller-side EOS, an input array (A9/A10)
    cs: np.ndarray        # sqrt(gamma p / rho_nom)
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    alpha: np.ndarray
    E: np.ndarray
    kappa: np.ndarray
    beta: float = 2.0
    c_light: float = 1.0
    notes: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.x.shape[0])


def _wrap(x: np.ndarray, lo: float, hi: float) -> np.ndarray:
    """Fold into [lo, hi) (periodic dimension); guards the x == hi rounding case."""
    L = hi - lo
    x = lo + np.mod(x - lo, L)
    return np.where(x >= hi, lo, x)


def _uniform_grid(lo, hi, periodic, h, min_cells=1):
    """A14: uniform-h rule ncell_d = floor(L_d / (2h))."""
    nc = []
    for d in range(3):
        L = hi[d] - lo[d]
        nc.append(max(min_cells, int(math.floor(L / (2.0 * h) * (1.0 + 1e-12)))))
    return Grid(tuple(lo), tuple(hi), tuple(nc), tuple(periodic), float(h))


def _finish(name, kernel, grid, gamma, x, y, z, h, m, rho, u, vx, vy, vz, E, kappa, notes=None):
    n = x.shape[0]
    p = (gamma - 1.0) * rho * u
    cs = np.sqrt(gamma * p / rho)
    c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    return Workload(name, kernel, grid, gamma, c(x), c(y), c(z), c(h), c(m), c(rho), c(u), c(p), c(cs),
                    c(vx), c(vy), c(vz), np.ones(n), c(E), c(kappa), notes=notes or {})


def _lattice(nx, ny, nz):
    i = np.arange(nx * ny * nz, dtype=np.int64)
    ix = i % nx
    iy = (i // nx) % ny
    iz = i // (nx * ny)
    return i, ix, iy, iz


# --------------------------------------------------------------------------- config 1
def config1(nside: int = 16, seed: int = SEEDS[1], jitter: float = 0.05) -> Workload:
    """Periodic unit cube, nside^3 jittered lattice, cubic spline h = 1.2 dx (BJ config 1)."""
    dx = 1.0 / nside
    i, ix, iy, iz = _lattice(nside, nside, nside)
    n = i.size
    jit = lambda ch: (2.0 * u01(seed, i, ch) - 1.0) * jitter * dx
    x = _wrap((ix + 0.5) * dx + jit(0), 0.0, 1.0)
    y = _wrap((iy + 0.5) * dx + jit(1), 0.0, 1.0)
    z = _wrap((iz + 0.5) * dx + jit(2), 0.0, 1.0)
    h = np.full(n, 1.2 * dx)
    m = np.full(n, 1.0 / n)
    rho = np.ones(n)
    u = 0.9 + 0.2 * u01(seed, i, 3)
    vx = 0.1 * normal(seed, i, 4)
    vy = 0.1 * normal(seed, i, 6)
    vz = 0.1 * normal(seed, i, 8)
    d2 = sum((np.abs(c - 0.5)) ** 2 for c in (x, y, z))   # |x-0.5| <= 0.5 already minimum image
    E = 1.0 + 0.5 * np.exp(-d2 / 0.02)
    kappa = np.ones(n)
    grid = _uniform_grid((0, 0, 0), (1, 1, 1), (1, 1, 1), 1.2 * dx)
    return _finish(f"c1_cube{nside}", KERNEL_CUBIC_SPLINE, grid, 5.0 / 3.0, x, y, z, h, m, rho, u, vx, vy, vz, E, kappa)


def lattice_hjitter(nside: int = 40, kernel: int = KERNEL_WENDLAND_C2, periodic=(1, 1, 1), seed: int = 2604201250,
                    hjit: float = 0.05, jitter: float = 0.05) -> Workload:
    """Jittered lattice in the unit cube with h = 1.2 dx (1 +- hjit) drawn per particle, on a grid with cell edge >= 2 max(h):
    every neighbourhood mixes different h, so the tiled path (which needs 2 h_max <= cell edge) runs its VARIABLE-h tile
    kernels on every tile (tests/test_gpu_edges.py).  Fields as config 1, unequal masses, variable rho and kappa."""
    dx = 1.0 / nside
    i, ix, iy, iz = _lattice(nside, nside, nside)
    n = i.size
    jit = lambda ch: (2.0 * u01(seed, i, ch) - 1.0) * jitter * dx
    pos = []
    for d, (c, ch) in enumerate(((ix, 0), (iy, 1), (iz, 2))):
        v = (c + 0.5) * dx + jit(ch)
        pos.append(_wrap(v, 0.0, 1.0) if periodic[d] else np.clip(v, 0.0, np.nextafter(1.0, 0.0)))
    x, y, z = pos
    h = 1.2 * dx * (1.0 + hjit * (2.0 * u01(seed, i, 3) - 1.0))
    hmax = 1.2 * dx * (1.0 + hjit)
    m = (0.8 + 0.4 * u01(seed, i, 10)) / n
    rho = 0.8 + 0.4 * u01(seed, i, 11)
    u = 0.9 + 0.2 * u01(seed, i, 12)
    vx, vy, vz = (0.1 * normal(seed, i, ch) for ch in (4, 6, 8))
    d2 = sum((np.abs(c - 0.5)) ** 2 for c in (x, y, z))
    E = 1.0 + 0.5 * np.exp(-d2 / 0.02)
    kappa = 0.5 + 2.0 * u01(seed, i, 13)
    grid = _uniform_grid((0, 0, 0), (1, 1, 1), tuple(periodic), hmax)
    w = _finish(f"hjit{nside}", kernel, grid, 5.0 / 3.0, x, y, z, h, m, rho, u, vx, vy, vz, E, kappa)
    w.alpha = 0.5 + u01(seed, i, 14)
    return w


# --------------------------------------------------------------------------- config 2
def config2(nl: int = 160, seed: int = SEEDS[2], jitter: float = 0.02, ly: float = 0.25) -> Workload:
    """Sod-style tube, periodic [0,2]x[0,.25]x[0,.25] (BJ config 2; Table 1).

    Left x<1: lattice dx_L = 1/nl, rho = 1, u = 2.5.  Right: lattice 2 dx_L, rho = 0.125, u = 2.0.
    Equal mass m = dx_L^3.  gamma = 1.4.  nl=160 gives 288 000 particles (the nominal
    262 144 cannot be met with equal masses and a density ratio of 8).  nl must be a multiple of 8.
    """
    assert nl % 8 == 0
    dxl = 1.0 / nl
    dxr = 2.0 * dxl
    nyl = int(round(ly * nl))          # ly = transverse box size (0.25 in BJ; tiny variants widen it)
    assert nyl % 2 == 0
    nxr, nyr = nl // 2, nyl // 2
    il, ixl, iyl, izl = _lattice(nl, nyl, nyl)
    ir, ixr, iyr, izr = _lattice(nxr, nyr, nyr)
    nL, nR = il.size, ir.size
    i = np.arange(nL + nR, dtype=np.int64)
    dxloc = np.concatenate([np.full(nL, dxl), np.full(nR, dxr)])
    jit = lambda ch: (2.0 * u01(seed, i, ch) - 1.0) * jitter * dxloc
    x = np.concatenate([(ixl + 0.5) * dxl, 1.0 + (ixr + 0.5) * dxr]) + jit(0)
    y = np.concatenate([(iyl + 0.5) * dxl, (iyr + 0.5) * dxr]) + jit(1)
    z = np.concatenate([(izl + 0.5) * dxl, (izr + 0.5) * dxr]) + jit(2)
    x, y, z = _wrap(x, 0.0, 2.0), _wrap(y, 0.0, ly), _wrap(z, 0.0, ly)
    h = 1.2 * dxloc
    m = np.full(nL + nR, dxl ** 3)
    rho = np.concatenate([np.ones(nL), np.full(nR, 0.125)])
    u = np.concatenate([np.full(nL, 2.5), np.full(nR, 2.0)])
    zeros = np.zeros(nL + nR)
    gamma = 1.4
    T = (gamma - 1.0) * u
    E = T ** 4
    kappa = rho.copy()
    hR = 1.2 * dxr
    grid = _uniform_grid((0, 0, 0), (2.0, ly, ly), (1, 1, 1), hR)
    return _finish(f"c2_sod{nl}", KERNEL_CUBIC_SPLINE, grid, gamma, x, y, z, h, m, rho, u, zeros, zeros, zeros, E, kappa)


# --------------------------------------------------------------------------- config 3
def config3(nside: int = 128, seed: int = SEEDS[3], jitter: float = 0.05) -> Workload:
    """Sedov-type blast, periodic unit cube, Wendland C2 h = 1.2 dx (BJ config 3)."""
    dx = 1.0 / nside
    i, ix, iy, iz = _lattice(nside, nside, nside)
    n = i.size
    jit = lambda ch: (2.0 * u01(seed, i, ch) - 1.0) * jitter * dx
    x = _wrap((ix + 0.5) * dx + jit(0), 0.0, 1.0)
    y = _wrap((iy + 0.5) * dx + jit(1), 0.0, 1.0)
    z = _wrap((iz + 0.5) * dx + jit(2), 0.0, 1.0)
    hval = 1.2 * dx
    h = np.full(n, hval)
    m = np.full(n, 1.0 / n)
    rho = np.ones(n)
    d2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
    hot = d2 < (2.0 * hval) ** 2
    nc = int(hot.sum())
    u = np.full(n, 1e-5)
    u[hot] = 1.0 / (nc * m[0])          # total energy 1 over the ~57-64 central particles
    zeros = np.zeros(n)
    gamma = 5.0 / 3.0
    T = (gamma - 1.0) * u
    E = T ** 4
    kappa = rho * T ** -3.5
    grid = _uniform_grid((0, 0, 0), (1, 1, 1), (1, 1, 1), hval)
    return _finish(f"c3_sedov{nside}", KERNEL_WENDLAND_C2, grid, gamma, x, y, z, h, m, rho, u, zeros, zeros, zeros, E, kappa,
                   notes={"n_hot": nc})


# --------------------------------------------------------------------------- config 4
def config4(res: int = 220, seed: int = SEEDS[4], rho_min: float = 1e-3, m_c_full: float = 1.25e-8,
            jitter: float = 0.1) -> Workload:
    """Laser-target slab + exponential corona, x open, y/z periodic 1x1 (BJ config 4).

    Slab x in [0, 0.1): nx_s x res x res lattice (dx = 1/res), rho = 1, T = 0.01.
    Corona s = x - x_s in [0, 0.05 ln(1/rho_min)): layers marched by s_{k+1} = s_k + d_k,
    d_k = (m_c / rho(s_k))^(1/3), rho = exp(-s/0.05); each layer an n_k x n_k lattice,
    n_k = round(1/d_k), particle mass rho(s_k) d_k / n_k^2.  h = 1.3 (m/rho)^(1/3).
    Wendland C2.  T(s) = 0.01 * 100^(s/s_max).  E = T^4, kappa = rho T^-3.5.
    ``res`` scales the resolution (220 = full size, ~5.2 M particles); m_c scales as (220/res)^3.
    """
    dx = 1.0 / res
    nxs = max(2, int(round(0.1 * res)))
    xs = nxs * dx                                   # slab thickness (0.1 at res = 220)
    m_c = m_c_full * (220.0 / res) ** 3
    smax = 0.05 * math.log(1.0 / rho_min)
    i_s, ixs, iys, izs = _lattice(nxs, res, res)
    X = [(ixs + 0.5) * dx]
    Y = [(iys + 0.5) * dx]
    Z = [(izs + 0.5) * dx]
    D = [np.full(i_s.size, dx)]
    M = [np.full(i_s.size, dx ** 3)]
    RHO = [np.ones(i_s.size)]
    S = [np.full(i_s.size, 0.0)]
    s = 0.0
    nlayers = 0
    while s < smax:
        rho_k = math.exp(-s / 0.05)
        d = (m_c / rho_k) ** (1.0 / 3.0)
        nk = max(1, int(round(1.0 / d)))
        j = np.arange(nk * nk, dtype=np.int64)
        X.append(np.full(j.size, xs + s + 0.5 * d))
        Y.append(((j % nk) + 0.5) / nk)
        Z.append(((j // nk) + 0.5) / nk)
        D.append(np.full(j.size, d))
        M.append(np.full(j.size, rho_k * d / (nk * nk)))
        RHO.append(np.full(j.size, rho_k))
        S.append(np.full(j.size, s))
        s += d
        nlayers += 1
    x, y, z, d, m, rho, sv = (np.concatenate(a) for a in (X, Y, Z, D, M, RHO, S))
    n = x.size
    i = np.arange(n, dtype=np.int64)
    corona = i >= i_s.size
    jamp = np.where(corona, jitter, 0.05) * d
    x = x + (2.0 * u01(seed, i, 0) - 1.0) * jamp
    y = _wrap(y + (2.0 * u01(seed, i, 1) - 1.0) * jamp, 0.0, 1.0)
    z = _wrap(z + (2.0 * u01(seed, i, 2) - 1.0) * jamp, 0.0, 1.0)
    h = 1.3 * (m / rho) ** (1.0 / 3.0)
    T = np.where(corona, 0.01 * 100.0 ** (sv / smax), 0.01)
    gamma = 5.0 / 3.0
    u = T / (gamma - 1.0)
    vx = np.where(corona, 0.01 * normal(seed, i, 4), 0.0)
    vy = np.where(corona, 0.01 * normal(seed, i, 6), 0.0)
    vz = np.where(corona, 0.01 * normal(seed, i, 8), 0.0)
    E = T ** 4
    kappa = rho * T ** -3.5
    # A14: edge = 2 * mean(h) (sequential fp64 sum), per-particle search range from h
    href = float(np.cumsum(h)[-1] / n)
    hmax = float(h.max())
    lo = (float(min(0.0, x.min())) - 1e-9, 0.0, 0.0)
    hi = (float(x.max()) + 1e-9, 1.0, 1.0)
    nc = tuple(max(1, int(math.floor((hi[k] - lo[k]) / (2.0 * href)))) for k in range(3))
    grid = Grid(lo, hi, nc, (0, 1, 1), hmax)
    return _finish(f"c4_slab{res}", KERNEL_WENDLAND_C2, grid, gamma, x, y, z, h, m, rho, u, vx, vy, vz, E, kappa,
                   notes={"n_slab": int(i_s.size), "n_corona": int(n - i_s.size), "layers": nlayers,
                          "h_min": float(h.min()), "h_max": hmax, "h_ref": href})


# --------------------------------------------------------------------------- config 5
def config5(nside: int = 256, seed: int = SEEDS[5], jitter: float = 0.05, vsigma: float = 0.0) -> Workload:
    """Two-fluid Rayleigh-Taylor interface, x/y periodic, z open, cubic spline h = 1.3 dx (BJ config 5).

    Heavy rho = 10 above z_i = 0.5 + 0.01 cos(2 pi x) cos(2 pi y), light rho = 1 below; m = rho dx^3;
    hydrostatic p(z) = p_top + int_z^1 rho dz' with p_top = 10, g = -1; u = p/((gamma-1) rho); v = 0
    (``vsigma`` > 0 gives the reported variant that exercises the viscosity arithmetic).
    """
    dx = 1.0 / nside
    i, ix, iy, iz = _lattice(nside, nside, nside)
    n = i.size
    jit = lambda ch: (2.0 * u01(seed, i, ch) - 1.0) * jitter * dx
    x0, y0, z0 = (ix + 0.5) * dx, (iy + 0.5) * dx, (iz + 0.5) * dx
    zi = 0.5 + 0.01 * np.cos(2 * math.pi * x0) * np.cos(2 * math.pi * y0)
    heavy = z0 > zi
    rho = np.where(heavy, 10.0, 1.0)
    m = rho * dx ** 3
    x = _wrap(x0 + jit(0), 0.0, 1.0)
    y = _wrap(y0 + jit(1), 0.0, 1.0)
    z = np.clip(z0 + jit(2), 0.0, np.nextafter(1.0, 0.0))
    p_top = 10.0
    p = np.where(heavy, p_top + 10.0 * (1.0 - z0), p_top + 10.0 * (1.0 - zi) + 1.0 * (zi - z0))
    gamma = 5.0 / 3.0
    u = p / ((gamma - 1.0) * rho)
    hval = 1.3 * dx
    h = np.full(n, hval)
    if vsigma > 0.0:
        vx, vy, vz = (vsigma * normal(seed, i, ch) for ch in (4, 6, 8))
    else:
        vx = vy = vz = np.zeros(n)
    T = p / rho
    E = T ** 4
    kappa = rho.copy()
    grid = _uniform_grid((0, 0, 0), (1, 1, 1), (1, 1, 0), hval)
    return _finish(f"c5_rt{nside}" + ("_v" if vsigma > 0 else ""), KERNEL_CUBIC_SPLINE, grid, gamma,
                   x, y, z, h, m, rho, u, vx, vy, vz, E, kappa)


# --------------------------------------------------------------------------- presets
PRESETS = {
    # the five BASELINE.json configs at full size
    "c1": lambda: config1(16),
    "c2": lambda: config2(160),
    "c3": lambda: config3(128),
    "c4": lambda: config4(220),
    "c5": lambda: config5(256),
    "c5_v": lambda: config5(256, vsigma=0.01),
    # tiny variants (N <= ~9k): brute-force O(N^2) oracle runs in seconds
    "c1_tiny": lambda: config1(16),
    "c2_tiny": lambda: config2(32, ly=0.5),
    "c3_tiny": lambda: config3(16),
    "c4_tiny": lambda: config4(24, rho_min=0.05),
    "c5_tiny": lambda: config5(16, vsigma=0.01),
    # mid sizes: several CTA tiles and a ragged tail, cell-list oracle in seconds
    "c2_mid": lambda: config2(64),
    "c3_mid": lambda: config3(40),
    "c4_mid": lambda: config4(48, rho_min=0.01),
    "c5_mid": lambda: config5(48, vsigma=0.01),
    # every tile of the tiled path has variable h (h jittered +-5 % on a grid with edge >= 2 max h)
    "hjit_w": lambda: lattice_hjitter(40, KERNEL_WENDLAND_C2, (1, 1, 1)),
    "hjit_c": lambda: lattice_hjitter(36, KERNEL_CUBIC_SPLINE, (1, 0, 1)),
}


def make(name: str) -> Workload:
    return PRESETS[name]()


def random_cloud(n: int, seed: int = 12345, kernel: int = KERNEL_WENDLAND_C2, periodic=(1, 1, 1),
                 hvar: float = 2.0, box=(1.0, 1.0, 1.0), ncell=None) -> Workload:
    """Uniform-random particles with log-uniform h in [h0, hvar*h0]: the adversarial variable-h case
    used by the conservation pins (T9-T11) and by the edge-case parity tests."""
    i = np.arange(n, dtype=np.int64)
    x = u01(seed, i, 0) * box[0]
    y = u01(seed, i, 1) * box[1]
    z = u01(seed, i, 2) * box[2]
    vol = box[0] * box[1] * box[2]
    h0 = 1.1 * (vol / max(n, 1)) ** (1.0 / 3.0)
    h = h0 * hvar ** u01(seed, i, 3)
    hmax = h0 * hvar
    for d in range(3):
        if periodic[d]:
            assert box[d] >= 6.0 * hmax, "periodic extent must be >= 3 * 2 h_max"
    m = (0.5 + u01(seed, i, 4)) * vol / max(n, 1)
    rho = 0.5 + u01(seed, i, 5)
    u = 0.5 + u01(seed, i, 6)
    vx, vy, vz = (0.3 * normal(seed, i, ch) for ch in (7, 9, 11))
    E = 0.5 + u01(seed, i, 13)
    kappa = 0.5 + 4.0 * u01(seed, i, 14)
    if ncell is None:
        href = float(np.cumsum(h)[-1] / max(n, 1)) if n else h0
        ncell = tuple(max(1, int(math.floor(box[d] / (2.0 * href)))) for d in range(3))
    grid = Grid((0.0, 0.0, 0.0), tuple(float(b) for b in box), tuple(ncell), tuple(periodic), float(hmax))
    w = _finish(f"cloud{n}", kernel, grid, 5.0 / 3.0, x, y, z, h, m, rho, u, vx, vy, vz, E, kappa)
    w.alpha = 0.2 + u01(seed, i, 15)
    return w


def level_edges(h: np.ndarray, ratio: float = 1.5, max_levels: int = 16):
    """Cell edges for the internal levels of the tiled path (spray_set_levels): a geometric sequence from 2 min(h) up to
    2 max(h), the last one exactly 2 max(h) (all with a 1e-6 margin), at most `max_levels` values.  A grid choice like
    `_uniform_grid` (A14): no SPH arithmetic."""
    lo, hi = 2.0 * float(np.min(h)) * (1.0 + 1e-6), 2.0 * float(np.max(h)) * (1.0 + 1e-6)
    if hi <= lo * (1.0 + 1e-9):
        return [hi]
    k = max(1, min(max_levels - 1, int(math.ceil(math.log(hi / lo) / math.log(ratio)))))
    r = (hi / lo) ** (1.0 / k)
    return [lo * r ** i for i in range(k)] + [hi]
