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
