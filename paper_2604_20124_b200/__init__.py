"""paper_2604_20124_b200 -- B200-native SPH pair-summation pass of SPRAY (arxiv/paper_2604_20124).

Thin Python binding over the C-ABI library ``libspray_b200.so`` (``include/spray.h``): argument marshalling
only -- every step of the path runs in the library's CUDA kernels.  PyTorch is used for device memory and
streams.  There is NO CPU fallback: if the library is missing or was not built, every entry point raises.

Build in-tree with ``python -m paper_2604_20124_b200.build`` (nvcc, sm_100a).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

__all__ = ["load", "Spray", "SprayError", "KERNEL_CUBIC_SPLINE", "KERNEL_WENDLAND_C2", "FLD_SYMMETRIC", "FLD_GATHER",
           "FLD_UPDATE_LIMITER", "FLD_FROZEN", "FLD_FROZEN_CHAINED", "EXPORTS", "cell_list_static", "STATIC_NMAX", "STATIC_NCELL_MAX"]

_LIBPATH = Path(__file__).resolve().parent / "libspray_b200.so"

KERNEL_CUBIC_SPLINE, KERNEL_WENDLAND_C2 = 0, 1
FLD_SYMMETRIC, FLD_GATHER = 0, 1
FLD_UPDATE_LIMITER, FLD_FROZEN, FLD_FROZEN_CHAINED = 0, 1, 2
COND_OPERATOR, COND_RHS = 0, 1
DEV_H_EXCEEDS_HMAX, DEV_OUTSIDE_BOX, DEV_LIST_OVERFLOW = 1, 2, 4

# every symbol include/spray.h declares
EXPORTS = ["spray_version", "spray_create", "spray_destroy", "spray_last_error", "spray_check", "spray_launch_count", "spray_set_path", "spray_set_levels", "spray_path_stats", "spray_build_timing",
           "spray_build_cells", "spray_density", "spray_hydro_rhs", "spray_hydro_rhs_limiter", "spray_fld_apply", "spray_get_cell_table",
           "spray_neighbor_counts", "spray_neighbor_lists", "spray_neighbor_digest", "spray_rad_jacobi", "spray_conduction", "spray_kgc_continuity", "spray_ray_deposit", "spray_conduction_implicit", "spray_fp64_peak_probe",
           "spray_cell_list_static", "spray_static_last_error"]


class SprayError(RuntimeError):
    pass


class Grid(C.Structure):
    """spray_grid_t"""
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3), ("ncell", C.c_int32 * 3),
                ("periodic", C.c_int32 * 3), ("h_max", C.c_double)]


_lib = None


def load():
    """dlopen libspray_b200.so and declare the prototypes.  Raises (loudly) if the library is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIBPATH.exists():
        raise SprayError(f"{_LIBPATH} not found: build it with `python -m paper_2604_20124_b200.build` "
                         "(there is no CPU fallback)")
    lib = C.CDLL(str(_LIBPATH))
    vp, i64, dbl, i32 = C.c_void_p, C.c_int64, C.c_double, C.c_int
    lib.spray_version.restype = C.c_char_p
    lib.spray_version.argtypes = []
    lib.spray_last_error.restype = C.c_char_p
    lib.spray_last_error.argtypes = [vp]
    lib.spray_create.argtypes = [C.POINTER(vp), i64, i64, i32]
    lib.spray_destroy.argtypes = [vp]
    lib.spray_check.argtypes = [vp, vp, C.POINTER(C.c_uint32)]
    lib.spray_set_path.argtypes = [vp, i32]
    lib.spray_launch_count.argtypes = [vp]
    lib.spray_path_stats.argtypes = [vp, vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.spray_set_levels.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    lib.spray_build_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.spray_build_cells.argtypes = [vp, C.POINTER(Grid), i32, i64, vp, vp, vp, vp, vp]
    lib.spray_density.argtypes = [vp, vp, vp, vp, vp]
    lib.spray_hydro_rhs.argtypes = [vp] + [vp] * 8 + [dbl] + [vp] * 5 + [vp]
    lib.spray_hydro_rhs_limiter.argtypes = [vp] + [vp] * 8 + [dbl] + [vp, vp, dbl] + [vp] * 7 + [vp]
    lib.spray_fld_apply.argtypes = [vp, vp, vp, vp, vp, dbl, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.spray_conduction.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.spray_kgc_continuity.argtypes = [vp] * 10
    lib.spray_conduction_implicit.argtypes = [vp] + [vp] * 11 + [dbl, i32, vp, vp, vp]
    lib.spray_rad_jacobi.argtypes = [vp] + [vp] * 8 + [dbl, dbl, dbl, i32, i32, vp, vp, vp, vp]
    lib.spray_ray_deposit.argtypes = [vp, vp, vp, vp, vp, i64, vp, dbl, i64, dbl, dbl, vp, vp, vp, vp, vp]
    lib.spray_get_cell_table.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.spray_neighbor_counts.argtypes = [vp, i32, vp, vp]
    lib.spray_neighbor_lists.argtypes = [vp, i32, vp, vp, vp]
    lib.spray_neighbor_digest.argtypes = [vp, i32, vp, vp, vp]
    lib.spray_fp64_peak_probe.argtypes = [i32, i32, i32, i64, vp, vp]
    lib.spray_cell_list_static.argtypes = [C.POINTER(Grid), i64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.spray_static_last_error.argtypes = []
    lib.spray_static_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("spray_version", "spray_last_error", "spray_static_last_error"):
            getattr(lib, name).restype = C.c_int
    lib.spray_launch_count.restype = C.c_int64
    _lib = lib
    return lib


def _ptr(t, dtype=None, n=None):
    """device pointer of a contiguous CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise SprayError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise SprayError(f"expected dtype {dtype}, got {t.dtype}")
    if n is not None and t.numel() < n:
        raise SprayError(f"tensor too short: {t.numel()} < {n}")
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


STATIC_NMAX, STATIC_NCELL_MAX = 262144, 16777216


def cell_list_static(grid, x, y, z, sorted_key=None, perm=None, cell_start=None, cell_end=None, dev_status=None):
    """spray_cell_list_static: cell key, stable sort and cell table without a context and without any allocation inside
    the library (its scratch is a static device array; calls that overlap on the GPU race on it).  Works on the current
    device.  Output tensors not supplied are allocated HERE with torch (a caller that must not allocate passes them)."""
    import torch
    lib = load()
    n = int(x.numel())
    ncell = int(grid.ncell[0]) * int(grid.ncell[1]) * int(grid.ncell[2])
    i32 = torch.int32   # u32 payloads viewed as int32 tensors
    dev = x.device
    sorted_key = torch.empty(n, dtype=i32, device=dev) if sorted_key is None else sorted_key
    perm = torch.empty(n, dtype=i32, device=dev) if perm is None else perm
    cell_start = torch.empty(ncell, dtype=i32, device=dev) if cell_start is None else cell_start
    cell_end = torch.empty(ncell, dtype=i32, device=dev) if cell_end is None else cell_end
    g = Grid((C.c_double * 3)(*grid.lo), (C.c_double * 3)(*grid.hi), (C.c_int32 * 3)(*grid.ncell),
             (C.c_int32 * 3)(*grid.periodic), float(grid.h_max))
    f64 = torch.float64
    rc = lib.spray_cell_list_static(C.byref(g), n, _ptr(x, f64, n), _ptr(y, f64, n), _ptr(z, f64, n), _ptr(sorted_key, i32, n),
                                    _ptr(perm, i32, n), _ptr(cell_start, i32, ncell), _ptr(cell_end, i32, ncell),
                                    _ptr(dev_status, i32, 1), _stream())
    if rc != 0:
        raise SprayError(f"spray_cell_list_static failed ({rc}): {lib.spray_static_last_error().decode()}")
    return dict(sorted_key=sorted_key, perm=perm, cell_start=cell_start, cell_end=cell_end)


class Spray:
    """One spray_ctx.  Methods mirror the C entry points (same names without the ``spray_`` prefix); tensors are
    fp64 CUDA tensors in caller order; outputs are allocated with torch when not supplied."""

    def __init__(self, n_max: int, ncell_max: int, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise SprayError("no CUDA device: the SPRAY pass has no CPU fallback")
        self.lib = load()
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.n = 0
        self.ncell = 0
        h = C.c_void_p()
        rc = self.lib.spray_create(C.byref(h), int(n_max), int(ncell_max), int(device))
        if rc != 0:
            raise SprayError(f"spray_create failed ({rc}): {self.lib.spray_last_error(None).decode()}")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.spray_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc, what):
        if rc != 0:
            raise SprayError(f"{what} failed ({rc}): {self.lib.spray_last_error(self.h).decode()}")

    def _out(self, t, dtype=None, n=None):
        dtype = dtype or self.torch.float64
        n = self.n if n is None else n
        if t is None:
            t = self.torch.empty(n, dtype=dtype, device=self.device)
        return t

    # -- spray_set_path / spray_check
    def set_path(self, path: int):
        self._ck(self.lib.spray_set_path(self.h, int(path)), "spray_set_path")

    def launch_count(self) -> int:
        return int(self.lib.spray_launch_count(self.h))

    def path_stats_full(self):
        """Statistics of the last build_cells (synchronises): tiles, particles served by the tiled kernels, list-builder
        work units (half tiles) that found non-uniform h, bytes of device scratch the context holds."""
        nt, nf, nn, nb = C.c_int64(0), C.c_int64(0), C.c_int64(0), C.c_int64(0)
        dec = (C.c_int64 * 4)()
        self._ck(self.lib.spray_path_stats(self.h, _stream(), C.byref(nt), C.byref(nf), C.byref(nn), C.byref(nb), dec), "spray_path_stats")
        return {"tiles": int(nt.value), "n_fast": int(nf.value), "nonuniform_units": int(nn.value), "scratch_bytes": int(nb.value),
                "declined": [int(x) for x in dec]}

    def set_levels(self, grid, edges):
        """Internal levels of the tiled path on the box of `grid`: one grid of cell edge >= edges[k] each (ascending)."""
        edges = [float(e) for e in edges]
        nc = []
        for e in edges:
            m = 1
            for d in range(3):
                m *= max(1, int((float(grid.hi[d]) - float(grid.lo[d])) / e * (1.0 + 1e-12)))
            nc.append(m)
        ea = (C.c_double * max(len(edges), 1))(*edges)
        na = (C.c_int64 * max(len(edges), 1))(*nc)
        self._ck(self.lib.spray_set_levels(self.h, len(edges), ea, na), "spray_set_levels")

    def build_timing(self):
        """Device milliseconds of the last build_cells: (cell list a1-a4, tiles + tables, neighbour-list builder); synchronises."""
        a, b, d = C.c_double(0), C.c_double(0), C.c_double(0)
        self._ck(self.lib.spray_build_timing(self.h, C.byref(a), C.byref(b), C.byref(d)), "spray_build_timing")
        return a.value, b.value, d.value

    def path_stats(self):
        """(tiles, particles served by the tiled kernels) of the last build_cells; synchronises."""
        st = self.path_stats_full()
        return st["tiles"], st["n_fast"]

    def check(self) -> int:
        st = C.c_uint32(0)
        self._ck(self.lib.spray_check(self.h, _stream(), C.byref(st)), "spray_check")
        return int(st.value)

    # -- spray_build_cells
    def build_cells(self, grid, kernel: int, x, y, z, h):
        g = Grid((C.c_double * 3)(*grid.lo), (C.c_double * 3)(*grid.hi), (C.c_int32 * 3)(*grid.ncell),
                 (C.c_int32 * 3)(*grid.periodic), float(grid.h_max))
        n = int(x.numel())
        f64 = self.torch.float64
        rc = self.lib.spray_build_cells(self.h, C.byref(g), int(kernel), n, _ptr(x, f64, n), _ptr(y, f64, n), _ptr(z, f64, n),
                                        _ptr(h, f64, n), _stream())
        self._ck(rc, "spray_build_cells")
        self.n = n
        self.ncell = int(grid.ncell[0]) * int(grid.ncell[1]) * int(grid.ncell[2])

    # -- spray_density
    def density(self, m, rho=None, nnbr=None, want_nnbr=False):
        f64 = self.torch.float64
        rho = self._out(rho)
        if want_nnbr and nnbr is None:
            nnbr = self.torch.empty(self.n, dtype=self.torch.int32, device=self.device)
        self._ck(self.lib.spray_density(self.h, _ptr(m, f64, self.n), _ptr(rho, f64, self.n), _ptr(nnbr), _stream()), "spray_density")
        return (rho, nnbr) if want_nnbr else rho

    # -- spray_hydro_rhs
    def hydro_rhs(self, m, rho, p, cs, vx, vy, vz, alpha, beta=2.0, out=None):
        f64 = self.torch.float64
        if out is None:
            out = [self._out(None) for _ in range(5)]
        ins = [_ptr(t, f64, self.n) for t in (m, rho, p, cs, vx, vy, vz, alpha)]
        outs = [_ptr(t, f64, self.n) for t in out]
        self._ck(self.lib.spray_hydro_rhs(self.h, *ins, float(beta), *outs, _stream()), "spray_hydro_rhs")
        return out   # ax, ay, az, dudt, divv_sum

    # -- spray_hydro_rhs_limiter
    def hydro_rhs_limiter(self, m, rho, p, cs, vx, vy, vz, alpha, E, kappa, beta=2.0, c_light=1.0, out=None, mu=None, gradE=None,
                          want_gradE=False):
        """Hydro right-hand sides and the FLD limiter pre-sweep in one sweep (include/spray.h).
        Returns ([ax, ay, az, dudt, divv_sum], mu, gradE or None)."""
        f64 = self.torch.float64
        if out is None:
            out = [self._out(None) for _ in range(5)]
        mu = self._out(mu)
        if want_gradE:
            gradE = self._out(gradE, n=3 * self.n)
        ins = [_ptr(t, f64, self.n) for t in (m, rho, p, cs, vx, vy, vz, alpha)]
        outs = [_ptr(t, f64, self.n) for t in out]
        rc = self.lib.spray_hydro_rhs_limiter(self.h, *ins, float(beta), _ptr(E, f64, self.n), _ptr(kappa, f64, self.n), float(c_light),
                                              *outs, _ptr(mu, f64, self.n), _ptr(gradE), _stream())
        self._ck(rc, "spray_hydro_rhs_limiter")
        return out, mu, gradE

    # -- spray_fld_apply
    def fld_apply(self, m, rho, kappa, E, c_light=1.0, kmode=FLD_SYMMETRIC, lmode=FLD_UPDATE_LIMITER, mu=None, y=None,
                  diag=None, offd=None, gradE=None, want_diag=True, want_gradE=False):
        f64 = self.torch.float64
        mu = self._out(mu)
        y = self._out(y)
        if want_diag:
            diag, offd = self._out(diag), self._out(offd)
        if want_gradE:
            gradE = self._out(gradE, n=3 * self.n)
        rc = self.lib.spray_fld_apply(self.h, _ptr(m, f64, self.n), _ptr(rho, f64, self.n), _ptr(kappa, f64, self.n),
                                      _ptr(E, f64, self.n), float(c_light), int(kmode), int(lmode), _ptr(mu, f64, self.n),
                                      _ptr(y, f64, self.n), _ptr(diag), _ptr(offd), _ptr(gradE), _stream())
        self._ck(rc, "spray_fld_apply")
        return dict(mu=mu, y=y, diag=diag, offd=offd, gradE=gradE)

    def conduction(self, m, rho, k, T, dudt=None):
        """Row N2: thermal-conduction term of eqs. (17)/(18) for one species (include/spray.h)."""
        f64 = self.torch.float64
        dudt = self._out(dudt)
        rc = self.lib.spray_conduction(self.h, _ptr(m, f64, self.n), _ptr(rho, f64, self.n), _ptr(k, f64, self.n), _ptr(T, f64, self.n),
                                       _ptr(dudt, f64, self.n), _stream())
        self._ck(rc, "spray_conduction")
        return dudt

    def conduction_implicit(self, m, rho, k_i, k_e, kei, dTdu_i, dTdu_e, T_i, T_e, u_i, u_e, dt, which):
        """Row N2, implicit two-temperature system eqs. (28)-(34): which = COND_OPERATOR (left-hand sides applied to (u_i, u_e);
        T_i, T_e may be None) or COND_RHS (b^i + c, b^e - c).  Returns (out_i, out_e)."""
        f64 = self.torch.float64
        out_i, out_e = self._out(None), self._out(None)
        a = [_ptr(t, f64, self.n) for t in (m, rho, k_i, k_e, kei, dTdu_i, dTdu_e, T_i, T_e, u_i, u_e)]
        rc = self.lib.spray_conduction_implicit(self.h, *a, float(dt), int(which), _ptr(out_i, f64, self.n), _ptr(out_e, f64, self.n), _stream())
        self._ck(rc, "spray_conduction_implicit")
        return out_i, out_e

    def kgc_continuity(self, m, rho, vx, vy, vz, want_L=True, want_raw=True):
        """Row N3: continuity equation eq. (37) with the KGC filter of eqs. (39)-(40) (include/spray.h).
        Returns dict(drhodt, L [9, n] or None, drhodt_raw or None)."""
        f64 = self.torch.float64
        drhodt = self._out(None)
        L = self.torch.empty((9, self.n), dtype=f64, device=self.device) if want_L else None
        raw = self._out(None) if want_raw else None
        a = [_ptr(t, f64, self.n) for t in (m, rho, vx, vy, vz)]
        rc = self.lib.spray_kgc_continuity(self.h, *a, _ptr(drhodt, f64, self.n), _ptr(L), _ptr(raw), _stream())
        self._ck(rc, "spray_kgc_continuity")
        return dict(drhodt=drhodt, L=L, drhodt_raw=raw)

    def rad_jacobi(self, m, rho, mu, kappa_p, E_n, u_n, T_n, dTdu, dt, c_light=1.0, a_rad=1.0, niter=1, kmode=FLD_SYMMETRIC,
                   E0=None, want_resid=True):
        """Row N1: niter Jacobi iterations of the implicit radiation step (include/spray.h).  Returns dict(E, u, resid)."""
        f64 = self.torch.float64
        E = (E_n if E0 is None else E0).clone()
        u = self._out(None)
        resid = self.torch.zeros(int(niter), dtype=f64, device=self.device) if want_resid else None
        a = [_ptr(t, f64, self.n) for t in (m, rho, mu, kappa_p, E_n, u_n, T_n, dTdu)]
        rc = self.lib.spray_rad_jacobi(self.h, *a, float(dt), float(c_light), float(a_rad), int(kmode), int(niter),
                                       _ptr(E, f64, self.n), _ptr(u, f64, self.n), _ptr(resid), _stream())
        self._ck(rc, "spray_rad_jacobi")
        return dict(E=E, u=u, resid=resid)

    def ray_deposit(self, m, rho, f, kib, rays, dt, nsteps, c_light=1.0, pmin=0.0, want_gradn=True):
        """Row N4: mesh-free laser ray tracing and deposition (include/spray.h).  rays: fp64 CUDA tensor (7, nrays) with
        rows x, y, z, vx, vy, vz, P.  Returns dict(gradn (3, n) or None, edep (n), rays (7, nrays), steps (nrays, int64))."""
        t = self.torch
        f64 = t.float64
        if rays.dim() != 2 or rays.shape[0] != 7:
            raise SprayError("rays must have shape (7, nrays)")
        nr = int(rays.shape[1])
        gradn = t.empty((3, self.n), dtype=f64, device=self.device) if want_gradn else None
        edep = self._out(None)
        rout = t.empty((7, nr), dtype=f64, device=self.device)
        steps = t.empty(nr, dtype=t.int64, device=self.device)
        a = [_ptr(x, f64, self.n) for x in (m, rho, f, kib)]
        rc = self.lib.spray_ray_deposit(self.h, *a, nr, _ptr(rays, f64, 7 * nr), float(dt), int(nsteps), float(c_light), float(pmin),
                                        _ptr(gradn), _ptr(edep, f64, self.n), _ptr(rout), _ptr(steps), _stream())
        self._ck(rc, "spray_ray_deposit")
        return dict(gradn=gradn, edep=edep, rays=rout, steps=steps)

    # -- parity exports
    def get_cell_table(self):
        t = self.torch
        i32 = t.int32   # u32 payloads viewed as int32 tensors
        sk = t.empty(self.n, dtype=i32, device=self.device)
        perm = t.empty(self.n, dtype=i32, device=self.device)
        cs = t.empty(self.ncell, dtype=i32, device=self.device)
        ce = t.empty(self.ncell, dtype=i32, device=self.device)
        self._ck(self.lib.spray_get_cell_table(self.h, _ptr(sk), _ptr(perm), _ptr(cs), _ptr(ce), _stream()), "spray_get_cell_table")
        return dict(sorted_key=sk, perm=perm, cell_start=cs, cell_end=ce)

    def neighbor_counts(self, symmetric: bool):
        cnt = self.torch.empty(self.n, dtype=self.torch.int32, device=self.device)
        self._ck(self.lib.spray_neighbor_counts(self.h, int(bool(symmetric)), _ptr(cnt), _stream()), "spray_neighbor_counts")
        return cnt

    def neighbor_lists(self, symmetric: bool):
        t = self.torch
        cnt = self.neighbor_counts(symmetric).to(t.int64)
        off = t.zeros(self.n + 1, dtype=t.int64, device=self.device)
        if self.n:
            off[1:] = t.cumsum(cnt, 0)
        total = int(off[-1].item())
        nbr = t.empty(max(total, 1), dtype=t.int32, device=self.device)
        self._ck(self.lib.spray_neighbor_lists(self.h, int(bool(symmetric)), _ptr(off), _ptr(nbr), _stream()), "spray_neighbor_lists")
        return off, nbr[:total]

    def neighbor_digest(self, symmetric: bool):
        t = self.torch
        ds = t.empty(self.n, dtype=t.int64, device=self.device)
        dx = t.empty(self.n, dtype=t.int64, device=self.device)
        self._ck(self.lib.spray_neighbor_digest(self.h, int(bool(symmetric)), _ptr(ds), _ptr(dx), _stream()), "spray_neighbor_digest")
        return ds, dx


def fp64_peak_probe(device: int, blocks: int, threads: int, iters: int, out) -> None:
    rc = load().spray_fp64_peak_probe(int(device), int(blocks), int(threads), int(iters), _ptr(out), _stream())
    if rc != 0:
        raise SprayError(f"spray_fp64_peak_probe failed ({rc})")
