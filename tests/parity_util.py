"""Helpers for the GPU parity tests: run the CUDA path through the C-ABI binding, run the oracle, compare.

Tolerance (BASELINE.json north_star): per-particle |gpu - oracle| <= 1e-11 * S_a, S_a = sum of the absolute pair
contributions (oracle normaliser, contract O8); exact equality where S_a = 0.  Integer outputs bit-exact.
"""
import numpy as np

import oracle as O

TOL = 1e-11
FIELDS = ("x", "y", "z", "h", "m", "rho_nom", "p", "cs", "vx", "vy", "vz", "alpha", "E", "kappa")


def upload(w, device="cuda"):
    import torch
    return {f: torch.from_numpy(np.ascontiguousarray(getattr(w, f))).to(device) for f in FIELDS}


def make_ctx(w, path=None, slack=0):
    from paper_2604_20124_b200 import Spray
    sp = Spray(w.n + slack, max(w.grid.ncell_total, 1))
    if path is not None:
        sp.set_path(path)
    return sp


def u32(t):
    """int32 CUDA tensor holding u32 payloads -> numpy uint32"""
    return t.cpu().numpy().view(np.uint32)


def u64(t):
    return t.cpu().numpy().view(np.uint64)


def norm_err(gpu, ref, S):
    gpu, ref, S = np.asarray(gpu), np.asarray(ref), np.asarray(S)
    d = np.abs(gpu - ref)
    z = S == 0
    assert np.array_equal(gpu[z], ref[z]), "exact equality required where the normaliser is 0"
    e = np.zeros_like(d)
    e[~z] = d[~z] / S[~z]
    assert np.isfinite(gpu).all()
    return float(e.max()) if e.size else 0.0


def check(name, gpu, ref, S, tol=TOL):
    e = norm_err(gpu, ref, S)
    assert e <= tol, f"{name}: normalised error {e:.3e} > {tol:.1e}"
    return e


def mu_tolerance(li):
    """contract O8: mu compared by relative error <= 1e-11 * max(1, (S_gradE/|gradE|) * R^2/(9+R^2))"""
    g = np.sqrt(li["gx"] ** 2 + li["gy"] ** 2 + li["gz"] ** 2)
    Sg = li["S_gx"] + li["S_gy"] + li["S_gz"]
    R = li["R"]
    amp = np.where(g > 0, Sg / np.where(g > 0, g, 1.0) * R * R / (9.0 + R * R), 0.0)
    return TOL * np.maximum(1.0, amp)


def check_mu(gpu_mu, li):
    rel = np.abs(gpu_mu - li["mu"]) / np.abs(li["mu"])
    tol = mu_tolerance(li)
    bad = rel > tol
    assert not bad.any(), f"mu: {bad.sum()} particles beyond tolerance, worst {float((rel / tol).max()):.3e} x tol"
    return float((rel / tol).max())


def gpu_isolated(sp, d, w, targets=None, mu_in=None, kmode=0):
    """Each sweep on its own with generator-supplied inputs (rho = rho_nom).  Returns numpy arrays (all particles)."""
    import torch
    rho, nn = sp.density(d["m"], want_nnbr=True)
    ax, ay, az, dudt, divv = sp.hydro_rhs(d["m"], d["rho_nom"], d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], w.beta)
    up = sp.fld_apply(d["m"], d["rho_nom"], d["kappa"], d["E"], w.c_light, kmode=kmode, lmode=0, want_gradE=True)
    # spray_hydro_rhs_limiter promises the results of the two calls above bit for bit, on every path and particle set
    fy, fmu, fg = sp.hydro_rhs_limiter(d["m"], d["rho_nom"], d["p"], d["cs"], d["vx"], d["vy"], d["vz"], d["alpha"], d["E"], d["kappa"],
                                       beta=w.beta, c_light=w.c_light, want_gradE=True)
    for k, a, b in zip(("ax", "ay", "az", "dudt", "divv"), (ax, ay, az, dudt, divv), fy):
        assert torch.equal(a, b), "fused " + k
    assert torch.equal(up["mu"], fmu) and torch.equal(up["gradE"], fg), "fused limiter"
    out = dict(rho=rho, nnbr=nn, ax=ax, ay=ay, az=az, dudt=dudt, divv=divv, mu=up["mu"], y_upd=up["y"],
               gradE=up["gradE"])
    if mu_in is not None:
        mu_t = torch.from_numpy(mu_in).to(rho.device)
        fr = sp.fld_apply(d["m"], d["rho_nom"], None, d["E"], w.c_light, kmode=kmode, lmode=1, mu=mu_t)
        out.update(y=fr["y"], diag=fr["diag"], offd=fr["offd"])
    torch.cuda.synchronize()
    res = {}
    for k, v in out.items():
        a = v.cpu().numpy()
        res[k] = a.view(np.uint32) if k == "nnbr" else a
    if targets is not None:
        n = w.n
        g = res.pop("gradE")
        res = {k: v[targets] for k, v in res.items()}
        res["gradE"] = np.stack([g[targets], g[n + targets], g[2 * n + targets]])
    else:
        res["gradE"] = res["gradE"].reshape(3, w.n)
    return res


def oracle_isolated(w, targets=None, sym_mode=True, mu_full=None):
    a = (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)
    d = O.density(*a, targets=targets)
    hy = O.hydro(*a, w.rho_nom, w.p, w.cs, w.vx, w.vy, w.vz, w.alpha, w.beta, targets=targets)
    li = O.limiter(*a, w.rho_nom, w.kappa, w.E, w.c_light, targets=targets)
    out = {**d, **hy, **{"li": li}}
    if mu_full is not None:
        out["ap"] = O.fld_apply(*a, w.rho_nom, mu_full, w.E, sym_mode=sym_mode, targets=targets)
    return out


def compare_isolated(g, o, with_apply=True):
    errs = {}
    assert np.array_equal(g["nnbr"], o["nnbr"]), "gather neighbour counts differ"
    errs["rho"] = check("rho", g["rho"], o["rho"], o["S_rho"])
    for k in ("ax", "ay", "az", "dudt", "divv"):
        errs[k] = check(k, g[k], o[k], o["S_" + k])
    li = o["li"]
    for i, k in enumerate(("gx", "gy", "gz")):
        errs[k] = check("gradE_" + k, g["gradE"][i], li[k], li["S_" + k])
    errs["mu"] = check_mu(g["mu"], li)
    if with_apply:
        ap = o["ap"]
        errs["y"] = check("y", g["y"], ap["y"], ap["S_y"])
        errs["diag"] = check("diag", g["diag"], ap["diag"], ap["S_diag"])
        errs["offd"] = check("offd", g["offd"], ap["offd"], ap["S_offd"])
    return errs
