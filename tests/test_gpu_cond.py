"""GPU parity of row N2 (spray_conduction, eqs. (17)/(18) second term) against oracle.conduction: |gpu - oracle| <= 1e-11 S_a,
S_a = sum of the absolute pair contributions; exact zero for a uniform temperature."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity_util import check, make_ctx, upload

pytestmark = pytest.mark.gpu


def workload(name):
    if name == "c1":
        return W.make("c1")
    if name == "lattice_wendland":
        return W.config3(nside=24)
    if name == "cloud_periodic":
        return W.random_cloud(5000, seed=12, periodic=(1, 1, 1), hvar=2.0, kernel=W.KERNEL_CUBIC_SPLINE)
    if name == "cloud_mixed":
        return W.random_cloud(4000, seed=13, periodic=(1, 0, 1), hvar=2.2)
    raise KeyError(name)


@pytest.mark.parametrize("name", ["c1", "lattice_wendland", "cloud_periodic", "cloud_mixed"])
def test_conduction_parity(name):
    import torch
    w = workload(name)
    k = 0.2 + w.kappa / (1.0 + w.kappa)
    T = 0.5 + w.E / np.max(w.E)
    o = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, k, T)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.conduction(d["m"], d["rho_nom"], t(k), t(T)).cpu().numpy()
    e = check("dudt", g, o["dudt"], o["S_dudt"])
    assert abs(np.sum(w.m * g)) <= 1e-11 * np.sum(w.m * o["S_dudt"])      # conservative on the GPU as well
    g0 = sp.conduction(d["m"], d["rho_nom"], t(k), t(np.full(w.n, 1.25))).cpu().numpy()
    assert np.all(g0 == 0.0)
    assert sp.check() == 0
    print(name, "max normalised error", e)


def test_conduction_full_size_sampled():
    """Config 5 (16.7M particles), the launch configuration of bench.py: 2000 sampled targets against the oracle."""
    import torch
    w = W.make("c5")
    i = np.arange(2000, dtype=np.uint64)
    sel = np.unique((W.splitmix64(i + np.uint64(91)) % np.uint64(w.n)).astype(np.int64))
    k = 0.2 + w.kappa / (1.0 + w.kappa)
    T = 0.5 + w.E / np.max(w.E) + 0.1 * np.sin(9.0 * w.x)
    o = O.conduction(w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m, w.rho_nom, k, T, targets=sel)
    d = upload(w)
    sp = make_ctx(w)
    sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = sp.conduction(d["m"], d["rho_nom"], t(k), t(T)).cpu().numpy()
    e = check("dudt", g[sel], o["dudt"], o["S_dudt"])
    assert sp.path_stats()[1] == w.n          # every particle was served by the tiled kernels
    print("c5 sampled: max normalised error", e)
