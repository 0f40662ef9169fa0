"""GPU parity of SURVEY.md 8(f) rank 4 through the C-ABI: short-range acceleration, jerk and potential over the
neighbour rows against the oracle (fp64 on both sides; tolerance 1e-11: the two differ only by fma contraction
and, for rows longer than 32 entries, by the summation order)."""
import numpy as np
import pytest

import oracle
from workloads import make_workload

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _P():
    import paper_2006_16560_b200 as P
    return P


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run(w, rout, off, idx):
    import torch
    P = _P()
    n = w.N
    ins = [_dev(a) for a in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rout)]
    out = [torch.full((n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(7)]
    ws = torch.empty(P.petar_short_range_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    P.petar_short_range_force(*ins, _dev(off), _dev(idx if len(idx) else np.zeros(1, np.int32)), n, w.G, w.r_in_over_r_out,
                              out[0:3], out[3:6], out[6], ws)
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in out]


def _pot_scale(w, off, idx):
    """sum_j G m_j / r_ij over the rows: the magnitude the potential terms are made of (W itself cancels to ~0 near r_out)."""
    rows = np.repeat(np.arange(w.N), np.diff(off))
    r = np.sqrt((w.x[rows] - w.x[idx]) ** 2 + (w.y[rows] - w.y[idx]) ** 2 + (w.z[rows] - w.z[idx]) ** 2)
    sc = np.zeros(w.N)
    ok = r > 0
    np.add.at(sc, rows[ok], w.G * w.m[idx[ok]] / r[ok])
    return sc


def _compare(g, o, psc):
    # scale: the sum of the magnitudes is not available, so compare against the vector norms, rows with a result only
    for lo in (0, 3):
        den = np.sqrt(o[lo] ** 2 + o[lo + 1] ** 2 + o[lo + 2] ** 2)
        err = np.sqrt(sum((g[lo + k] - o[lo + k]) ** 2 for k in range(3)))
        sel = den > 0
        assert np.all(err[~sel] == 0)
        assert np.max(err[sel] / den[sel]) < TOL
    sel = psc > 0
    assert np.all(g[6][~sel] == 0) and np.max(np.abs(g[6][sel] - o[6][sel]) / psc[sel]) < TOL
    return int((o[6] != 0).sum())


@pytest.mark.parametrize("cfg,N,scale", [(1, None, 1.0), (2, 20011, 10.0), (2, None, 1.0)])
def test_short_range_small(cfg, N, scale):
    w = make_workload(cfg, N=N, velocities=True)
    rout = scale * w.r_out
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, rout, oracle.OracleParams.from_workload(w))
    off, idx = T.neighbors()
    o = oracle.short_range(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rout, off, idx, w.G, w.r_in_over_r_out)
    g = _run(w, rout, off, idx)
    assert _compare(g, o, _pot_scale(w, off, idx)) > 100
    # momentum conservation of the result itself
    for k in range(6):
        assert abs(np.sum(w.m * g[k])) < 1e-10 * np.sum(w.m * np.abs(g[k]))


def test_short_range_full_size_config4_long_row():
    """Config 4 (N = 2^20, central mass with a row of > 1000 neighbours): the GPU's own neighbour list, every row."""
    import torch
    P = _P()
    w = make_workload(4, velocities=True)
    t = P.Tree(w.N, P.PetarParams.from_workload(w))
    t.upload(w.x, w.y, w.z, w.m, w.r_out)
    t.build()
    off, idx = t.neighbors()
    off, idx = off.cpu().numpy(), idx.cpu().numpy()
    assert np.diff(off).max() > 1000
    o = oracle.short_range(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, w.r_out, off, idx, w.G, w.r_in_over_r_out)
    g = _run(w, w.r_out, off, idx)
    assert _compare(g, o, _pot_scale(w, off, idx)) > 10000
    t.close()


def test_short_range_edge_cases():
    import torch
    P = _P()
    w = make_workload(1, N=300, velocities=True)
    # empty list: zeros everywhere; NULL outputs are skipped; N = 0; bad arguments
    off = np.zeros(w.N + 1, dtype=np.int64)
    g = _run(w, w.r_out, off, np.zeros(0, np.int32))
    assert all(np.all(v == 0) for v in g)
    ins = [_dev(a) for a in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, w.r_out)]
    ws = torch.empty(P.petar_short_range_workspace_bytes(w.N), dtype=torch.uint8, device="cuda")
    ax = torch.zeros(w.N, dtype=torch.float64, device="cuda")
    P.petar_short_range_force(*ins, _dev(off), _dev(np.zeros(1, np.int32)), w.N, 1.0, 0.1, (ax, None, None), (None, None, None), None, ws)
    P.petar_short_range_force(*ins, _dev(off), _dev(np.zeros(1, np.int32)), 0, 1.0, 0.1, (ax, None, None), (None, None, None), None, ws)
    with pytest.raises(P.PetarError):
        P.petar_short_range_force(*ins, _dev(off), _dev(np.zeros(1, np.int32)), w.N, 1.0, 1.5, (ax, None, None), (None, None, None), None, ws)
    with pytest.raises(P.PetarError):
        P.petar_short_range_force(*ins, _dev(off), _dev(np.zeros(1, np.int32)), w.N, 1.0, 0.1, (ax, None, None), (None, None, None), None, None)
