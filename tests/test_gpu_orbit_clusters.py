"""GPU parity of SURVEY.md 8(f) ranks 1-2 through the C-ABI: Eq. 24 search radii, the orbit-dependent
two-stage neighbour criterion (rule O10) and the clustering, against the oracle, bit for bit."""
import numpy as np
import pytest

import oracle
from workloads import make_workload

pytestmark = pytest.mark.gpu
C_R, C_V = 3.0, 1.5


def _P():
    import paper_2006_16560_b200 as P
    return P


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _np(t):
    return t.cpu().numpy()


def _setup(cfg, N=None, dt_factor=1.0):
    import torch
    P = _P()
    w = make_workload(cfg, N=N, velocities=True)
    dt = w.dt_L * dt_factor
    v = [_dev(a) for a in (w.vx, w.vy, w.vz)]
    rnb_dev = torch.empty(w.N, dtype=torch.float64, device="cuda")
    P.petar_search_radii(*v, _dev(w.r_out), C_R, dt, w.N, rnb_dev)
    rnb = oracle.search_radii(w.vx, w.vy, w.vz, w.r_out, C_R, dt)
    assert np.array_equal(_np(rnb_dev), rnb)                                    # Eq. 24, bit for bit
    params = P.PetarParams.from_workload(w)
    t = P.Tree(w.N, params)
    t.upload(w.x, w.y, w.z, w.m, w.r_out, rnb)
    t.build()
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, oracle.OracleParams.from_workload(w), rsearch=rnb)
    return w, v, rnb, t, T


def _sorted_rows(off, idx, n):
    rows = np.repeat(np.arange(n), np.diff(off))
    return idx[np.lexsort((idx, rows))]


def _check_clusters(t, off_dev, idx_dev, off, idx, n):
    lab, ncl, coff, mem = t.clusters(off_dev, idx_dev)
    olab, onc = oracle.clusters(off, idx)
    assert int(ncl.item()) == onc
    assert np.array_equal(_np(lab), olab)
    coff, mem = _np(coff), _np(mem)
    assert coff[onc] == n and coff[0] == 0
    # clusters in ascending label order, members ascending: exactly a stable sort by label
    order = np.lexsort((np.arange(n), olab))
    assert np.array_equal(mem, order)
    starts = np.flatnonzero(np.r_[True, olab[order][1:] != olab[order][:-1]])
    assert np.array_equal(coff[:onc], starts)
    return olab, onc


@pytest.mark.parametrize("cfg,N,dtf", [(1, None, 1.0), (2, 20011, 8.0), (2, None, 1.0)])
def test_orbit_neighbours_and_clusters_small(cfg, N, dtf):
    w, v, rnb, t, T = _setup(cfg, N, dtf)
    off_dev, idx_dev = t.neighbors_orbit(*v, C_V)
    off, idx = _np(off_dev), _np(idx_dev)
    ooff, oidx = T.neighbors_orbit(w.vx, w.vy, w.vz, C_V)
    assert np.array_equal(off, ooff)
    assert np.array_equal(_sorted_rows(off, idx, w.N), oidx)
    # the filter is a subset of the plain list with the same radii, and the plain list is unchanged by it
    off0, idx0 = t.neighbors()
    poff, pidx = T.neighbors()
    assert np.array_equal(_np(off0), poff) and off[-1] <= poff[-1]
    assert np.array_equal(_sorted_rows(_np(off0), _np(idx0), w.N), pidx)
    if dtf > 1:
        assert off[-1] < poff[-1]                                               # stage (ii) removes candidates here
    off_dev, idx_dev = t.neighbors_orbit(*v, C_V)
    _check_clusters(t, off_dev, idx_dev, off, _sorted_rows(off, idx, w.N), w.N)
    assert _P().petar_tree_status(t.handle) == 0
    t.close()


def test_orbit_and_clusters_full_size_config3():
    """Config 3 (N = 2^20, 100 % binaries): rows of sampled i-groups against the oracle; clusters against the oracle's
    union-find run on the GPU's own (bit-exact, see above) list."""
    w, v, rnb, t, T = _setup(3)
    off_dev, idx_dev = t.neighbors_orbit(*v, C_V)
    off, idx = _np(off_dev), _np(idx_dev)
    rng = np.random.default_rng(3)
    sel = np.sort(rng.choice(T.n_groups, size=300, replace=False))
    ooff, oidx = T.neighbors_orbit(w.vx, w.vy, w.vz, C_V, sel)
    key, perm = T.keys()
    gb, ge, *_ = T.groups()
    checked = 0
    for g in sel:
        for o in perm[gb[g]:ge[g]]:
            row = np.sort(idx[off[o]:off[o + 1]])
            assert np.array_equal(row, oidx[ooff[o]:ooff[o + 1]])
            checked += len(row)
    assert checked > 1000
    rows = np.repeat(np.arange(w.N), np.diff(off))
    assert np.array_equal(np.sort(rows * (1 << 21) + idx), np.sort(idx.astype(np.int64) * (1 << 21) + rows))   # symmetric
    olab, onc = _check_clusters(t, off_dev, idx_dev, off, _sorted_rows(off, idx, w.N), w.N)
    assert np.all(olab[idx] == olab[rows])
    assert 0.4 * w.N < onc < 0.6 * w.N                                           # mostly the binaries themselves
    t.close()


def test_clusters_edge_cases():
    import torch
    P = _P()
    # no edges: every particle its own cluster; a single chain: one cluster; labels only (no member lists)
    n = 1000
    off = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    idx = torch.zeros(1, dtype=torch.int32, device="cuda")
    lab = torch.empty(n, dtype=torch.int32, device="cuda"); ncl = torch.zeros(1, dtype=torch.int64, device="cuda")
    P.petar_clusters(off, idx, n, lab, ncl)
    assert int(ncl.item()) == n and np.array_equal(_np(lab), np.arange(n))
    chain = np.array([[max(i - 1, 0), min(i + 1, n - 1)] for i in range(n)], dtype=np.int32)
    offc = np.arange(0, 2 * n + 1, 2, dtype=np.int64)
    P.petar_clusters(_dev(offc), _dev(chain.ravel()), n, lab, ncl)
    assert int(ncl.item()) == 1 and np.all(_np(lab) == 0)
    # random sparse symmetric graph against the oracle
    rng = np.random.default_rng(5)
    e = rng.integers(0, n, size=(600, 2)); e = e[e[:, 0] != e[:, 1]]
    e = np.unique(np.concatenate([e, e[:, ::-1]]), axis=0)
    offr = np.zeros(n + 1, dtype=np.int64); np.add.at(offr, e[:, 0] + 1, 1); offr = np.cumsum(offr)
    idxr = e[:, 1].astype(np.int32)
    P.petar_clusters(_dev(offr), _dev(idxr), n, lab, ncl)
    olab, onc = oracle.clusters(offr, idxr)
    assert int(ncl.item()) == onc and np.array_equal(_np(lab), olab)
    # N = 0 and bad arguments
    P.petar_clusters(off, idx, 0, lab, ncl)
    assert int(ncl.item()) == 0
    with pytest.raises(P.PetarError):
        P.petar_clusters(off, idx, n, lab, ncl, torch.zeros(n + 1, dtype=torch.int64, device="cuda"), None, None)    # no workspace
    with pytest.raises(P.PetarError):
        P.petar_search_radii(lab, lab, lab, lab, -1.0, 0.1, n, lab)


def test_orbit_list_degenerate_cases():
    """At rest r_nb = r_out and stage (ii) keeps every candidate (all are inside their changeover radius): the orbit
    list equals the plain one.  N = 0 and bad arguments."""
    import torch
    P = _P()
    w = make_workload(2, N=9001)
    z = torch.zeros(w.N, dtype=torch.float64, device="cuda")
    t = P.Tree(w.N, P.PetarParams.from_workload(w))
    t.upload(w.x, w.y, w.z, w.m, w.r_out)
    t.build()
    off0, idx0 = (_np(v).copy() for v in t.neighbors())
    off1, idx1 = (_np(v).copy() for v in t.neighbors_orbit(z, z, z, 0.0))
    assert np.array_equal(off0, off1) and np.array_equal(_sorted_rows(off0, idx0, w.N), _sorted_rows(off1, idx1, w.N))
    with pytest.raises(P.PetarError):
        P.petar_neighbor_list_orbit(t.handle, z, z, z, -1.0, t.offsets, None, 0)
    with pytest.raises(P.PetarError):
        P.petar_neighbor_list_orbit(t.handle, None, z, z, 1.5, t.offsets, None, 0)
    t.close()
    h = P.petar_tree_build(None, None, None, None, None, None, 0, P.PetarParams.make(theta=0.3, multipole=2), None)
    off = torch.full((1,), 7, dtype=torch.int64, device="cuda")
    P.petar_neighbor_list_orbit(h, None, None, None, 1.5, off, None, 0)
    torch.cuda.synchronize()
    assert int(off[0]) == 0
    P.petar_tree_destroy(h)
