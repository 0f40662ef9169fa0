"""Pins of the oracle's part (C): Eq. 24 search radii, the Kepler-pericentre filter
 and the clustering.  Closed forms of conics, invariants, the O(N^2)
definition, scipy's connected components -- nothing here calls the CUDA path."""
import numpy as np
import pytest
from scipy.sparse import csr_matrix
from scipy.sparse.csgraph import connected_components

import oracle
from workloads import make_workload


def _rot(rng):
    q = rng.normal(size=4); q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def _conic_state(p, e, f, mu):
    """Position/velocity on a conic with semi-latus rectum p, eccentricity e at true anomaly f (textbook)."""
    r = p / (1 + e * np.cos(f))
    pos = np.array([r * np.cos(f), r * np.sin(f), 0.0])
    vel = np.sqrt(mu / p) * np.array([-np.sin(f), e + np.cos(f), 0.0])
    return pos, vel


@pytest.mark.parametrize("e", [0.0, 0.3, 0.9, 0.999, 1.0, 1.5, 7.0])
def test_pericentre_closed_form(e):
    """r_p = p / (1 + e): a(1-e) for an ellipse, p/2 for a parabola, a(e-1) for a hyperbola, at any phase."""
    rng = np.random.default_rng(int(e * 1000))
    for _ in range(20):
        mu, p = 10 ** rng.uniform(-6, 1), 10 ** rng.uniform(-5, 0)
        fmax = np.pi if e < 1 else 0.9 * np.arccos(-1 / e) if e > 1 else 0.9 * np.pi
        f = rng.uniform(-fmax, fmax)
        pos, vel = _conic_state(p, e, f, mu)
        R = _rot(rng)
        rp = oracle.pericentre(R @ pos, R @ vel, mu)
        # sqrt(mu^2 + 2 eps h^2) = mu e cancels for e -> 0: the formula is good to ~sqrt(ulp) there
        assert rp == pytest.approx(p / (1 + e), rel=1e-7)
        if e < 1:
            a = p / (1 - e * e)
            assert rp == pytest.approx(a * (1 - e), rel=1e-7)


def test_pericentre_special_cases():
    rng = np.random.default_rng(1)
    # mu = 0: straight line, r_p = impact parameter
    d, w = rng.normal(size=3), rng.normal(size=3)
    b = np.linalg.norm(np.cross(d, w)) / np.linalg.norm(w)
    assert oracle.pericentre(d, w, 0.0) == pytest.approx(b, rel=1e-12)
    # radial orbit: r_p = 0; at rest with mu = 0: r_p = r; coincident: 0
    assert oracle.pericentre(d, 2.5 * d, 1.0) == pytest.approx(0.0, abs=1e-14)
    assert oracle.pericentre(d, np.zeros(3), 0.0) == pytest.approx(np.linalg.norm(d))
    assert oracle.pericentre(np.zeros(3), w, 1.0) == 0.0
    # circular orbit: r_p = r
    r = 0.37; mu = 2.0
    assert oracle.pericentre([r, 0, 0], [0, np.sqrt(mu / r), 0], mu) == pytest.approx(r, rel=1e-12)
    # r_p <= r always, and symmetric under i <-> j (d, w -> -d, -w), bit for bit
    for _ in range(200):
        d, w, mu = rng.normal(size=3), rng.normal(size=3) * 10 ** rng.uniform(-2, 2), 10 ** rng.uniform(-3, 2)
        rp = oracle.pericentre(d, w, mu)
        assert 0.0 <= rp <= np.linalg.norm(d) * (1 + 1e-12)
        assert rp == oracle.pericentre(-d, -w, mu)


def test_eq24_search_radii():
    w = make_workload(2, N=3000, velocities=True)
    rnb = oracle.search_radii(w.vx, w.vy, w.vz, w.r_out, 3.0, w.dt_L)
    ref = w.r_out + 3.0 * np.sqrt(w.vx ** 2 + w.vy ** 2 + w.vz ** 2) * w.dt_L
    assert np.allclose(rnb, ref, rtol=1e-14) and np.all(rnb >= w.r_out)
    z = np.zeros(w.N)
    assert np.array_equal(oracle.search_radii(z, z, z, w.r_out, 3.0, w.dt_L), w.r_out)      # at rest: r_nb = r_out


def _rows(off, idx):
    return [set(idx[off[i]:off[i + 1]].tolist()) for i in range(len(off) - 1)]


@pytest.fixture(scope="module")
def small():
    w = make_workload(2, N=1500, velocities=True)
    # 8 dt_L: at N = 1500 the sphere is sparse; the longer step makes the fast particles' spheres sweep up candidates
    rnb = oracle.search_radii(w.vx, w.vy, w.vz, w.r_out, 3.0, 8 * w.dt_L)
    return w, rnb


def test_orbit_filter_definition_properties(small):
    w, rnb = small
    off, idx = oracle.neighbors_orbit_direct(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rnb, w.r_out, w.G, 1.5)
    rows = _rows(off, idx)
    assert all(i in rows[j] for i in range(w.N) for j in rows[i])                      # symmetric
    off0, idx0 = oracle.neighbors_direct(w.x, w.y, w.z, rnb)                           # stage (i) alone
    cand = _rows(off0, idx0)
    assert all(rows[i] <= cand[i] for i in range(w.N)) and off[-1] < off0[-1]          # a strict subset here
    offi, idxi = oracle.neighbors_orbit_direct(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rnb, w.r_out, w.G, 1e30)
    assert np.array_equal(offi, off0) and np.array_equal(idxi, idx0)                   # C_V -> inf: rule O9
    # every pair inside its changeover radius survives, whatever C_V
    offo, idxo = oracle.neighbors_direct(w.x, w.y, w.z, w.r_out)
    inner = _rows(offo, idxo)
    offz, idxz = oracle.neighbors_orbit_direct(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rnb, w.r_out, w.G, 0.0)
    assert all(inner[i] <= rows[i] for i in range(w.N)) and offo[-1] > 0
    assert np.array_equal(offz, offo) and np.array_equal(idxz, idxo)                   # C_V = 0: only those pairs
    # brute force in numpy for a few particles (independent restatement with the conic formula p/(1+e))
    for i in np.random.default_rng(0).choice(w.N, 12, replace=False):
        keep = set()
        for j in cand[i]:
            d = np.array([w.x[i] - w.x[j], w.y[i] - w.y[j], w.z[i] - w.z[j]])
            v = np.array([w.vx[i] - w.vx[j], w.vy[i] - w.vy[j], w.vz[i] - w.vz[j]])
            mu = w.G * (w.m[i] + w.m[j]); r = np.linalg.norm(d); h = np.cross(d, v)
            evec = np.cross(v, h) / mu - d / r
            rp = h.dot(h) / mu / (1 + np.linalg.norm(evec))
            if r < max(w.r_out[i], w.r_out[j]) or rp < 1.5 * min(rnb[i], rnb[j]):
                keep.add(j)
        assert keep == rows[i]


def test_orbit_filter_tree_equals_definition(small):
    w, rnb = small
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, oracle.OracleParams.from_workload(w), rsearch=rnb)
    off, idx = T.neighbors_orbit(w.vx, w.vy, w.vz, 1.5)
    offd, idxd = oracle.neighbors_orbit_direct(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rnb, w.r_out, w.G, 1.5)
    assert np.array_equal(off, offd) and np.array_equal(idx, idxd)


def test_clusters_are_connected_components(small):
    w, rnb = small
    off, idx = oracle.neighbors_orbit_direct(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rnb, w.r_out, w.G, 1.5)
    lab, nc = oracle.clusters(off, idx)
    g = csr_matrix((np.ones(len(idx)), idx, off), shape=(w.N, w.N))
    nref, lref = connected_components(g, directed=False)
    assert nc == nref
    # same partition, and the label is the smallest member
    first = {}
    for i, c in enumerate(lref):
        first.setdefault(c, i)
    assert np.array_equal(lab, np.array([first[c] for c in lref]))
    rows = _rows(off, idx)
    assert all(lab[j] == lab[i] for i in range(w.N) for j in rows[i])
    assert nc < w.N and np.sum(np.bincount(lab, minlength=w.N) == 1) > 0               # pairs and singletons both occur
    # degenerate graphs
    lab0, nc0 = oracle.clusters(np.zeros(6, dtype=np.int64), np.zeros(0, dtype=np.int32))
    assert nc0 == 5 and np.array_equal(lab0, np.arange(5))
    ring = np.array([[(i - 1) % 7, (i + 1) % 7] for i in range(7)], dtype=np.int32).ravel()
    lab1, nc1 = oracle.clusters(np.arange(0, 15, 2), ring)
    assert nc1 == 1 and np.all(lab1 == 0)


def test_generator_velocities():
    """Plummer model in Henon units: kinetic energy 1/4, sigma_1D = 0.409; binaries are bound with
    the semi-major axis that was drawn (vis-viva)."""
    w = make_workload(1, velocities=True)
    v2 = w.vx ** 2 + w.vy ** 2 + w.vz ** 2
    assert 0.5 * np.sum(w.m * v2) == pytest.approx(0.25, rel=0.05)
    assert np.sqrt(np.mean(v2) / 3) == pytest.approx(0.409, rel=0.05)
    assert w.dt_L == 2.0 ** -6
    w2 = make_workload(2, N=4000, velocities=True)
    plain = make_workload(2, N=4000)
    assert np.array_equal(w2.x, plain.x) and np.array_equal(w2.m, plain.m)            # positions do not depend on the flag
    off, idx = oracle.neighbors_direct(w2.x, w2.y, w2.z, np.full(w2.N, 1.1e-3))
    n_bound = 0
    for i in range(w2.N):
        for j in idx[off[i]:off[i + 1]]:
            d = np.array([w2.x[i] - w2.x[j], w2.y[i] - w2.y[j], w2.z[i] - w2.z[j]])
            v = np.array([w2.vx[i] - w2.vx[j], w2.vy[i] - w2.vy[j], w2.vz[i] - w2.vz[j]])
            mu = w2.m[i] + w2.m[j]
            inv_a = 2 / np.linalg.norm(d) - v.dot(v) / mu
            if inv_a > 0 and 0.99e-5 <= 1 / inv_a <= 1.01e-3:
                n_bound += 1
    assert n_bound >= 0.9 * 2 * w2.meta["n_pairs"] * 0.5      # most drawn pairs show up as bound pairs with a in range
