"""Pins of the oracle's tree algorithm (rules O1-O9) -- no GPU."""
import numpy as np
import pytest

import oracle
from workloads import make_workload


def _norm(a):
    return np.sqrt(a[0] ** 2 + a[1] ** 2 + a[2] ** 2)


@pytest.fixture(scope="module")
def w2k():
    w = make_workload(2, N=2048, seed=11)
    w.r_out = w.r_out * 4.0
    return w


def test_theta0_equals_direct_sum(w2k):
    """theta = 0: every leaf is opened, the tree result IS the definition."""
    w = w2k
    p = oracle.OracleParams.from_workload(w, theta=0.0)
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p)
    c, epep, epsp = T.walk_counts()
    assert np.all(c[:, 1] == w.N) and np.all(c[:, 2] == 0) and epsp == 0 and epep == w.N * w.N
    a = T.force()
    d = oracle.direct(w.x, w.y, w.z, w.m, w.r_out, p, "long")
    assert np.max(_norm([a[k] - d[k] for k in range(3)]) / _norm(d)) < 1e-11
    assert np.max(np.abs(a[3] - d[3]) / np.abs(d[3])) < 1e-12
    tot = np.array([np.sum(w.m * a[k]) for k in range(3)])
    assert np.all(np.abs(tot) < 1e-12 * np.sum(w.m * _norm(a)))


@pytest.mark.parametrize("theta", [0.3, 0.7])
def test_walk_partition_invariant(w2k, theta):
    """Every group's lists tile the whole system: n_ep + sum count(SP) = N, masses add up, no overlap."""
    w = w2k
    p = oracle.OracleParams.from_workload(w, theta=theta)
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p)
    nd = T.nodes()
    key, perm = T.keys()
    ms = w.m[perm]
    counts, epep, epsp = T.walk_counts()
    assert epsp > 0
    for g in range(0, T.n_groups, max(1, T.n_groups // 25)):
        sp, ep = T.walk_lists(g)
        cover = np.zeros(w.N, dtype=np.int32)
        for c in sp:
            cover[nd.begin[c]:nd.end[c]] += 1
        for b, e, near in ep:
            cover[b:e] += 1
        assert np.all(cover == 1)
        mass = sum(nd.M[c] for c in sp) + sum(ms[b:e].sum() for b, e, _ in ep)
        assert mass == pytest.approx(ms.sum(), rel=1e-12)
        assert counts[g, 1] == sum(e - b for b, e, _ in ep) and counts[g, 2] == len(sp)


def test_forced_open_gives_exact_neighbours(w2k):
    """Reading P9: every pair with r_ij < R_ij is an EP pair, so tree neighbours == O(N^2) definition."""
    w = w2k
    for theta in (0.3, 1.0):
        p = oracle.OracleParams.from_workload(w, theta=theta)
        T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p)
        off, idx = T.neighbors()
        off2, idx2 = oracle.neighbors_direct(w.x, w.y, w.z, w.r_out)
        assert off[-1] > 500
        assert np.array_equal(off, off2) and np.array_equal(idx, idx2)


def test_search_radius_hook(w2k):
    """r_search (NEXT-1 hook, Eq. 24): neighbours use max(rs_i, rs_j) and the walk opens accordingly."""
    w = w2k
    rs = w.r_out * 2.5
    p = oracle.OracleParams.from_workload(w)
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p, rsearch=rs)
    off, idx = T.neighbors()
    off2, idx2 = oracle.neighbors_direct(w.x, w.y, w.z, rs)
    assert np.array_equal(off, off2) and np.array_equal(idx, idx2)


def test_tree_structure_geometry(w2k):
    """Keys/sort/octree are consistent with geometry: each node's members lie in ONE grid cube of its level."""
    w = w2k
    p = oracle.OracleParams.from_workload(w)
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p)
    c, h = T.root()
    pos = np.stack([w.x, w.y, w.z], 1)
    assert h == 2.0 ** round(np.log2(h)) and np.all(np.abs(pos - c) < h)
    key, perm = T.keys()
    assert np.array_equal(np.sort(perm), np.arange(w.N))
    assert np.all(np.diff(key.astype(np.float64)) >= 0)
    same = np.diff(key.astype(np.int64)) == 0
    assert np.all(np.diff(perm)[same] > 0)                       # ties by original index (O4)
    nd = T.nodes()
    ps = pos[perm]
    assert nd.level[0] == 0 and nd.begin[0] == 0 and nd.end[0] == w.N
    for n in range(T.n_nodes):
        b, e, l = nd.begin[n], nd.end[n], nd.level[n]
        edge = 2 * h / 2 ** l
        cell = np.floor((ps[b:e] - (c - h)) / edge)
        assert np.all(cell == cell[0])
        cnt = e - b
        assert nd.leaf[n] == int(cnt <= 8 or l == 21)
        assert np.all(nd.lo[n] == ps[b:e].min(0)) and np.all(nd.hi[n] == ps[b:e].max(0))
        assert nd.rmax[n] == w.r_out[perm][b:e].max()
    # children tile the parent: nodes of one level are disjoint and sorted
    for l in range(1, nd.level.max() + 1):
        sel = nd.level == l
        assert np.all(nd.begin[sel][1:] >= nd.end[sel][:-1])
    # moments of the root and of every node against numpy
    ms = w.m[perm]
    assert nd.M[0] == pytest.approx(ms.sum(), rel=1e-14)
    assert np.allclose(nd.com[0], (ms[:, None] * ps).sum(0) / ms.sum(), rtol=0, atol=1e-13)
    for n in range(0, T.n_nodes, 7):
        b, e = nd.begin[n], nd.end[n]
        M = ms[b:e].sum()
        com = (ms[b:e, None] * ps[b:e]).sum(0) / M
        d = ps[b:e] - com
        Q = np.array([(ms[b:e] * d[:, i] * d[:, j]).sum() for i, j in ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))])
        assert nd.M[n] == pytest.approx(M, rel=1e-13)
        assert np.allclose(nd.com[n], com, rtol=0, atol=1e-12)
        assert np.allclose(nd.Q[n], Q, rtol=1e-9, atol=1e-18)
    # groups: <= 64 members, consecutive, cover everything
    gb, ge, glo, ghi, grmax = T.groups()
    assert gb[0] == 0 and ge[-1] == w.N and np.array_equal(gb[1:], ge[:-1]) and np.all(ge - gb <= 64)
    for g in range(T.n_groups):
        assert np.all(glo[g] == ps[gb[g]:ge[g]].min(0)) and np.all(ghi[g] == ps[gb[g]:ge[g]].max(0))


def test_multipole_error_orders():
    """Two equal masses at +-d seen from distance r: monopole error ~ (d/r)^2, quadrupole error ~ (d/r)^4."""
    errs = {1: [], 2: []}
    for mult in (1, 2):
        for d in (0.02, 0.01):
            x = np.array([10.0, -0.3 + d, -0.3 - d]); y = np.array([0.2, -0.3, -0.3 + 0.0]); z = np.array([0.1, -0.3, -0.3])
            m = np.array([1.0, 0.5, 0.5]); rout = np.full(3, 1e-3)
            p = oracle.OracleParams.make(theta=1.0, multipole=mult, n_leaf=2, n_group=1)
            T = oracle.OracleTree(x, y, z, m, rout, p)
            sp, ep = T.walk_lists(int(np.where(T.keys()[1] == 0)[0][0]) if False else 0)
            a = T.force()
            ex = oracle.direct(x, y, z, m, rout, p, "newton")
            # the far particle (index 0) must have used the pair's cell as a super-particle
            counts, _, epsp = T.walk_counts()
            assert epsp >= 1
            errs[mult].append((abs(a[0][0] - ex[0][0]) / abs(ex[0][0]), abs(a[3][0] - ex[3][0]) / abs(ex[3][0])))
    r1 = errs[1][0][0] / errs[1][1][0]; r2 = errs[2][0][0] / errs[2][1][0]
    assert 3.5 < r1 < 4.5, errs
    assert 13.0 < r2 < 19.0, errs
    assert 3.5 < errs[1][0][1] / errs[1][1][1] < 4.5 and 13.0 < errs[2][0][1] / errs[2][1][1] < 19.0
    assert errs[2][0][0] < errs[1][0][0] * 1e-2


def test_single_particle_cell_is_exact():
    """A one-particle cell accepted as super-particle gives exactly the pair term (Q = 0, com = position)."""
    x = np.array([5.0, -1.0, -1.2, 3.0]); y = np.array([0.1, -1.0, 0.7, -2.0]); z = np.array([0.3, 0.2, -1.0, 1.0])
    m = np.array([0.4, 0.3, 0.2, 0.1]); rout = np.full(4, 1e-3)
    p = oracle.OracleParams.make(theta=2.0, multipole=2, n_leaf=1, n_group=1)
    T = oracle.OracleTree(x, y, z, m, rout, p)
    _, epep, epsp = T.walk_counts()
    assert epsp > 0
    a = T.force(); ex = oracle.direct(x, y, z, m, rout, p, "newton")
    for k in range(4):
        assert np.allclose(a[k], ex[k], rtol=1e-13)


def test_unpinned_sanity_counts_and_error_vs_theta():
    """PARITY UNPINNED (the paper prints no counts or errors): only monotonicity with theta, quadrupole < monopole."""
    w = make_workload(1, N=4096)
    d = oracle.direct(w.x, w.y, w.z, w.m, w.r_out, oracle.OracleParams.from_workload(w), "long")
    last_n, last_err = None, None
    for theta in (0.2, 0.4, 0.8):
        e = {}
        for mult in (1, 2):
            p = oracle.OracleParams.from_workload(w, theta=theta, multipole=mult)
            T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, p)
            _, epep, epsp = T.walk_counts()
            a = T.force()
            rel = _norm([a[k] - d[k] for k in range(3)]) / _norm(d)
            e[mult] = np.sqrt(np.mean(rel ** 2))
        assert e[2] < e[1]
        if last_n is not None:
            assert epep + epsp < last_n and e[2] > last_err
        last_n, last_err = epep + epsp, e[2]
    assert last_err < 5e-3      # theta < 1 keeps the force accurate enough for relaxation


def test_degenerate_inputs():
    p = oracle.OracleParams.make(theta=0.3, multipole=2)
    T = oracle.OracleTree(np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(0), p)
    assert T.n_nodes == 0 and T.n_groups == 0
    # N <= leaf limit: root is a leaf and the only group
    rng = np.random.default_rng(3)
    pos = rng.normal(size=(5, 3)); m = np.full(5, 0.2); rout = np.full(5, 0.01)
    T = oracle.OracleTree(pos[:, 0], pos[:, 1], pos[:, 2], m, rout, p)
    assert T.n_nodes == 1 and T.n_groups == 1
    a = T.force(); d = oracle.direct(pos[:, 0], pos[:, 1], pos[:, 2], m, rout, p, "long")
    assert np.allclose(a[0], d[0], rtol=1e-13)
    # 100 coincident particles: over-full level-21 leaf cut into chunks of 64; zero force, finite potential
    n = 100
    T = oracle.OracleTree(np.full(n, 0.5), np.full(n, -0.25), np.full(n, 2.0), np.full(n, 0.01), np.full(n, 0.1), p)
    gb, ge, *_ = T.groups()
    assert list(ge - gb) == [64, 36]
    a = T.force()
    assert np.all(a[0] == 0) and np.allclose(a[3], -99 * 0.01 * 2.0 / (0.1 + 0.01), rtol=1e-13)
    # zero-mass measure points are ordinary i-particles
    m0 = m.copy(); m0[2] = 0.0
    T = oracle.OracleTree(pos[:, 0], pos[:, 1], pos[:, 2], m0, rout, p)
    a = T.force(); d = oracle.direct(pos[:, 0], pos[:, 1], pos[:, 2], m0, rout, p, "long")
    assert np.allclose(a[1], d[1], rtol=1e-13) and np.all(np.isfinite(a[0]))


@pytest.mark.parametrize("mirror", [(0, 0, 0), (1, 0, 0), (1, 1, 1)])
def test_opening_criterion_flips_at_hand_computed_theta(mirror):
    """Pin of reading P8 (PAPER.md:207 "inside theta ... centre-of-the-mass", :152 theta < 1): a cell is accepted iff
    l < theta * d, l = edge of its CUBE, d = distance from the group's tight BOX to the cell's CENTRE OF MASS.

    Worked by hand on dyadic coordinates (all values exact in binary).  Anchors at (0,0,0) and (15,15,15) give, by rule O1,
    c = 7.5, L = 15, v = 7.5 (1 + 2^-20), h = 8: the root cube is [-0.5, 15.5]^3, level-1 edges are 8, level-2 edges 4.
      cell C  = level-2 cube [11.5,15.5] x [-0.5,3.5] x [-0.5,3.5], l = 4, holding p1 = (12,1,1) with mass 3 and
                p2 = (15,3,1) with mass 1: com = (12.75, 1.5, 1) -- not the cube centre (13.5, 1.5, 1.5);
                a leaf with n_leaf = 2; its level-1 parent also holds p3 = (9,6,6), so the parent is split;
      group G = level-1 cube [-0.5,7.5]^3 with (0,0,0) and (2,1,0): 2 = n_group members, box [0,2] x [0,1] x [0,0].
    d^2 = (12.75-2)^2 + (1.5-1)^2 + (1-0)^2 = 115.5625 + 0.25 + 1 = 116.8125, so C flips at theta* = 4/sqrt(116.8125) = 0.370099...
    Thresholds a misreading would give instead (each at least 6 % away from theta*):
      half edge (l = 2)                       2/sqrt(116.8125) = 0.18505
      tight box of C as l (longest side 3)    3/sqrt(116.8125) = 0.27757
      cube centre of C instead of its com     4/sqrt(11.5^2 + 0.5^2 + 1.5^2) = 4/sqrt(134.75)   = 0.34458
      centre of G (1, 0.5, 0) instead of box  4/sqrt(11.75^2 + 1 + 1)        = 4/sqrt(140.0625) = 0.33799
      box of G to tight box of C              4/sqrt(10^2 + 0 + 1)           = 4/sqrt(101)      = 0.39801
      l^2 < theta d^2 (theta not squared)     16/116.8125                                       = 0.13697
    All but one lie below theta* (they would still accept C just below it), box-to-box lies above (it would still open C
    just above it); both sides of the flip are asserted.  The mirrored cases put the cell on the low side of the group, so
    both arms of max(0, lo_g - com, com - hi_g) are used on every axis."""
    pts = np.array([[0, 0, 0], [2, 1, 0],                    # group G
                    [12, 1, 1], [15, 3, 1],                  # cell C
                    [9, 6, 6],                               # makes C's level-1 parent split
                    [15, 15, 15]], dtype=np.float64)         # anchor
    m = np.array([1.0, 1.0, 3.0, 1.0, 1.0, 1.0])
    for k in range(3):
        if mirror[k]:
            pts[:, k] = 15.0 - pts[:, k]                     # the root cube [-0.5, 15.5] maps onto itself
    rout = np.full(6, 1e-3)                                  # nothing comes near: the forced-open rule stays out of it
    d2 = 10.75 ** 2 + 0.5 ** 2 + 1.0 ** 2
    assert d2 == 116.8125
    theta_star = 4.0 / np.sqrt(d2)
    for wrong in (2 / np.sqrt(d2), 3 / np.sqrt(d2), 4 / np.sqrt(134.75), 4 / np.sqrt(140.0625), 4 / np.sqrt(101.0), 16 / d2):
        assert abs(wrong / theta_star - 1.0) > 0.06

    def lists(theta):
        p = oracle.OracleParams.make(theta=theta, multipole=2, n_leaf=2, n_group=2)
        T = oracle.OracleTree(pts[:, 0], pts[:, 1], pts[:, 2], m, rout, p)
        c, h = T.root()
        assert np.array_equal(c, [7.5, 7.5, 7.5]) and h == 8.0                               # rule O1 as worked above
        nd = T.nodes()
        lo_c, hi_c = pts[2:4].min(0), pts[2:4].max(0)
        cell = [n for n in range(T.n_nodes) if nd.level[n] == 2 and np.array_equal(nd.lo[n], lo_c) and np.array_equal(nd.hi[n], hi_c)]
        assert len(cell) == 1 and nd.leaf[cell[0]] == 1 and nd.M[cell[0]] == 4.0
        com = (3.0 * pts[2] + 1.0 * pts[3]) / 4.0
        assert np.array_equal(nd.com[cell[0]], com) and abs(com[0] - 7.5) == 5.25            # 12.75 or its mirror image 2.25
        gb, ge, glo, ghi, _ = T.groups()
        grp = [g for g in range(T.n_groups) if np.array_equal(glo[g], pts[0:2].min(0)) and np.array_equal(ghi[g], pts[0:2].max(0))]
        assert len(grp) == 1 and ge[grp[0]] - gb[grp[0]] == 2
        sp, ep = T.walk_lists(grp[0])
        return cell[0], (int(nd.begin[cell[0]]), int(nd.end[cell[0]])), set(sp.tolist()), {(int(b), int(e)) for b, e, _ in ep}

    cid, rng_c, sp, ep = lists(theta_star * (1 + 1e-12))
    assert cid in sp and rng_c not in ep                     # l < theta d: accepted as one super-particle
    cid, rng_c, sp, ep = lists(theta_star * (1 - 1e-12))
    assert cid not in sp and rng_c in ep                     # l > theta d: opened, and C being a leaf its two particles are listed
    # far from the flip on either side, for good measure
    cid, rng_c, sp, ep = lists(0.36)
    assert cid not in sp and rng_c in ep
    cid, rng_c, sp, ep = lists(0.38)
    assert cid in sp and rng_c not in ep
