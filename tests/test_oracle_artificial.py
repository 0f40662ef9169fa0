"""Pins of the oracle's part (E): kick, pseudoparticles (Eq. 36-38), tidal-tensor measure points and fit
(Eq. 25-28, Table 1).  The expected values are the paper's own prints (tests/golden/tidal_tensor_table1.txt,
Eq. 36, Eq. 37, the condition numbers of :414) and textbook facts -- nothing here calls the CUDA path."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import artificial as A

GOLD = os.path.join(os.path.dirname(__file__), "golden", "tidal_tensor_table1.txt")


def _golden_rows():
    rows = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, body = line.split(":")
        order, name = head.split()
        terms = []
        for t in body.split(";"):
            val, comp, pt = t.split()
            terms.append((eval(val, {"s2": np.sqrt(2.0)}), "xyz".index(comp), int(pt)))
        rows[(int(order), name)] = terms
    return rows


def test_generalized_inverse_reproduces_table1():
    """The least-squares inverse of Eq. 28 built from Table 1's polynomial and measure points has exactly the rows
    the paper prints (all 22 rows of the table: 6 of the second order, 16 of the third)."""
    rows = _golden_rows()
    assert len(rows) == 22 and sum(1 for (o, _) in rows if o == 2) == 6
    for order in (2, 3):
        Pi = np.linalg.pinv(A.tidal_design_matrix(order))
        names = A.T2_NAMES if order == 2 else A.T3_NAMES
        for (o, name), terms in rows.items():
            if o != order:
                continue
            expect = np.zeros(Pi.shape[1])
            for val, comp, pt in terms:
                expect[3 * (pt - 1) + comp] = val
            assert np.allclose(Pi[names.index(name)], expect, atol=1e-12), (order, name)


def test_condition_numbers_of_the_paper():
    """"the condition numbers ... are small: 2 and 12.7" -- these are the ratios of the extreme
    singular values of M^T M (the normal equations), i.e. cond(M)^2."""
    c2 = np.linalg.cond(A.tidal_design_matrix(2)) ** 2
    c3 = np.linalg.cond(A.tidal_design_matrix(3)) ** 2
    assert c2 == pytest.approx(2.0, rel=1e-12)
    assert round(c3, 1) == 12.7
    # an octahedron (6 points) does not give full rank for the third order (:410)
    octa = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=float)
    M = np.concatenate([A._design_rows(3, p) for p in octa])
    assert np.linalg.matrix_rank(M) < 16
    # geometry: the tetrahedron is regular with edge 2 d_c
    P = A.TT_POINTS[2]
    assert np.allclose([np.linalg.norm(P[i] - P[j]) for i in range(4) for j in range(i)], 2.0)


def _point_mass_field(r, src, m):
    d = src - r
    return m * d / np.linalg.norm(d) ** 3


def test_tidal_fit_recovers_a_tidal_field():
    rng = np.random.default_rng(0)
    cm = rng.normal(size=3)
    src = cm + np.array([3.0, -2.0, 1.5]); m = 2.5
    acm = _point_mass_field(cm, src, m)
    errs = {2: [], 3: []}
    for order in (2, 3):
        for d_c in (0.02, 0.01):
            pts = A.tidal_points(order, cm, d_c)
            T = A.tidal_fit(order, d_c, np.array([_point_mass_field(p, src, m) for p in pts]), acm)
            probe = np.array([0.3, -0.7, 0.5]) * d_c
            err = np.linalg.norm(A.tidal_eval(order, T, acm, probe) - _point_mass_field(cm + probe, src, m))
            errs[order].append(err)
            if order == 2:
                # A_ij is the tidal tensor of the point mass: m (3 n n^T - 1) / R^3, symmetric and traceless
                R = np.linalg.norm(src - cm); n = (src - cm) / R
                tt = m * (3 * np.outer(n, n) - np.eye(3)) / R ** 3
                fit = np.array([[T[0], T[1], T[2]], [T[1], T[3], T[4]], [T[2], T[4], T[5]]])
                assert np.allclose(fit, tt, atol=0.05 * d_c)       # the 4 points see the next order at O(d_c / R)
    # truncation error falls like d_c^2 (second order) and d_c^3 (third order)
    assert errs[2][0] / errs[2][1] == pytest.approx(4.0, rel=0.1)
    assert errs[3][0] / errs[3][1] == pytest.approx(8.0, rel=0.15)
    assert errs[3][1] < 0.05 * errs[2][1]
    # an exactly quadratic field is reproduced exactly by the third-order fit
    Tq = rng.normal(size=16)
    pts = A.TT_POINTS[3] * 0.3
    acc = np.array([A.tidal_eval(3, Tq, np.zeros(3), p) for p in pts])
    assert np.allclose(A.tidal_fit(3, 0.3, acc, np.zeros(3)), Tq, atol=1e-12)


@pytest.mark.parametrize("e", [0.0, 0.3, 0.9])
def test_eq36_eq37_eq38(e):
    m1, m2, a = 0.7, 0.2, 1.3
    mu = m1 * m2 / (m1 + m2)
    Aavg = A.orbit_average_quadrupole(m1, m2, a, e)
    eq36 = mu * a * a * np.diag([2 * e * e + 0.5, 0.5 - 0.5 * e * e, 0.0])
    assert np.allclose(Aavg, eq36, atol=1e-9)
    eq37 = 0.25 * mu * a * a * np.diag([9 * e * e + 1, 1 - 6 * e * e, -3 * e * e - 2])
    assert np.allclose(1.5 * eq36 - 0.5 * np.trace(eq36) * np.eye(3), eq37, atol=1e-14)        # Eq. 31
    # Eq. 38: three equal masses with no dipole and exactly that quadrupole
    P, Q = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    pos, mp = A.pseudoparticles(m1, m2, a, e, P, Q, np.zeros(3))
    assert mp == pytest.approx((m1 + m2) / 3)
    assert np.allclose(pos.sum(axis=0), 0, atol=1e-15)
    quad = mp * np.einsum("ni,nj->ij", pos, pos)
    assert np.allclose(quad, eq36, atol=1e-14)


def test_kepler_elements_and_artificial_particles():
    rng = np.random.default_rng(3)
    for _ in range(20):
        m1, m2 = 10 ** rng.uniform(-3, 0, 2)
        a, e, E = 10 ** rng.uniform(-4, -1), rng.uniform(0, 0.95), rng.uniform(0, 2 * np.pi)
        mu = m1 + m2
        # state from Eq. 32 and its time derivative, random orientation
        q = rng.normal(size=4); q /= np.linalg.norm(q)
        w_, x_, y_, z_ = q
        Rm = np.array([[1 - 2 * (y_ * y_ + z_ * z_), 2 * (x_ * y_ - z_ * w_), 2 * (x_ * z_ + y_ * w_)],
                       [2 * (x_ * y_ + z_ * w_), 1 - 2 * (x_ * x_ + z_ * z_), 2 * (y_ * z_ - x_ * w_)],
                       [2 * (x_ * z_ - y_ * w_), 2 * (y_ * z_ + x_ * w_), 1 - 2 * (x_ * x_ + y_ * y_)]])
        d = Rm @ np.array([a * (np.cos(E) - e), a * np.sqrt(1 - e * e) * np.sin(E), 0])
        fac = np.sqrt(mu / a ** 3) * a / (1 - e * np.cos(E))
        w = Rm @ np.array([-fac * np.sin(E), fac * np.sqrt(1 - e * e) * np.cos(E), 0])
        el = A.kepler_elements(d, w, mu)
        assert el["bound"] and el["a"] == pytest.approx(a, rel=1e-9) and el["e"] == pytest.approx(e, abs=1e-8)
        if e > 1e-3:
            assert np.allclose(el["P"], Rm[:, 0], atol=1e-6) and np.allclose(el["W"], Rm[:, 2], atol=1e-9)
        x1 = rng.normal(size=3); v1 = rng.normal(size=3)
        art = A.artificial_particles(x1, v1, m1, x1 + d, v1 + w, m2, 1.0, 3, 2.0)
        assert art["pos"].shape == (12, 3) and art["d_c"] == pytest.approx(2.0 * a, rel=1e-9)
        assert np.all(art["mass"][:9] == 0) and np.allclose(art["mass"][9:], (m1 + m2) / 3)
        assert np.allclose(art["pos"][8], art["cm"])
        assert np.allclose((art["mass"][:, None] * art["pos"]).sum(axis=0), (m1 + m2) * art["cm"], rtol=1e-12)   # same monopole, no dipole
    # unbound pair: flagged, everything at the centre of mass
    art = A.artificial_particles([0, 0, 0], [0, 0, 0], 1.0, [1, 0, 0], [0, 5.0, 0], 1.0, 1.0, 2, 2.0)
    assert not art["bound"] and np.allclose(art["pos"], art["cm"])
    assert np.array_equal(A.kick(np.array([1.0, 2.0]), np.array([0.5, -1.0]), 0.25), np.array([1.125, 1.75]))


@pytest.mark.parametrize("e", [0.0, 0.5, 0.9])
def test_orbit_sampling_eq29(e):
    m1, m2, a = 0.7, 0.2, 1.3
    P, Q, cm = np.array([1.0, 0, 0]), np.array([0, 1.0, 0]), np.array([0.3, -0.2, 0.1])
    pos, mass = A.orbit_sampling(m1, m2, a, e, P, Q, cm, 8)
    assert pos.shape == (16, 3)                                              # "dE = pi/4, 16 particles"
    # the mean-anomaly intervals tile the orbit: the samples of a component carry exactly its mass
    assert mass[:8].sum() == pytest.approx(m1, rel=1e-14) and mass[8:].sum() == pytest.approx(m2, rel=1e-14)
    # Eq. 29's two forms agree: dE - e [sin(E + dE/2) - sin(E - dE/2)] = dE - 2 e cos E sin(dE/2)
    dE = np.pi / 4; E = np.arange(8) * dE
    assert np.allclose(mass[:8] * 2 * np.pi / m1, dE - e * (np.sin(E + dE / 2) - np.sin(E - dE / 2)), rtol=1e-13)
    # no dipole about the centre of mass pair by pair, and the sampled quadrupole converges to Eq. 36
    assert np.allclose(m1 * (pos[:8] - cm) + m2 * (pos[8:] - cm), 0, atol=1e-15)
    mu = m1 * m2 / (m1 + m2)
    eq36 = mu * a * a * np.diag([2 * e * e + 0.5, 0.5 - 0.5 * e * e, 0.0])
    errs = []
    for n in (8, 64):
        p_, m_ = A.orbit_sampling(m1, m2, a, e, P, Q, np.zeros(3), n)
        errs.append(np.abs(np.einsum("n,ni,nj->ij", m_, p_, p_) - eq36).max())
    assert errs[1] < 1e-2 * mu * a * a and errs[1] <= errs[0] + 1e-15
