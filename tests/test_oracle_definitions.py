"""Pins of the oracle's O(N^2) definitions (Eq. 7, Eq. 11) -- no GPU."""
import numpy as np
import pytest

import oracle
from workloads import make_workload, plummer_positions, PLUMMER_A


def _norm(a):
    return np.sqrt(a[0] ** 2 + a[1] ** 2 + a[2] ** 2)


@pytest.fixture(scope="module")
def small():
    # Kroupa masses + 50 % binaries, radii large enough that many pairs sit inside the changeover zone
    w = make_workload(2, N=768, seed=7)
    w.r_out = w.r_out * 8.0
    return w, oracle.OracleParams.from_workload(w)


def test_long_plus_short_is_newton(small):
    """Eq. 7 / Eq. 11: H = H_L + H_S  =>  a_L + a_S = a_Newton and phi_L + phi_S = phi_Newton."""
    w, p = small
    args = (w.x, w.y, w.z, w.m, w.r_out, p)
    L, S, Nw = (oracle.direct(*args, k) for k in ("long", "short", "newton"))
    scale = _norm(Nw)
    for k in range(3):
        assert np.max(np.abs(L[k] + S[k] - Nw[k]) / scale) < 1e-11
    assert np.max(np.abs(L[3] + S[3] - Nw[3]) / np.abs(Nw[3])) < 1e-12
    # the split is not trivial: both parts carry a sizeable share somewhere
    assert np.max(_norm(S) / scale) > 0.5 and np.max(_norm(L) / scale) > 0.5


def test_newton_against_numpy_definition(small):
    """The Newtonian leg against the textbook double sum written with numpy broadcasting."""
    w, p = small
    d = np.stack([w.x, w.y, w.z], 1)
    dr = d[None, :, :] - d[:, None, :]
    r2 = (dr ** 2).sum(-1)
    np.fill_diagonal(r2, np.inf)
    acc = (w.m[None, :, None] * dr / r2[:, :, None] ** 1.5).sum(1)
    pot = -(w.m[None, :] / np.sqrt(r2)).sum(1)
    Nw = oracle.direct(w.x, w.y, w.z, w.m, w.r_out, p, "newton")
    for k in range(3):
        assert np.allclose(Nw[k], acc[:, k], rtol=1e-10, atol=1e-12 * np.abs(acc).max())
    assert np.allclose(Nw[3], pot, rtol=1e-12)


def test_momentum_conservation(small):
    """PAPER.md:286 'the force is symmetric'  =>  sum_i m_i a_L,i = 0."""
    w, p = small
    L = oracle.direct(w.x, w.y, w.z, w.m, w.r_out, p, "long")
    tot = np.array([np.sum(w.m * L[k]) for k in range(3)])
    ref = np.sum(w.m * _norm(L))
    assert np.all(np.abs(tot) < 1e-12 * ref)


def test_two_body_limits():
    """r >= r_out: pure Newton.  r <= r_in: no long-range force, constant potential -2Gm/(R + r_in)."""
    p = oracle.OracleParams.make(theta=0.3, multipole=1, rho=0.1)
    m = np.array([0.3, 0.7]); rout = np.array([0.2, 0.5])     # pair radius = max = 0.5
    for r, inside in ((0.6, False), (0.5, False), (0.04, True), (0.05, True)):
        x = np.array([0.0, r]); y = np.zeros(2); z = np.zeros(2)
        ax, ay, az, pot = oracle.direct(x, y, z, m, rout, p, "long")
        if inside:
            assert ax[0] == 0.0 and ax[1] == 0.0
            assert pot[0] == pytest.approx(-m[1] * 2.0 / (0.5 + 0.05), rel=1e-13)
            assert pot[1] == pytest.approx(-m[0] * 2.0 / (0.5 + 0.05), rel=1e-13)
        else:
            assert ax[0] == pytest.approx(m[1] / r ** 2, rel=1e-13)
            assert ax[1] == pytest.approx(-m[0] / r ** 2, rel=1e-13)
            assert pot[0] == pytest.approx(-m[1] / r, rel=1e-13)
    # coincident pair (reading P4): zero force, the same constant potential
    ax, ay, az, pot = oracle.direct(np.zeros(2), np.zeros(2), np.zeros(2), m, rout, p, "long")
    assert ax[0] == 0.0 and pot[0] == pytest.approx(-m[1] * 2.0 / 0.55, rel=1e-13)


def test_neighbour_symmetry_and_definition(small):
    w, p = small
    off, idx = oracle.neighbors_direct(w.x, w.y, w.z, w.r_out)
    assert off[-1] > w.N // 4                      # binaries guarantee plenty of neighbours
    pairs = set()
    for i in range(w.N):
        for j in idx[off[i]:off[i + 1]]:
            pairs.add((i, int(j)))
    assert all((j, i) in pairs for (i, j) in pairs)
    # brute force in numpy
    d = np.stack([w.x, w.y, w.z], 1)
    r = np.sqrt(((d[None] - d[:, None]) ** 2).sum(-1))
    R = np.maximum(w.r_out[None], w.r_out[:, None])
    ref = (r < R) & ~np.eye(w.N, dtype=bool)
    band = np.abs(r - R) < 1e-9 * R
    got = np.zeros_like(ref)
    for (i, j) in pairs:
        got[i, j] = True
    assert np.array_equal(got | band, ref | band)


def test_plummer_potential_energy():
    """Plummer closed form W = -(3 pi/32) G M^2 / a; Henon units fix a = 3 pi/16, so W = -1/2 (reading P13)."""
    p = oracle.OracleParams.make(theta=0.3, multipole=1)
    vals = []
    for seed in range(4):
        rng = np.random.Generator(np.random.PCG64(100 + seed))
        pos = plummer_positions(2048, rng)
        m = np.full(2048, 1.0 / 2048)
        Nw = oracle.direct(pos[:, 0], pos[:, 1], pos[:, 2], m, np.full(2048, 0.01), p, "newton")
        vals.append(0.5 * np.sum(m * Nw[3]))
    assert PLUMMER_A * np.mean(vals) == pytest.approx(-3.0 * np.pi / 32.0, rel=0.02)
    # generator: half-mass radius a / sqrt(2^{2/3} - 1) = 0.7686 (Henon units)
    rng = np.random.Generator(np.random.PCG64(5))
    r = np.linalg.norm(plummer_positions(200000, rng), axis=1)
    assert np.median(r) == pytest.approx(PLUMMER_A / np.sqrt(2 ** (2 / 3) - 1), rel=0.01)


def test_changeover_radii_eq12():
    """Eq. 12: r_out,i = max(1, m_i/<m>)^(1/3) r_out,ref with <m> the average mass of the system
    (reading P5).  Pins workloads.changeover_radii -- the one piece of the paper's arithmetic in the input generators --
    against numbers worked out by hand from the formula: config 4's central mass 0.01 among N - 1 stars of total
    mass 0.99 has m/<m> = 0.01 N = 10485.76, so 21.888 x 0.003 = 0.06566; a 150 Msun star at <m> = 0.586 Msun
    (Kroupa 0.08-150) gets 6.35 x; every star at or below the mean keeps r_out,ref."""
    from workloads.generators import changeover_radii
    N = 1 << 20
    m = np.full(N, 0.99 / (N - 1)); m[0] = 0.01
    r = changeover_radii(m, 0.003)
    assert r[0] == pytest.approx(0.003 * (0.01 * N) ** (1.0 / 3.0), rel=1e-14)
    assert r[0] == pytest.approx(0.0657, abs=5e-5) and r[0] / 0.003 == pytest.approx(21.9, abs=0.05)
    assert np.all(r[1:] == 0.003)                                   # below the mean: exactly r_out,ref
    m = np.full(10000, (5860.0 - 150.0 - 0.08 - 0.3) / 9997.0); m[0], m[1], m[2] = 150.0, 0.08, 0.3      # mean 0.586
    r = changeover_radii(m, 0.01)
    assert m.sum() / m.size == pytest.approx(0.586, rel=1e-12)
    assert r[0] / 0.01 == pytest.approx((150.0 / 0.586) ** (1.0 / 3.0), rel=1e-12) and r[0] / 0.01 == pytest.approx(6.35, abs=0.005)
    assert r[1] == 0.01 and r[2] == 0.01 and np.all(r[3:] == 0.01)
    # equal masses: a no-op; the radius grows as the cube root of the mass (8 x the mean mass -> twice the radius)
    assert np.all(changeover_radii(np.full(100, 0.01), 0.05) == 0.05)
    m = np.ones(1000); m[0] = 8.0 * (999.0 / 992.0)                # m_0 / <m> = 8 exactly: <m> = (999 + m_0)/1000
    assert changeover_radii(m, 1.0)[0] == pytest.approx(2.0, rel=1e-12)
