"""Pins of the oracle's changeover functions against what the paper fixes (no GPU)."""
import os

import numpy as np
import pytest

import oracle

LAMS = [9.0 / 11.0, 0.5, 1.0 / 3.0]
HERE = os.path.dirname(os.path.abspath(__file__))


def test_golden_fig3_case():
    """Values for r_in=1, r_out=10 (Eq. 15/17)."""
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "changeover_fig3.txt")) if l.strip() and l[0] != "#"]
    lam = 9.0 / 11.0
    for xs, ks, ws in rows:
        x = float(xs)
        # W(0) from the x<=0 branch and the 0<x<1 branch agree; use a point just inside for 0 and 1
        assert oracle.K(x, lam) == pytest.approx(float(ks), abs=2e-12)
        assert oracle.W(x, lam) == pytest.approx(float(ws), abs=2e-12)


@pytest.mark.parametrize("lam", LAMS)
def test_eq19_boundary_values(lam):
    """Eq. 19: W(1)=0, K(0)=1, K(1)=0, K', K'', K''' vanish at both ends (from inside)."""
    eps = 1e-9
    assert oracle.W(1.0 - eps, lam) == pytest.approx(0.0, abs=1e-8)
    assert oracle.K(eps, lam) == pytest.approx(1.0, abs=1e-12)
    assert oracle.K(1.0 - eps, lam) == pytest.approx(0.0, abs=1e-12)
    h = 1e-3
    for x0, sgn in ((0.0, +1.0), (1.0, -1.0)):
        # one-sided finite differences on 0..4 steps inside the interval
        pts = np.array([oracle.K(x0 + sgn * k * h, lam) for k in range(5)])
        d1 = (-25 * pts[0] + 48 * pts[1] - 36 * pts[2] + 16 * pts[3] - 3 * pts[4]) / (12 * h)
        d2 = (35 * pts[0] - 104 * pts[1] + 114 * pts[2] - 56 * pts[3] + 11 * pts[4]) / (12 * h * h)
        d3 = (-5 * pts[0] + 18 * pts[1] - 24 * pts[2] + 14 * pts[3] - 3 * pts[4]) / (2 * h ** 3)
        # K - K(end) = O(h^4), so the n-th difference quotient is O(h^{4-n})
        assert abs(d1) < 50 * h ** 3 * 300
        assert abs(d2) < 50 * h ** 2 * 300
        assert abs(d3) < 50 * h * 300
    # and they are NOT zero in the middle (the test above is not vacuous)
    assert abs((oracle.K(0.5 + h, lam) - oracle.K(0.5 - h, lam)) / (2 * h)) > 1.0


@pytest.mark.parametrize("lam", LAMS)
def test_eq18_second_formula(lam):
    """Eq. 18: W = f - f(1) r/r_out,  K = f - (x + r_in/(r_out-r_in)) f'(x)."""
    # Lambda = (r_out - r_in)/(r_out + r_in)  =>  r_in/r_out = (1-Lambda)/(1+Lambda)
    rho = (1.0 - lam) / (1.0 + lam)
    r_out, r_in = 1.0, rho
    q = r_in / (r_out - r_in)
    h = 1e-4
    for x in np.linspace(0.02, 0.98, 49):
        r = r_in + x * (r_out - r_in)
        f = oracle.f(x, lam)
        fp = (-oracle.f(x + 2 * h, lam) + 8 * oracle.f(x + h, lam) - 8 * oracle.f(x - h, lam) + oracle.f(x - 2 * h, lam)) / (12 * h)
        assert oracle.W(x, lam) == pytest.approx(f - oracle.f(1.0, lam) * r / r_out, abs=1e-13)
        assert oracle.K(x, lam) == pytest.approx(f - (x + q) * fp, abs=1e-9)


@pytest.mark.parametrize("lam", LAMS)
def test_force_is_gradient_of_potential(lam):
    """Pair potential -G m W/r  =>  force weight K = W - r dW/dr  (ties Eq. 17 to Eq. 15; also across x<=0)."""
    rho = (1.0 - lam) / (1.0 + lam)
    r_out, r_in = 1.0, rho
    h = 1e-5

    def Wr(r):
        return oracle.W((r - r_in) / (r_out - r_in), lam)

    for r in np.concatenate([np.linspace(0.05 * r_in, 0.95 * r_in, 5), np.linspace(r_in * 1.02, 0.99, 40), [1.1, 2.0]]):
        dW = (-Wr(r + 2 * h) + 8 * Wr(r + h) - 8 * Wr(r - h) + Wr(r - 2 * h)) / (12 * h)
        x = (r - r_in) / (r_out - r_in)
        assert oracle.K(x, lam) == pytest.approx(Wr(r) - r * dW, abs=2e-9)


def test_monotone_and_range():
    lam = 9.0 / 11.0
    xs = np.linspace(-0.5, 1.5, 401)
    k = np.array([oracle.K(x, lam) for x in xs])
    assert np.all(np.diff(k) <= 1e-15) and k.max() == 1.0 and k.min() == 0.0
    # long-range force weight 1-K rises from 0 at r_in to 1 at r_out (north_star)
    assert 1.0 - oracle.K(0.0, lam) == 0.0 and 1.0 - oracle.K(1.0, lam) == 1.0
