"""Pins of the oracle's part (D): short-range acceleration, jerk and potential over the neighbour rows
(H_S of Eq. 11, with the changeover functions of Eq. 15-19)."""
import numpy as np
import pytest

import oracle
from workloads import make_workload

def _K(x):
    return np.array([oracle.K(v, LAM) for v in np.atleast_1d(x)])


def _f(x):
    return np.array([oracle.f(v, LAM) for v in np.atleast_1d(x)])


RHO = 0.1
LAM = (1 - RHO) / (1 + RHO)
Q = RHO / (1 - RHO)


def test_dK_closed_form_against_difference_quotient_of_eq17():
    x = np.linspace(0.001, 0.999, 400)
    h = 1e-6
    fd = (_K(x + h) - _K(x - h)) / (2 * h)
    assert np.max(np.abs(oracle.dK(x, LAM, Q) - fd)) < 1e-8
    # Eq. 19: K' vanishes at both ends, and outside
    assert np.all(oracle.dK(np.array([-0.5, 0.0, 1.0, 1.5]), LAM, Q) == 0.0)
    # and Eq. 18 itself: K = f - (x + q) f'  with f' by a difference quotient of Eq. 16
    fp = (_f(x + h) - _f(x - h)) / (2 * h)
    assert np.max(np.abs(_K(x) - (_f(x) - (x + Q) * fp))) < 1e-8


@pytest.fixture(scope="module")
def small():
    w = make_workload(2, N=1500, velocities=True)
    # radii large enough that singles have neighbours too (the sphere is sparse at this N)
    rout = 25.0 * w.r_out
    off, idx = oracle.neighbors_direct(w.x, w.y, w.z, rout)
    return w, rout, off, idx


def test_rows_equal_the_short_range_definition(small):
    w, rout, off, idx = small
    s = oracle.short_range(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rout, off, idx, w.G, RHO)
    p = oracle.OracleParams.from_workload(w)
    d = oracle.direct(w.x, w.y, w.z, w.m, rout, p, "short")
    den = np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)
    sel = den > 0
    assert sel.sum() > 1000
    err = np.sqrt((s[0] - d[0]) ** 2 + (s[1] - d[1]) ** 2 + (s[2] - d[2]) ** 2)[sel] / den[sel]
    assert err.max() < 1e-12
    assert np.max(np.abs(s[6] - d[3])[sel] / np.abs(d[3][sel])) < 1e-12
    # momentum: sum m a_S = 0 and sum m j_S = 0 (the list and the weights are symmetric)
    for k in (0, 1, 2, 3, 4, 5):
        assert abs(np.sum(w.m * s[k])) < 1e-12 * np.sum(w.m * np.abs(s[k]))


def test_jerk_is_time_derivative_of_acceleration(small):
    w, rout, off, idx = small
    s = oracle.short_range(w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m, rout, off, idx, w.G, RHO)
    # the same neighbour rows a moment earlier / later (the pairs stay inside their radii for such a small dt
    # unless they sit at the very edge, where K and all its derivatives vanish anyway)
    vmax = np.max(np.sqrt(w.vx ** 2 + w.vy ** 2 + w.vz ** 2))
    dt = 1e-7 / vmax          # displacement 1e-7: resolved to 2e-9 by coordinates of order one, truncation ~1e-8
    ap = oracle.short_range(w.x + dt * w.vx, w.y + dt * w.vy, w.z + dt * w.vz, w.vx, w.vy, w.vz, w.m, rout, off, idx, w.G, RHO)
    am = oracle.short_range(w.x - dt * w.vx, w.y - dt * w.vy, w.z - dt * w.vz, w.vx, w.vy, w.vz, w.m, rout, off, idx, w.G, RHO)
    fd = [(ap[k] - am[k]) / (2 * dt) for k in range(3)]
    jn = np.sqrt(s[3] ** 2 + s[4] ** 2 + s[5] ** 2)
    err = np.sqrt(sum((fd[k] - s[3 + k]) ** 2 for k in range(3)))
    # singles: separations ~1e-2, dt*v ~ 1e-9 -> difference quotient good to ~1e-6; tight binaries (a ~ 1e-5) are
    # checked on their own below
    wide = np.array([off[i + 1] > off[i] and np.all(np.hypot(np.hypot(w.x[i] - w.x[idx[off[i]:off[i + 1]]], w.y[i] - w.y[idx[off[i]:off[i + 1]]]),
                                                          w.z[i] - w.z[idx[off[i]:off[i + 1]]]) > 1e-3) for i in range(w.N)])
    assert wide.sum() > 100
    rel = err[wide] / jn[wide]
    # difference-quotient noise only; a dropped or mis-signed term of the jerk gives O(1) on changeover pairs
    assert np.max(rel) < 1e-5 and np.median(rel) < 1e-7


def test_two_body_newtonian_jerk_inside_r_in():
    """r < r_in: K = 1, K' = 0 -> the textbook jerk  -G m [ w/r^3 - 3 (d.w) d / r^5 ]."""
    x = np.array([0.0, 3e-4]); y = np.array([0.0, 1e-4]); z = np.array([0.0, -2e-4])
    vx = np.array([0.1, -0.3]); vy = np.array([0.0, 0.2]); vz = np.array([0.05, 0.0])
    m = np.array([2.0, 3.0]); rout = np.array([0.01, 0.008])
    off = np.array([0, 1, 2]); idx = np.array([1, 0], dtype=np.int32)
    s = oracle.short_range(x, y, z, vx, vy, vz, m, rout, off, idx, 1.0, RHO)
    d = np.array([x[0] - x[1], y[0] - y[1], z[0] - z[1]]); wv = np.array([vx[0] - vx[1], vy[0] - vy[1], vz[0] - vz[1]])
    r = np.linalg.norm(d)
    assert r < RHO * 0.01
    a0 = -m[1] * d / r ** 3
    j0 = -m[1] * (wv / r ** 3 - 3 * d.dot(wv) * d / r ** 5)
    assert np.allclose([s[0][0], s[1][0], s[2][0]], a0, rtol=1e-13)
    assert np.allclose([s[3][0], s[4][0], s[5][0]], j0, rtol=1e-13)
    # potential inside r_in: W = Lambda (1 - 2x) with x < 0 (reading P4): phi = -m [1/r - (1+Lambda)/R + ...] -> check value
    R = 0.01; rin = RHO * R; xx = (r - rin) / (R - rin)
    assert s[6][0] == pytest.approx(-m[1] * LAM * (1 - 2 * xx) / r, rel=1e-13)
    # beyond r_out nothing; coincident pair skipped
    s2 = oracle.short_range(x * 100, y * 100, z * 100, vx, vy, vz, m, rout, off, idx, 1.0, RHO)
    assert all(np.all(v == 0) for v in s2)
    s3 = oracle.short_range(x * 0, y * 0, z * 0, vx, vy, vz, m, rout, off, idx, 1.0, RHO)
    assert all(np.all(v == 0) for v in s3)
