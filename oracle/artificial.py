"""Oracle part (E) -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/petar_oracle.c's header).

P3T-kick and the artificial particles around the long-range force (PAPER.md section
6.4, :352-482 and Table 1 :482-570), in plain numpy, fp64, one binary at a time, in the paper's order:

  * kick                      v += a_L dt_L                                   (Fig. 2 :294)
  * Kepler elements of a pair (a, e and the orbital frame in which Eq. 32 holds)
  * pseudoparticles           Eq. 38 (:473-478): three particles of mass (m1+m2)/3 that carry the orbit-averaged
                              quadrupole of the binary, Eq. 36-37 (:457-470)
  * orbit-sampling particles  Eq. 29 (:420-428): 2 n_split particles along the two orbits
  * tidal-tensor measure points: 4 at the corners of a regular tetrahedron (2nd order) or 8 at the corners of
                              the paper's "cube" (3rd order), coordinates of Table 1 part (3)
  * tidal-tensor fit          the generalized inverse of Eq. 28 (:404-406): least squares of the polynomial of
                              Table 1 part (2) through A'(r_k) = A(r_k) - A(r_cm)
  * tidal-tensor evaluation   Table 1 part (2)

Readings (P24-P26): the polynomial keeps the paper's convention A_i(r) = A_i(cm) + A_ij r'_j +
A_ijk r'_j r'_k (no 1/2); d_c = tt_scale * a; the frame of Eq. 32 has x along the pericentre direction
(eccentricity vector), z along the angular momentum; e = 0 takes x along the current separation.
"""
from __future__ import annotations

import numpy as np

SQ2H = np.sqrt(2.0) / 2.0
# Table 1 part (3): r'_k / d_c.  Tetrahedron: read off the printed A_xx, A_yy, A_zz rows;
# "cube": the printed list.
TT_POINTS = {
    2: np.array([[1.0, 0.0, -SQ2H], [-1.0, 0.0, -SQ2H], [0.0, 1.0, SQ2H], [0.0, -1.0, SQ2H]]),
    3: np.array([[1.0, 0.0, -1.0], [0.0, 1.0, -1.0], [-1.0, 0.0, -1.0], [0.0, -1.0, -1.0],
                 [1.0, 0.0, 1.0], [0.0, 1.0, 1.0], [-1.0, 0.0, 1.0], [0.0, -1.0, 1.0]]),
}
# order of the coefficients, Eq. 26
T2_NAMES = ["xx", "xy", "xz", "yy", "yz", "zz"]
T3_NAMES = T2_NAMES + ["xxx", "xxy", "xxz", "xyy", "xyz", "xzz", "yyy", "yyz", "yzz", "zzz"]


def kick(v, a, dt):
    """P3T-kick: v + a dt (the caller applies it with dt_L/2 at both ends of a step)."""
    return np.asarray(v, dtype=np.float64) + np.asarray(a, dtype=np.float64) * dt


def kepler_elements(d, w, mu):
    """Relative position d = x_2 - x_1, relative velocity w, mu = G (m1 + m2)  ->  dict(a, e, P, Q, W, bound).
    P: unit vector to the pericentre of the relative orbit, W: along d x w, Q = W x P: the frame of Eq. 32."""
    d = np.asarray(d, dtype=np.float64); w = np.asarray(w, dtype=np.float64)
    r = np.linalg.norm(d)
    h = np.cross(d, w)
    hn = np.linalg.norm(h)
    inv_a = 2.0 / r - w.dot(w) / mu
    evec = np.cross(w, h) / mu - d / r
    e = np.linalg.norm(evec)
    bound = bool(inv_a > 0.0 and hn > 0.0)
    if not bound:
        return dict(a=np.inf if inv_a == 0 else 1.0 / inv_a, e=e, P=np.array([1.0, 0, 0]), Q=np.array([0, 1.0, 0]),
                    W=np.array([0, 0, 1.0]), bound=False)
    W = h / hn
    P = evec / e if e > 1e-12 else d / r          # circular orbit: any direction in the plane serves (Eq. 36 is isotropic there)
    P = P - W * P.dot(W); P /= np.linalg.norm(P)
    Q = np.cross(W, P)
    return dict(a=1.0 / inv_a, e=e, P=P, Q=Q, W=W, bound=True)


def orbit_average_quadrupole(m1, m2, a, e, n=20000):
    """<A> of Eq. 34 by quadrature over the eccentric anomaly (Eq. 30, 32, 33, 35), orbital frame."""
    E = (np.arange(n) + 0.5) * 2 * np.pi / n
    dr = np.stack([a * (np.cos(E) - e), a * np.sqrt(1 - e * e) * np.sin(E), np.zeros(n)], axis=1)      # Eq. 32
    mt = m1 + m2
    r1 = -(m2 / mt) * dr; r2 = (m1 / mt) * dr                                                          # Eq. 33
    wgt = (1 - e * np.cos(E)) / n                                                                       # dt/P, Eq. 35
    A = m1 * np.einsum("n,ni,nj->ij", wgt, r1, r1) + m2 * np.einsum("n,ni,nj->ij", wgt, r2, r2)         # Eq. 30, 34
    return A


def pseudoparticles(m1, m2, a, e, P, Q, cm):
    """Eq. 38: three positions (3x3) and their common mass (m1+m2)/3."""
    mt = m1 + m2
    mu_red = m1 * m2 / mt
    s = a * np.sqrt(mu_red / mt)
    bx = np.sqrt(3 * e * e + 0.75); by = np.sqrt(1 - e * e)
    loc = s * np.array([[0.0, by], [bx, -0.5 * by], [-bx, -0.5 * by]])
    pos = np.asarray(cm)[None, :] + loc[:, 0:1] * P[None, :] + loc[:, 1:2] * Q[None, :]
    return pos, mt / 3.0


def orbit_sampling(m1, m2, a, e, P, Q, cm, n_split):
    """Orbit-sampling particles (Eq. 29): n_split points per component at equal eccentric-anomaly
    intervals dE = 2 pi / n_split, E_k = k dE (reading P27: the first sample at the pericentre), masses
    m_i dM_k / (2 pi) with dM_k = dE - 2 e cos(E_k) sin(dE / 2).  Returns (pos (2 n_split x 3), mass (2 n_split)):
    the samples of component 1, then those of component 2."""
    dE = 2.0 * np.pi / n_split
    E = np.arange(n_split) * dE
    dM = dE - 2.0 * e * np.cos(E) * np.sin(0.5 * dE)
    rel = (a * (np.cos(E) - e))[:, None] * P[None, :] + (a * np.sqrt(1.0 - e * e) * np.sin(E))[:, None] * Q[None, :]     # Eq. 32
    mt = m1 + m2
    pos = np.concatenate([np.asarray(cm)[None, :] - (m2 / mt) * rel, np.asarray(cm)[None, :] + (m1 / mt) * rel])      # Eq. 33
    mass = np.concatenate([m1 * dM, m2 * dM]) / (2.0 * np.pi)
    return pos, mass


def tidal_points(order, cm, d_c):
    return np.asarray(cm)[None, :] + d_c * TT_POINTS[order]


def _design_rows(order, rp):
    """Rows of M (Eq. 28) for one point r' = rp: the three components of Table 1 part (2) minus A(cm)."""
    x, y, z = rp
    n = 6 if order == 2 else 16
    M = np.zeros((3, n))
    # A_x = A_xx x + A_xy y + A_xz z ; A_y = A_xy x + A_yy y + A_yz z ; A_z = A_xz x + A_yz y + A_zz z
    M[0, 0], M[0, 1], M[0, 2] = x, y, z
    M[1, 1], M[1, 3], M[1, 4] = x, y, z
    M[2, 2], M[2, 4], M[2, 5] = x, y, z
    if order == 3:
        # A_x += A_xxx x^2 + 2 A_xxy xy + 2 A_xxz xz + A_xyy y^2 + 2 A_xyz yz + A_xzz z^2, etc.
        q = dict(xx=x * x, xy=2 * x * y, xz=2 * x * z, yy=y * y, yz=2 * y * z, zz=z * z)
        idx = {nme: 6 + k for k, nme in enumerate(T3_NAMES[6:])}
        for i, comp in enumerate("xyz"):
            for jk, val in q.items():
                name = "".join(sorted(comp + jk))
                M[i, idx[name]] += val
    return M


def tidal_design_matrix(order, d_c=1.0):
    """M of Eq. 28: (3 n_points) x (6 | 16), rows ordered A'_x(r_1), A'_y(r_1), A'_z(r_1), A'_x(r_2), ... (Eq. 27)."""
    return np.concatenate([_design_rows(order, d_c * p) for p in TT_POINTS[order]], axis=0)


def tidal_fit(order, d_c, acc_points, acc_cm):
    """Least-squares solution of Eq. 28 for the coefficients T (Eq. 26 order)."""
    Ap = (np.asarray(acc_points) - np.asarray(acc_cm)[None, :]).reshape(-1)          # Eq. 27
    T, *_ = np.linalg.lstsq(tidal_design_matrix(order, d_c), Ap, rcond=None)
    return T


def tidal_eval(order, T, acc_cm, rp):
    """Table 1 part (2): acceleration at r' = r - r_cm from the fitted coefficients."""
    return np.asarray(acc_cm) + _design_rows(order, np.asarray(rp)) @ np.asarray(T)


def artificial_particles(x1, v1, m1, x2, v2, m2, G, order, tt_scale):
    """Everything for one binary: dict(pos (n_art x 3), mass (n_art), d_c, a, e, cm, bound).
    Layout: n_tt measure points (mass 0), the centre-of-mass point (mass 0), three pseudoparticles."""
    x1, v1, x2, v2 = (np.asarray(q, dtype=np.float64) for q in (x1, v1, x2, v2))
    mt = m1 + m2
    cm = (m1 * x1 + m2 * x2) / mt
    el = kepler_elements(x2 - x1, v2 - v1, G * mt)
    ntt = TT_POINTS[order].shape[0]
    pos = np.tile(cm, (ntt + 4, 1)); mass = np.zeros(ntt + 4)
    mass[ntt + 1:] = mt / 3.0
    d_c = 0.0
    if el["bound"]:
        d_c = tt_scale * el["a"]
        pos[:ntt] = tidal_points(order, cm, d_c)
        pos[ntt + 1:], _ = pseudoparticles(m1, m2, el["a"], el["e"], el["P"], el["Q"], cm)
    return dict(pos=pos, mass=mass, d_c=d_c, a=el["a"], e=el["e"], cm=cm, bound=el["bound"])
