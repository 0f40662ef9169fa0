"""Synthetic initial conditions for the long-range P3T force path.

Recipe (also stated in DESIGN.md, "Input recipe"):

* Plummer sphere in Henon units (G = M = 1, virial radius 1  =>  a = 3*pi/16;
  PAPER.md:625 "The Plummer model ... virial radius is 1.0 in the Henon unit").
  Radius by inverting the enclosed-mass profile  M(<r) = r^3 / (r^2 + a^2)^{3/2};
  samples with r > 20 are redrawn (keeps the tree's root cube small).
* Kroupa (2001) IMF, two power-law segments (index 1.3 on [0.08, 0.5) Msun,
  2.3 on [0.5, m_max] Msun), sampled by inverse CDF, rescaled to total mass 1.
* Binaries: stars are shuffled and paired; semi-major axis log-uniform on the
  configured range, thermal eccentricity e = sqrt(u), uniform mean
  anomaly (Kepler's equation solved by Newton iteration), random orientation;
  the two components sit at the centre of mass -/+ the mass-weighted offsets
  (Eq. 33), the centres of mass being Plummer-sampled.
* Changeover radii: r_out,i = max(1, m_i/<m>)^{1/3} r_out,ref (Eq. 12).

Everything is drawn from numpy's PCG64 with seed 20061656 + k for config k.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

PLUMMER_A = 3.0 * np.pi / 16.0
R_CUT = 20.0
SEED_BASE = 20061656


@dataclass
class Workload:
    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    m: np.ndarray
    r_out: np.ndarray
    theta: float
    multipole: int            # 1 = monopole, 2 = quadrupole
    r_out_ref: float
    r_in_over_r_out: float = 0.1
    n_leaf_limit: int = 8
    n_group_limit: int = 64
    G: float = 1.0
    meta: dict = field(default_factory=dict)
    vx: np.ndarray | None = None      # velocities (make_workload(velocities=True)); None on the force path
    vy: np.ndarray | None = None
    vz: np.ndarray | None = None
    dt_L: float | None = None         # tree time step that goes with r_out_ref (Eq. 41)

    @property
    def N(self) -> int:
        return int(self.x.shape[0])


def plummer_positions(n: int, rng: np.random.Generator, a: float = PLUMMER_A,
                      r_cut: float = R_CUT) -> np.ndarray:
    """n x 3 positions of a Plummer sphere with scale radius a, truncated at r_cut."""
    r = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u = rng.random(todo.size)
        u = np.clip(u, 1e-300, 1.0)
        rr = a / np.sqrt(np.maximum(u ** (-2.0 / 3.0) - 1.0, 1e-300))
        ok = rr <= r_cut
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    cos_t = rng.uniform(-1.0, 1.0, n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    pos = np.empty((n, 3))
    pos[:, 0] = r * sin_t * np.cos(phi)
    pos[:, 1] = r * sin_t * np.sin(phi)
    pos[:, 2] = r * cos_t
    return pos


def kroupa_masses(n: int, rng: np.random.Generator, m_lo: float = 0.08,
                  m_break: float = 0.5, m_hi: float = 150.0) -> np.ndarray:
    """Kroupa (2001) two-segment IMF in Msun by inverse-CDF sampling (not yet rescaled)."""
    a1, a2 = 1.3, 2.3
    # dN/dm = k1 m^-a1 on [m_lo, m_break), k2 m^-a2 on [m_break, m_hi], continuous at m_break
    k1 = 1.0
    k2 = k1 * m_break ** (a2 - a1)
    n1 = k1 * (m_break ** (1 - a1) - m_lo ** (1 - a1)) / (1 - a1)
    n2 = k2 * (m_hi ** (1 - a2) - m_break ** (1 - a2)) / (1 - a2)
    u = rng.random(n)
    seg1 = u < n1 / (n1 + n2)
    m = np.empty(n)
    v = rng.random(n)
    m[seg1] = (m_lo ** (1 - a1) + v[seg1] * (m_break ** (1 - a1) - m_lo ** (1 - a1))) ** (1.0 / (1 - a1))
    m[~seg1] = (m_break ** (1 - a2) + v[~seg1] * (m_hi ** (1 - a2) - m_break ** (1 - a2))) ** (1.0 / (1 - a2))
    return m


def changeover_radii(m: np.ndarray, r_out_ref: float) -> np.ndarray:
    """Eq. 12: r_out,i = max(1, m_i/<m>)^{1/3} r_out,ref, <m> = M_total/N."""
    mean = m.sum() / m.shape[0]
    return np.maximum(1.0, m / mean) ** (1.0 / 3.0) * r_out_ref


def _solve_kepler(mean_anom: np.ndarray, ecc: np.ndarray) -> np.ndarray:
    E = mean_anom + ecc * np.sin(mean_anom)
    for _ in range(60):
        dE = (E - ecc * np.sin(E) - mean_anom) / (1.0 - ecc * np.cos(E))
        E = E - dE
        if np.max(np.abs(dE)) < 1e-15:
            break
    return E


def _random_rotations(n: int, rng: np.random.Generator) -> np.ndarray:
    """n uniformly random rotation matrices (from unit quaternions)."""
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def plummer_speeds(r: np.ndarray, rng: np.random.Generator, a: float = PLUMMER_A) -> np.ndarray:
    """Speeds of a Plummer model (G = M = 1) at radii r: v = q v_esc(r), q drawn by rejection from
    g(q) = q^2 (1 - q^2)^(7/2) (Aarseth, Henon & Wielen 1974)."""
    n = r.shape[0]
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        xq = rng.random(todo.size)
        yq = 0.1 * rng.random(todo.size)
        ok = yq < xq * xq * (1.0 - xq * xq) ** 3.5
        q[todo[ok]] = xq[ok]
        todo = todo[~ok]
    vesc = np.sqrt(2.0 / a) * (1.0 + (r / a) ** 2) ** -0.25
    return q * vesc


def _isotropic(speed: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    n = speed.shape[0]
    cos_t = rng.uniform(-1.0, 1.0, n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    return np.stack([speed * sin_t * np.cos(phi), speed * sin_t * np.sin(phi), speed * cos_t], axis=1)


def _place_with_binaries(m: np.ndarray, n_pairs: int, a_lo: float, a_hi: float,
                         rng: np.random.Generator, vel_rng: np.random.Generator | None = None):
    """Positions for stars of mass m where stars (2k, 2k+1), k < n_pairs, form binaries.
    With vel_rng: returns (pos, vel); the velocities use their own generator and the orbital elements
    already drawn, so the positions are the same with and without them."""
    n = m.shape[0]
    n_single = n - 2 * n_pairs
    cm = plummer_positions(n_pairs + n_single, rng)
    pos = np.empty((n, 3))
    if n_pairs:
        semi = np.exp(rng.uniform(np.log(a_lo), np.log(a_hi), n_pairs))
        ecc = np.sqrt(rng.random(n_pairs))
        E = _solve_kepler(rng.uniform(0.0, 2.0 * np.pi, n_pairs), ecc)
        rel = np.zeros((n_pairs, 3))
        rel[:, 0] = semi * (np.cos(E) - ecc)                       # Eq. 32
        rel[:, 1] = semi * np.sqrt(1.0 - ecc * ecc) * np.sin(E)
        rot = _random_rotations(n_pairs, rng)
        rel = np.einsum("nij,nj->ni", rot, rel)
        m1 = m[0:2 * n_pairs:2]
        m2 = m[1:2 * n_pairs:2]
        mt = m1 + m2
        pos[0:2 * n_pairs:2] = cm[:n_pairs] - (m2 / mt)[:, None] * rel   # Eq. 33
        pos[1:2 * n_pairs:2] = cm[:n_pairs] + (m1 / mt)[:, None] * rel
    pos[2 * n_pairs:] = cm[n_pairs:]
    if vel_rng is None:
        return pos
    vcm = _isotropic(plummer_speeds(np.linalg.norm(cm, axis=1), vel_rng), vel_rng)
    vel = np.empty((n, 3))
    if n_pairs:
        # Kepler relative velocity in the orbital plane (G = 1), rotated like the relative position
        nmean = np.sqrt(mt / semi ** 3)
        fac = semi * nmean / (1.0 - ecc * np.cos(E))
        relv = np.zeros((n_pairs, 3))
        relv[:, 0] = -fac * np.sin(E)
        relv[:, 1] = fac * np.sqrt(1.0 - ecc * ecc) * np.cos(E)
        relv = np.einsum("nij,nj->ni", rot, relv)
        vel[0:2 * n_pairs:2] = vcm[:n_pairs] - (m2 / mt)[:, None] * relv
        vel[1:2 * n_pairs:2] = vcm[:n_pairs] + (m1 / mt)[:, None] * relv
    vel[2 * n_pairs:] = vcm[n_pairs:]
    return pos, vel


# BASELINE.json configs 1..5 (index k-1); theta of config 4 is swept by the caller.
CONFIGS = {
    1: dict(N=4096, masses="equal", bin_frac=0.0, a_range=None, r_out_ref=0.05, theta=0.3, multipole=1),
    2: dict(N=65536, masses="kroupa", bin_frac=0.5, a_range=(1e-5, 1e-3), r_out_ref=0.01, theta=0.3, multipole=2),
    3: dict(N=1048576, masses="kroupa", bin_frac=1.0, a_range=(1e-5, 1e-3), r_out_ref=0.003, theta=0.3, multipole=2),
    4: dict(N=1048576, masses="central", bin_frac=0.0, a_range=None, r_out_ref=0.003, theta=0.3, multipole=2),
    5: dict(N=10485760, masses="equal", bin_frac=0.1, a_range=(1e-6, 1e-4), r_out_ref=0.0015, theta=0.3, multipole=2),
}


def tree_time_step(r_out_ref: float) -> float:
    """dt_L that goes with r_out_ref: Eq. 41 r_out = 10 dt_L sigma_1D with sigma_1D = 0.409
    (Henon units), rounded to a power of two as in Table 3 (0.004 <-> 1/1024 for N1m, :666)."""
    return float(2.0 ** np.round(np.log2(r_out_ref / 4.09)))


def make_workload(config: int, N: int | None = None, seed: int | None = None, theta: float | None = None,
                  uniform_radii: bool = False, velocities: bool = False) -> Workload:
    """Build BASELINE.json config `config` (1..5); N overrides the size (same recipe, for tests).
    velocities=True adds Plummer velocities (+ binary orbital motion) from a separate generator."""
    c = dict(CONFIGS[config])
    n = int(N if N is not None else c["N"])
    base_seed = SEED_BASE + config if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(base_seed))
    vel_rng = np.random.Generator(np.random.PCG64([base_seed, 24])) if velocities else None
    vel = None
    kind = c["masses"]
    if kind == "equal":
        m = np.full(n, 1.0 / n)
    elif kind == "kroupa":
        m = kroupa_masses(n, rng)
        m /= m.sum()
    elif kind == "central":
        m = np.full(n, 0.99 / max(n - 1, 1))
        m[0] = 0.01
    else:
        raise ValueError(kind)
    n_pairs = int(round(c["bin_frac"] * n)) // 2
    if kind == "central":
        pos = np.empty((n, 3))
        pos[0] = 0.0
        pos[1:] = plummer_positions(n - 1, rng)
        if velocities:
            vel = np.zeros((n, 3))
            vel[1:] = _isotropic(plummer_speeds(np.linalg.norm(pos[1:], axis=1), vel_rng), vel_rng)
    else:
        if n_pairs:
            perm = rng.permutation(n)       # "shuffle stars, pair consecutive ones"
            m = m[perm]
        a_lo, a_hi = c["a_range"] if c["a_range"] else (1.0, 1.0)
        if velocities:
            pos, vel = _place_with_binaries(m, n_pairs, a_lo, a_hi, rng, vel_rng)
        else:
            pos = _place_with_binaries(m, n_pairs, a_lo, a_hi, rng)
        # final shuffle so that the input order carries no structure
        perm2 = rng.permutation(n)
        pos = pos[perm2]
        m = m[perm2]
        if vel is not None:
            vel = vel[perm2]
        inv2 = np.empty(n, dtype=np.int64); inv2[perm2] = np.arange(n)
        pair_idx = np.stack([inv2[0:2 * n_pairs:2], inv2[1:2 * n_pairs:2]], axis=1).astype(np.int32)
    if kind == "central":
        pair_idx = np.zeros((0, 2), dtype=np.int32)
    r_out_ref = c["r_out_ref"]
    r_out = np.full(n, r_out_ref) if uniform_radii else changeover_radii(m, r_out_ref)
    return Workload(
        name=f"config{config}_N{n}",
        x=np.ascontiguousarray(pos[:, 0]), y=np.ascontiguousarray(pos[:, 1]), z=np.ascontiguousarray(pos[:, 2]),
        m=np.ascontiguousarray(m), r_out=np.ascontiguousarray(r_out),
        theta=float(c["theta"] if theta is None else theta), multipole=c["multipole"], r_out_ref=r_out_ref,
        meta=dict(config=config, n_pairs=n_pairs, masses=kind, pairs=pair_idx),     # pairs: member indices of the binaries
        vx=None if vel is None else np.ascontiguousarray(vel[:, 0]),
        vy=None if vel is None else np.ascontiguousarray(vel[:, 1]),
        vz=None if vel is None else np.ascontiguousarray(vel[:, 2]),
        dt_L=tree_time_step(r_out_ref),
    )
