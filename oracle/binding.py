"""ctypes binding of oracle/petar_oracle.c (test infrastructure; see the C file's header)."""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "petar_oracle.c")
_LIB = None


def build_library(force: bool = False) -> str:
    """Compile petar_oracle.c with gcc (no contraction, explicit fma only) and return the .so path."""
    with open(_SRC, "rb") as fh:
        tag = hashlib.sha1(fh.read()).hexdigest()[:12]
    out_dir = os.path.join(_HERE, "build")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"libpetar_oracle_{tag}.so")
    if force or not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-mfma",
               "-fno-fast-math", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


def _lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build_library())
        L.ora_f.restype = C.c_double; L.ora_f.argtypes = [C.c_double, C.c_double]
        L.ora_W.restype = C.c_double; L.ora_W.argtypes = [C.c_double, C.c_double]
        L.ora_K.restype = C.c_double; L.ora_K.argtypes = [C.c_double, C.c_double]
        L.ora_tree_build.restype = C.c_void_p
        L.ora_tree_n_nodes.restype = C.c_int64; L.ora_tree_n_nodes.argtypes = [C.c_void_p]
        L.ora_tree_n_groups.restype = C.c_int64; L.ora_tree_n_groups.argtypes = [C.c_void_p]
        L.ora_num_threads.restype = C.c_int
        _LIB = L
    return _LIB


class OracleParams(C.Structure):
    _fields_ = [("G", C.c_double), ("theta", C.c_double), ("rho", C.c_double),
                ("multipole", C.c_int32), ("n_leaf", C.c_int32), ("n_group", C.c_int32), ("pad", C.c_int32)]

    @classmethod
    def make(cls, theta, multipole, G=1.0, rho=0.1, n_leaf=8, n_group=64):
        return cls(float(G), float(theta), float(rho), int(multipole), int(n_leaf), int(n_group), 0)

    @classmethod
    def from_workload(cls, w, theta=None, multipole=None):
        return cls.make(w.theta if theta is None else theta, w.multipole if multipole is None else multipole,
                        G=w.G, rho=w.r_in_over_r_out, n_leaf=w.n_leaf_limit, n_group=w.n_group_limit)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def K(x, lam):
    return _lib().ora_K(float(x), float(lam))


def W(x, lam):
    return _lib().ora_W(float(x), float(lam))


def f(x, lam):
    return _lib().ora_f(float(x), float(lam))


def set_num_threads(n: int) -> None:
    """Number of OpenMP threads of the following calls (bench.py's single-thread baseline)."""
    _lib().ora_set_num_threads(C.c_int(int(n)))


def num_threads() -> int:
    return int(_lib().ora_num_threads())


def direct(x, y, z, m, rout, params: OracleParams, which: str, targets=None):
    """O(N^2) definition sums.  which in {'newton','long','short'}.  Returns (ax, ay, az, pot)."""
    x, y, z, m, rout = map(_f64, (x, y, z, m, rout))
    n = x.shape[0]
    code = {"newton": 0, "long": 1, "short": 2}[which]
    if targets is None:
        nt, tp = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = targets.shape[0], _p(targets, C.c_int64)
    out = [np.zeros(nt) for _ in range(4)]
    _lib().ora_direct(C.c_int64(n), _p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(m, C.c_double),
                      _p(rout, C.c_double), C.byref(params), C.c_int(code), C.c_int64(nt), tp,
                      *[_p(o, C.c_double) for o in out])
    return tuple(out)


def neighbors_direct(x, y, z, rs):
    """O(N^2) neighbour definition.  Returns (offsets int64[N+1], indices int32[total]) rows ascending."""
    x, y, z, rs = map(_f64, (x, y, z, rs))
    n = x.shape[0]
    off = np.zeros(n + 1, dtype=np.int64)
    args = [C.c_int64(n), _p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(rs, C.c_double), _p(off, C.c_int64)]
    _lib().ora_neighbors_direct(*args, None)
    idx = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
    _lib().ora_neighbors_direct(*args, _p(idx, C.c_int32))
    return off, idx[: int(off[-1])]


def search_radii(vx, vy, vz, rout, Cr: float, dt: float):
    """Eq. 24: r_nb = r_out + C_r |v| dt_L."""
    vx, vy, vz, rout = map(_f64, (vx, vy, vz, rout))
    out = np.zeros_like(rout)
    _lib().ora_search_radii(C.c_int64(rout.shape[0]), _p(vx, C.c_double), _p(vy, C.c_double), _p(vz, C.c_double),
                            _p(rout, C.c_double), C.c_double(Cr), C.c_double(dt), _p(out, C.c_double))
    return out


def pericentre(d, w, mu: float) -> float:
    """Kepler pericentre separation of a pair: relative position d[3], relative velocity w[3], mu = G (m_i + m_j)."""
    L = _lib()
    L.ora_pericentre.restype = C.c_double
    L.ora_pericentre.argtypes = [C.c_double] * 7
    return float(L.ora_pericentre(*[float(v) for v in d], *[float(v) for v in w], float(mu)))


def neighbors_orbit_direct(x, y, z, vx, vy, vz, m, rnb, rout, G: float, Cv: float):
    """O(N^2) definition of the two-stage neighbour criterion (rule O10c).  Rows ascending."""
    a = list(map(_f64, (x, y, z, vx, vy, vz, m, rnb, rout)))
    n = a[0].shape[0]
    off = np.zeros(n + 1, dtype=np.int64)
    args = [C.c_int64(n)] + [_p(v, C.c_double) for v in a] + [C.c_double(G), C.c_double(Cv), _p(off, C.c_int64)]
    _lib().ora_neighbors_orbit_direct(*args, None)
    idx = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
    _lib().ora_neighbors_orbit_direct(*args, _p(idx, C.c_int32))
    return off, idx[: int(off[-1])]


def dK(x, lam, q):
    L = _lib()
    L.ora_dK.restype = C.c_double; L.ora_dK.argtypes = [C.c_double] * 3
    return np.vectorize(lambda v: L.ora_dK(float(v), float(lam), float(q)))(np.asarray(x, dtype=np.float64))


def short_range(x, y, z, vx, vy, vz, m, rout, offsets, indices, G: float, rho: float):
    """H_S over the neighbour rows: (ax, ay, az, jx, jy, jz, pot), see ora_short_range."""
    a = list(map(_f64, (x, y, z, vx, vy, vz, m, rout)))
    n = a[0].shape[0]
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    idx = np.ascontiguousarray(indices, dtype=np.int32)
    if idx.size == 0:
        idx = np.zeros(1, dtype=np.int32)
    out = [np.zeros(n) for _ in range(7)]
    _lib().ora_short_range(C.c_int64(n), *[_p(v, C.c_double) for v in a], _p(off, C.c_int64), _p(idx, C.c_int32),
                           C.c_double(G), C.c_double(rho), *[_p(o, C.c_double) for o in out])
    return tuple(out)


def clusters(offsets, indices):
    """Connected components of the neighbour graph: (label int32[N] = smallest member, n_clusters)."""
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    idx = np.ascontiguousarray(indices, dtype=np.int32)
    n = off.shape[0] - 1
    lab = np.zeros(max(n, 1), dtype=np.int32)
    L = _lib()
    L.ora_clusters.restype = C.c_int64
    nc = int(L.ora_clusters(C.c_int64(n), _p(off, C.c_int64), _p(idx if idx.size else np.zeros(1, np.int32), C.c_int32), _p(lab, C.c_int32)))
    return lab[:n], nc


@dataclass
class NodeTable:
    level: np.ndarray; begin: np.ndarray; end: np.ndarray; leaf: np.ndarray; nchild: np.ndarray
    M: np.ndarray; com: np.ndarray; lo: np.ndarray; hi: np.ndarray; rmax: np.ndarray; Q: np.ndarray


class OracleTree:
    """Rules O1-O9 on the CPU in fp64."""

    def __init__(self, x, y, z, m, rout, params: OracleParams, rsearch=None):
        self.params = params
        self._arr = tuple(map(_f64, (x, y, z, m, rout)))
        self.N = self._arr[0].shape[0]
        rs = None if rsearch is None else _f64(rsearch)
        self._rs = rs
        L = _lib()
        self._h = C.c_void_p(L.ora_tree_build(C.c_int64(self.N), *[_p(a, C.c_double) for a in self._arr],
                                              None if rs is None else _p(rs, C.c_double), C.byref(params)))
        self.n_nodes = int(L.ora_tree_n_nodes(self._h))
        self.n_groups = int(L.ora_tree_n_groups(self._h))

    def __del__(self):
        try:
            if self._h:
                _lib().ora_tree_free(self._h)
                self._h = None
        except Exception:
            pass

    def root(self):
        out = np.zeros(4)
        _lib().ora_tree_root(self._h, _p(out, C.c_double))
        return out[:3].copy(), float(out[3])

    def keys(self):
        key = np.zeros(self.N, dtype=np.uint64); perm = np.zeros(self.N, dtype=np.int32)
        if self.N:
            _lib().ora_tree_keys(self._h, _p(key, C.c_uint64), _p(perm, C.c_int32))
        return key, perm

    def nodes(self) -> NodeTable:
        I = np.zeros((self.n_nodes, 5), dtype=np.int64); D = np.zeros((self.n_nodes, 17))
        if self.n_nodes:
            _lib().ora_tree_nodes(self._h, _p(I, C.c_int64), _p(D, C.c_double))
        return NodeTable(I[:, 0], I[:, 1], I[:, 2], I[:, 3], I[:, 4], D[:, 0], D[:, 1:4], D[:, 4:7], D[:, 7:10],
                         D[:, 10], D[:, 11:17])

    def groups(self):
        I = np.zeros((self.n_groups, 2), dtype=np.int64); D = np.zeros((self.n_groups, 7))
        if self.n_groups:
            _lib().ora_tree_groups(self._h, _p(I, C.c_int64), _p(D, C.c_double))
        return I[:, 0], I[:, 1], D[:, 0:3], D[:, 3:6], D[:, 6]

    def walk_counts(self):
        """(per-group int64[n_groups,4] = n_i, n_ep, n_sp, n_ep_ranges ; N_epep ; N_epsp)."""
        out = np.zeros((self.n_groups, 4), dtype=np.int64); tot = np.zeros(2, dtype=np.int64)
        if self.n_groups:
            _lib().ora_walk_counts(self._h, _p(out, C.c_int64), _p(tot, C.c_int64))
        return out, int(tot[0]), int(tot[1])

    def walk_lists(self, g: int):
        """(sp canonical ids int64[n_sp], ep int64[n_ranges,3] = begin,end,near) of group g."""
        n2 = np.zeros(2, dtype=np.int64)
        _lib().ora_walk_lists(self._h, C.c_int64(g), None, C.c_int64(0), None, C.c_int64(0), _p(n2, C.c_int64))
        sp = np.zeros(max(int(n2[0]), 1), dtype=np.int64); ep = np.zeros((max(int(n2[1]), 1), 3), dtype=np.int64)
        _lib().ora_walk_lists(self._h, C.c_int64(g), _p(sp, C.c_int64), C.c_int64(sp.shape[0]), _p(ep, C.c_int64),
                              C.c_int64(ep.shape[0]), _p(n2, C.c_int64))
        return sp[: int(n2[0])], ep[: int(n2[1])]

    def force(self, groups=None):
        """Long-range acc/pot (original order) from self-built lists; NaN where not computed."""
        out = [np.full(self.N, np.nan) for _ in range(4)]
        if groups is None:
            ns, sp = 0, None
        else:
            groups = np.ascontiguousarray(groups, dtype=np.int64)
            ns, sp = groups.shape[0], _p(groups, C.c_int64)
        if self.N:
            _lib().ora_tree_force(self._h, C.c_int64(ns), sp, *[_p(o, C.c_double) for o in out])
        return tuple(out)

    def eval_lists(self, gb, ge, sp_canon, ep_ranges):
        """Mode 2: evaluate imported lists for sorted positions [gb, ge).  Returns full-length arrays (NaN elsewhere)."""
        out = [np.full(self.N, np.nan) for _ in range(4)]
        sp = np.ascontiguousarray(sp_canon, dtype=np.int64)
        ep = np.ascontiguousarray(ep_ranges, dtype=np.int64).reshape(-1, 2)
        _lib().ora_eval_lists(self._h, C.c_int64(gb), C.c_int64(ge), C.c_int64(sp.shape[0]), _p(sp, C.c_int64),
                              C.c_int64(ep.shape[0]), _p(ep, C.c_int64), *[_p(o, C.c_double) for o in out])
        return tuple(out)

    def neighbors_orbit(self, vx, vy, vz, Cv: float, groups=None):
        """Rule O10: orbit-filtered CSR neighbour list (velocities in the caller's order; rows ascending)."""
        vx, vy, vz = map(_f64, (vx, vy, vz))
        off = np.zeros(self.N + 1, dtype=np.int64)
        if self.N == 0:
            return off, np.zeros(0, dtype=np.int32)
        if groups is None:
            ns, sp = 0, None
        else:
            groups = np.ascontiguousarray(groups, dtype=np.int64)
            ns, sp = groups.shape[0], _p(groups, C.c_int64)
        a = [self._h, C.c_int64(ns), sp, _p(vx, C.c_double), _p(vy, C.c_double), _p(vz, C.c_double), C.c_double(Cv), _p(off, C.c_int64)]
        _lib().ora_tree_neighbors_orbit_sel(*a, None)
        idx = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
        _lib().ora_tree_neighbors_orbit_sel(*a, _p(idx, C.c_int32))
        return off, idx[: int(off[-1])]

    def neighbors(self, groups=None):
        """CSR neighbour list (rows ascending).  groups: only the particles of these i-groups get rows."""
        off = np.zeros(self.N + 1, dtype=np.int64)
        if self.N == 0:
            return off, np.zeros(0, dtype=np.int32)
        if groups is None:
            ns, sp = 0, None
        else:
            groups = np.ascontiguousarray(groups, dtype=np.int64)
            ns, sp = groups.shape[0], _p(groups, C.c_int64)
        _lib().ora_tree_neighbors_sel(self._h, C.c_int64(ns), sp, _p(off, C.c_int64), None)
        idx = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
        _lib().ora_tree_neighbors_sel(self._h, C.c_int64(ns), sp, _p(off, C.c_int64), _p(idx, C.c_int32))
        return off, idx[: int(off[-1])]
