"""ctypes binding of include/petar.h -- argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libpetar_b200.so")
_LIB = None

EXPORTS = [
    "petar_workspace_bytes", "petar_tree_build", "petar_tree_rebuild", "petar_long_range_force", "petar_neighbor_list",
    "petar_tree_status", "petar_tree_destroy", "petar_strerror", "petar_debug_export",
    "petar_set_profiling", "petar_stage_times", "petar_launch_count", "petar_probe_fp32",
    "petar_search_radii", "petar_neighbor_list_orbit", "petar_clusters_workspace_bytes", "petar_clusters",
    "petar_short_range_workspace_bytes", "petar_short_range_force", "petar_short_range_force_noalloc",
    "petar_kick", "petar_artificial_particles", "petar_tidal_tensor_fit", "petar_orbit_sampling",
]
STAGE_NAMES = ["bbox_keys", "sort", "gather", "tree", "moments", "groups", "walk", "force", "neighbor", "force_units", "walk_super", "force_refine"]
DBG = dict(HEADER=0, ROOT=1, KEYS=2, PERM=3, NODE_INT=4, NODE_DBL=5, GROUP_INT=6, GROUP_DBL=7, GROUP_CNT=8,
           LIST_OFFS=9, LISTS=10, GROUP_SUPER=11)


class PetarError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: error {code}: {petar_strerror(code)}")


class PetarParams(C.Structure):
    _fields_ = [("G", C.c_double), ("theta", C.c_double), ("r_in_over_r_out", C.c_double),
                ("multipole", C.c_int32), ("n_leaf_limit", C.c_int32), ("n_group_limit", C.c_int32),
                ("flags", C.c_int32), ("list_entries_per_particle", C.c_double), ("nodes_per_particle", C.c_double)]

    @classmethod
    def make(cls, theta, multipole, G=1.0, rho=0.1, n_leaf=8, n_group=64, list_entries_per_particle=0.0, nodes_per_particle=0.0):
        return cls(float(G), float(theta), float(rho), int(multipole), int(n_leaf), int(n_group), 0,
                   float(list_entries_per_particle), float(nodes_per_particle))

    @classmethod
    def from_workload(cls, w, theta=None, multipole=None, **kw):
        return cls.make(w.theta if theta is None else theta, w.multipole if multipole is None else multipole,
                        G=w.G, rho=w.r_in_over_r_out, n_leaf=w.n_leaf_limit, n_group=w.n_group_limit, **kw)


class PetarCounts(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_groups", "n_nodes", "n_epep", "n_epsp", "n_epep_near", "n_ep_list",
                                         "n_sp_list", "list_entries_used", "n_epsp_common", "n_refined")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


def library_path() -> str:
    return _LIB_PATH


def lib():
    """Loads the CUDA library; raises if it has not been built (there is no fallback)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(_LIB_PATH):
            raise FileNotFoundError(f"{_LIB_PATH} is missing: run `python -m paper_2006_16560_b200.build` "
                                    "(the CUDA extension is the only implementation; there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.petar_workspace_bytes.restype = C.c_size_t
        L.petar_workspace_bytes.argtypes = [C.c_int64, C.POINTER(PetarParams)]
        L.petar_tree_build.restype = C.c_int
        L.petar_tree_build.argtypes = [C.c_void_p] * 6 + [C.c_int64, C.POINTER(PetarParams), C.c_void_p, C.c_size_t,
                                                          C.c_void_p, C.POINTER(C.c_void_p)]
        L.petar_tree_rebuild.restype = C.c_int
        L.petar_tree_rebuild.argtypes = [C.c_void_p] * 7 + [C.c_void_p]
        L.petar_long_range_force.restype = C.c_int
        L.petar_long_range_force.argtypes = [C.c_void_p] * 5 + [C.POINTER(PetarCounts), C.c_void_p]
        L.petar_neighbor_list.restype = C.c_int
        L.petar_neighbor_list.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.petar_search_radii.restype = C.c_int
        L.petar_search_radii.argtypes = [C.c_void_p] * 4 + [C.c_double, C.c_double, C.c_int64, C.c_void_p, C.c_void_p]
        L.petar_neighbor_list_orbit.restype = C.c_int
        L.petar_neighbor_list_orbit.argtypes = [C.c_void_p] * 4 + [C.c_double, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.petar_clusters_workspace_bytes.restype = C.c_size_t
        L.petar_clusters_workspace_bytes.argtypes = [C.c_int64]
        L.petar_clusters.restype = C.c_int
        L.petar_clusters.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_size_t, C.c_void_p]
        L.petar_short_range_workspace_bytes.restype = C.c_size_t
        L.petar_short_range_workspace_bytes.argtypes = [C.c_int64]
        L.petar_short_range_force.restype = C.c_int
        L.petar_short_range_force.argtypes = ([C.c_void_p] * 10 + [C.c_int64, C.c_double, C.c_double] + [C.c_void_p] * 7
                                              + [C.c_void_p, C.c_size_t, C.c_void_p])
        L.petar_short_range_force_noalloc.restype = C.c_int
        L.petar_short_range_force_noalloc.argtypes = ([C.c_void_p] * 10 + [C.c_int64, C.c_double, C.c_double] + [C.c_void_p] * 7
                                                      + [C.c_void_p])
        L.petar_kick.restype = C.c_int
        L.petar_kick.argtypes = [C.c_void_p] * 6 + [C.c_double, C.c_int64, C.c_void_p]
        L.petar_artificial_particles.restype = C.c_int
        L.petar_artificial_particles.argtypes = [C.c_void_p] * 8 + [C.c_int64, C.c_double, C.c_int32, C.c_double] + [C.c_void_p] * 6
        L.petar_orbit_sampling.restype = C.c_int
        L.petar_orbit_sampling.argtypes = [C.c_void_p] * 8 + [C.c_int64, C.c_double, C.c_int32] + [C.c_void_p] * 5
        L.petar_tidal_tensor_fit.restype = C.c_int
        L.petar_tidal_tensor_fit.argtypes = [C.c_void_p] * 4 + [C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
        L.petar_tree_status.restype = C.c_int
        L.petar_tree_status.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.c_void_p]
        L.petar_tree_destroy.restype = C.c_int
        L.petar_tree_destroy.argtypes = [C.c_void_p]
        L.petar_strerror.restype = C.c_char_p
        L.petar_strerror.argtypes = [C.c_int]
        L.petar_debug_export.restype = C.c_int
        L.petar_debug_export.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
        L.petar_set_profiling.restype = C.c_int
        L.petar_set_profiling.argtypes = [C.c_int]
        L.petar_stage_times.restype = C.c_int
        L.petar_stage_times.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        L.petar_launch_count.restype = C.c_int64
        L.petar_probe_fp32.restype = C.c_int
        L.petar_probe_fp32.argtypes = [C.c_int64, C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        _LIB = L
    return _LIB


def exported_symbols():
    L = lib()
    return [s for s in EXPORTS if hasattr(L, s)]


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


# ---- same names as the C ABI -----------------------------------------------------------------------
def petar_workspace_bytes(N: int, params: PetarParams) -> int:
    return int(lib().petar_workspace_bytes(C.c_int64(N), C.byref(params)))


def petar_strerror(code: int) -> str:
    return lib().petar_strerror(int(code)).decode()


def petar_tree_build(x, y, z, m, r_out, r_search, N, params, workspace, stream=None):
    """Returns the opaque tree handle (int).  All tensors are CUDA fp64 tensors, workspace a CUDA uint8 tensor."""
    h = C.c_void_p()
    rc = lib().petar_tree_build(_ptr(x), _ptr(y), _ptr(z), _ptr(m), _ptr(r_out), _ptr(r_search), C.c_int64(N),
                                C.byref(params), _ptr(workspace), C.c_size_t(0 if workspace is None else workspace.numel()),
                                _stream(stream), C.byref(h))
    if rc:
        raise PetarError(rc, "petar_tree_build")
    return h


def petar_tree_rebuild(tree, x, y, z, m, r_out, r_search, stream=None) -> None:
    """Steps S0-S6 into an existing handle (same N, parameters and workspace)."""
    rc = lib().petar_tree_rebuild(tree, _ptr(x), _ptr(y), _ptr(z), _ptr(m), _ptr(r_out), _ptr(r_search), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_tree_rebuild")


def petar_long_range_force(tree, acc_x, acc_y, acc_z, pot, want_counts=False, stream=None):
    counts = PetarCounts() if want_counts else None
    rc = lib().petar_long_range_force(tree, _ptr(acc_x), _ptr(acc_y), _ptr(acc_z), _ptr(pot),
                                      C.byref(counts) if want_counts else None, _stream(stream))
    if rc:
        raise PetarError(rc, "petar_long_range_force")
    return counts


def petar_neighbor_list(tree, offsets, indices, capacity, status_dev=None, stream=None):
    rc = lib().petar_neighbor_list(tree, _ptr(offsets), _ptr(indices), C.c_int64(capacity), _ptr(status_dev), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_neighbor_list")


def petar_search_radii(vx, vy, vz, r_out, C_r: float, dt_L: float, N: int, r_search_out, stream=None) -> None:
    rc = lib().petar_search_radii(_ptr(vx), _ptr(vy), _ptr(vz), _ptr(r_out), C.c_double(C_r), C.c_double(dt_L), C.c_int64(N),
                                  _ptr(r_search_out), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_search_radii")


def petar_neighbor_list_orbit(tree, vx, vy, vz, C_V: float, offsets, indices, capacity, status_dev=None, stream=None) -> None:
    rc = lib().petar_neighbor_list_orbit(tree, _ptr(vx), _ptr(vy), _ptr(vz), C.c_double(C_V), _ptr(offsets), _ptr(indices),
                                         C.c_int64(capacity), _ptr(status_dev), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_neighbor_list_orbit")


def petar_clusters_workspace_bytes(N: int) -> int:
    return int(lib().petar_clusters_workspace_bytes(C.c_int64(N)))


def petar_clusters(offsets, indices, N: int, label, n_clusters_dev=None, cluster_offsets=None, members=None, workspace=None,
                   stream=None) -> None:
    rc = lib().petar_clusters(_ptr(offsets), _ptr(indices), C.c_int64(N), _ptr(label), _ptr(n_clusters_dev), _ptr(cluster_offsets),
                              _ptr(members), _ptr(workspace), C.c_size_t(0 if workspace is None else workspace.numel()), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_clusters")


def petar_short_range_workspace_bytes(N: int) -> int:
    return int(lib().petar_short_range_workspace_bytes(C.c_int64(N)))


def petar_short_range_force(x, y, z, vx, vy, vz, m, r_out, offsets, indices, N: int, G: float, rho: float,
                            acc, jerk, pot, workspace, stream=None) -> None:
    """acc, jerk: 3-tuples of CUDA fp64 tensors (entries may be None); pot: tensor or None."""
    rc = lib().petar_short_range_force(*[_ptr(a) for a in (x, y, z, vx, vy, vz, m, r_out, offsets, indices)], C.c_int64(N),
                                       C.c_double(G), C.c_double(rho), *[_ptr(a) for a in acc], *[_ptr(a) for a in jerk], _ptr(pot),
                                       _ptr(workspace), C.c_size_t(0 if workspace is None else workspace.numel()), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_short_range_force")


SHORT_RANGE_NOALLOC_MAX_N = 65536     # PETAR_SHORT_RANGE_NOALLOC_MAX_N of include/petar.h


def petar_short_range_force_noalloc(x, y, z, vx, vy, vz, m, r_out, offsets, indices, N: int, G: float, rho: float,
                                    acc, jerk, pot, stream=None) -> None:
    """petar_short_range_force without the workspace argument, for callers that cannot allocate device memory (a plug-in
    that only receives pointers, a spent memory pool, a loop that must not stall on cudaMalloc).  The scratch is a fixed
    array inside the library, so N <= SHORT_RANGE_NOALLOC_MAX_N (else PetarError with code -6) and calls that overlap on
    the GPU must be ordered by the caller.  Arguments as petar_short_range_force."""
    rc = lib().petar_short_range_force_noalloc(*[_ptr(a) for a in (x, y, z, vx, vy, vz, m, r_out, offsets, indices)], C.c_int64(N),
                                               C.c_double(G), C.c_double(rho), *[_ptr(a) for a in acc], *[_ptr(a) for a in jerk],
                                               _ptr(pot), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_short_range_force_noalloc")


def petar_kick(vx, vy, vz, ax, ay, az, dt: float, N: int, stream=None) -> None:
    rc = lib().petar_kick(*[_ptr(a) for a in (vx, vy, vz, ax, ay, az)], C.c_double(dt), C.c_int64(N), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_kick")


def art_count(order: int) -> int:
    return 8 if order == 2 else 12


def petar_artificial_particles(x, y, z, vx, vy, vz, m, pairs, n_bin: int, G: float, order: int, tt_scale: float,
                               art_x, art_y, art_z, art_m, elem=None, stream=None) -> None:
    rc = lib().petar_artificial_particles(*[_ptr(a) for a in (x, y, z, vx, vy, vz, m, pairs)], C.c_int64(n_bin), C.c_double(G),
                                          C.c_int32(order), C.c_double(tt_scale), *[_ptr(a) for a in (art_x, art_y, art_z, art_m, elem)],
                                          _stream(stream))
    if rc:
        raise PetarError(rc, "petar_artificial_particles")


def petar_orbit_sampling(x, y, z, vx, vy, vz, m, pairs, n_bin: int, G: float, n_split: int, out_x, out_y, out_z, out_m,
                         stream=None) -> None:
    rc = lib().petar_orbit_sampling(*[_ptr(a) for a in (x, y, z, vx, vy, vz, m, pairs)], C.c_int64(n_bin), C.c_double(G),
                                    C.c_int32(n_split), *[_ptr(a) for a in (out_x, out_y, out_z, out_m)], _stream(stream))
    if rc:
        raise PetarError(rc, "petar_orbit_sampling")


def petar_tidal_tensor_fit(acc_x, acc_y, acc_z, elem, n_bin: int, order: int, T, stream=None) -> None:
    rc = lib().petar_tidal_tensor_fit(_ptr(acc_x), _ptr(acc_y), _ptr(acc_z), _ptr(elem), C.c_int64(n_bin), C.c_int32(order), _ptr(T),
                                      _stream(stream))
    if rc:
        raise PetarError(rc, "petar_tidal_tensor_fit")


def petar_tree_status(tree, stream=None) -> int:
    st = C.c_int32(0)
    rc = lib().petar_tree_status(tree, C.byref(st), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_tree_status")
    return int(st.value)


def petar_tree_destroy(tree) -> None:
    lib().petar_tree_destroy(tree)


def petar_debug_export(tree, what: int, dst, stream=None) -> None:
    rc = lib().petar_debug_export(tree, int(what), _ptr(dst), C.c_size_t(dst.numel() * dst.element_size()), _stream(stream))
    if rc:
        raise PetarError(rc, f"petar_debug_export({what})")


def petar_set_profiling(on: bool) -> None:
    lib().petar_set_profiling(1 if on else 0)


def petar_stage_times(tree):
    arr = (C.c_float * len(STAGE_NAMES))()
    rc = lib().petar_stage_times(tree, arr)
    if rc:
        raise PetarError(rc, "petar_stage_times")
    return {n: float(arr[i]) for i, n in enumerate(STAGE_NAMES)}


def petar_probe_fp32(iters: int, scratch, stream=None) -> float:
    """Enqueues the FFMA probe kernel; returns the flops it executes (time it with CUDA events)."""
    fl = C.c_double(0.0)
    rc = lib().petar_probe_fp32(C.c_int64(iters), C.byref(fl), _ptr(scratch), _stream(stream))
    if rc:
        raise PetarError(rc, "petar_probe_fp32")
    return float(fl.value)


def petar_launch_count() -> int:
    return int(lib().petar_launch_count())


# ---- convenience holder (owns the torch tensors; still marshalling only) --------------------------------
class Tree:
    """Device buffers + tree handle for one particle set.  `build()` may be called repeatedly."""

    def __init__(self, N: int, params: PetarParams, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2006_16560_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.N, self.params, self.device = int(N), params, torch.device(device)
        nbytes = petar_workspace_bytes(self.N, params)
        if nbytes == 0:
            raise PetarError(-1, "petar_workspace_bytes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        assert self.workspace.data_ptr() % 256 == 0
        self.handle = None
        self.inputs = None
        f64 = dict(dtype=torch.float64, device=self.device)
        self.acc_x, self.acc_y, self.acc_z, self.pot = (torch.empty(self.N, **f64) for _ in range(4))
        self.offsets = torch.empty(self.N + 1, dtype=torch.int64, device=self.device)
        self.indices = None
        self.nb_status = torch.zeros(1, dtype=torch.int32, device=self.device)

    def upload(self, x, y, z, m, r_out, r_search=None):
        t = self.torch
        conv = lambda a: None if a is None else t.as_tensor(a, dtype=t.float64).to(self.device, non_blocking=True).contiguous()
        self.inputs = tuple(conv(a) for a in (x, y, z, m, r_out, r_search))
        return self.inputs

    def build(self, stream=None):
        if self.handle is None:
            self.handle = petar_tree_build(*self.inputs, self.N, self.params, self.workspace, stream)
        else:
            petar_tree_rebuild(self.handle, *self.inputs, stream)
        return self.handle

    def force(self, want_counts=False, stream=None):
        return petar_long_range_force(self.handle, self.acc_x, self.acc_y, self.acc_z, self.pot, want_counts, stream)

    def neighbors(self, stream=None):
        """Two-phase neighbour output; returns (offsets, indices) device tensors."""
        t = self.torch
        petar_neighbor_list(self.handle, self.offsets, None, 0, None, stream)
        total = int(self.offsets[-1].item()) if self.N else 0
        if self.indices is None or self.indices.numel() < max(total, 1):
            self.indices = t.empty(max(total, 1), dtype=t.int32, device=self.device)
        petar_neighbor_list(self.handle, self.offsets, self.indices, self.indices.numel(), self.nb_status, stream)
        return self.offsets, self.indices[:total]

    def neighbors_orbit(self, vx, vy, vz, C_V: float = 1.5, stream=None):
        """Two-phase output of the orbit-dependent criterion (velocities: CUDA fp64 tensors, caller's order)."""
        t = self.torch
        petar_neighbor_list_orbit(self.handle, vx, vy, vz, C_V, self.offsets, None, 0, None, stream)
        total = int(self.offsets[-1].item()) if self.N else 0
        if self.indices is None or self.indices.numel() < max(total, 1):
            self.indices = t.empty(max(total, 1), dtype=t.int32, device=self.device)
        petar_neighbor_list_orbit(self.handle, vx, vy, vz, C_V, self.offsets, self.indices, self.indices.numel(), self.nb_status, stream)
        return self.offsets, self.indices[:total]

    def clusters(self, offsets, indices, members: bool = True, stream=None):
        """Connected components of a neighbour list: (label, n_clusters tensor, cluster_offsets, members)."""
        t = self.torch
        n = self.N
        label = t.empty(max(n, 1), dtype=t.int32, device=self.device)
        ncl = t.zeros(1, dtype=t.int64, device=self.device)
        coff = mem = ws = None
        if members:
            coff = t.zeros(n + 1, dtype=t.int64, device=self.device)
            mem = t.empty(max(n, 1), dtype=t.int32, device=self.device)
            ws = t.empty(petar_clusters_workspace_bytes(n), dtype=t.uint8, device=self.device)
        petar_clusters(offsets, indices, n, label, ncl, coff, mem, ws, stream)
        return label[:n], ncl, coff, None if mem is None else mem[:n]

    def export(self, name: str):
        """Test hook: returns a torch tensor with the intermediate `name` (see petar_debug_export)."""
        t = self.torch
        hdr = t.zeros(8, dtype=t.int64, device=self.device)
        petar_debug_export(self.handle, DBG["HEADER"], hdr)
        nn, ng = int(hdr[0]), int(hdr[1])
        if name == "HEADER":
            return hdr
        n = self.N
        spec = dict(ROOT=(4, t.float64), KEYS=(n, t.int64), PERM=(n, t.int32), NODE_INT=(nn * 4, t.int32),
                    NODE_DBL=(nn * 17, t.float64), GROUP_INT=(ng * 2, t.int32), GROUP_DBL=(ng * 7, t.float64),
                    GROUP_CNT=(ng * 4, t.int32), GROUP_SUPER=(ng * 8, t.int32), LIST_OFFS=(ng * 3 + 1, t.int64))
        if name == "LISTS":
            offs = self.export("LIST_OFFS")
            total = int(offs[-1])
            out = t.zeros(max(total, 1), dtype=t.int32, device=self.device)
            petar_debug_export(self.handle, DBG["LISTS"], out)
            return offs, out[:total]
        cnt, dt = spec[name]
        out = t.zeros(max(cnt, 1), dtype=dt, device=self.device)
        petar_debug_export(self.handle, DBG[name], out)
        return out[:cnt]

    def close(self):
        if self.handle is not None:
            petar_tree_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
