"""petar_short_range_force_noalloc against petar_short_range_force (GPU, through the C ABI).

Who needs the entry point: callers that cannot allocate device memory -- a plug-in that a host application hands
device pointers to, code living inside a memory pool that is already fully handed out, an integrator loop that must not
stall on cudaMalloc -- and so cannot give petar_short_range_force its workspace.  The variant keeps the packed records
and the long-row queue in a fixed array inside the library (at most SHORT_RANGE_NOALLOC_MAX_N particles).

What is checked: the variant returns what the existing path returns (the tolerance of tests/test_gpu_short.py; the
kernels are the same, so the difference is in fact zero) on two calls in a row.  The calls differ in N, in the radii
and in the neighbour list, and the first one leaves long rows queued: the second would go wrong if the counter it shares
with the first were not cleared, or if it read records the first call packed.  Sizes beyond the limit are refused.

The file is named so that pytest collects it after every other test file: with `pytest -x` a failure here hides nothing.
It uses no state of other tests and passes alone in a fresh process as well (the first call on the device looks up the
array's address)."""
import numpy as np
import pytest

from workloads import make_workload

pytestmark = pytest.mark.gpu
TOL = 1e-11          # tests/test_gpu_short.py


def _brute_force_neighbours(x, y, z, rout):
    """CSR list { j != i : r_ij < max(rout_i, rout_j) } by the double loop in numpy blocks (input of both paths)."""
    n = len(x)
    rows = []
    for b in range(0, n, 512):
        e = min(n, b + 512)
        d2 = (x[b:e, None] - x[None, :]) ** 2 + (y[b:e, None] - y[None, :]) ** 2 + (z[b:e, None] - z[None, :]) ** 2
        R = np.maximum(rout[b:e, None], rout[None, :])
        hit = d2 < R * R
        hit[np.arange(e - b), np.arange(b, e)] = False
        rows.extend(np.nonzero(h)[0].astype(np.int32) for h in hit)
    off = np.zeros(n + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(r) for r in rows])
    idx = np.concatenate(rows) if off[-1] else np.zeros(0, np.int32)
    return off, idx


def _both_paths(w, n, rout):
    import torch
    import paper_2006_16560_b200 as P

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a)).cuda()

    arrs = [a[:n] for a in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m)] + [rout[:n]]
    off, idx = _brute_force_neighbours(arrs[0], arrs[1], arrs[2], arrs[7])
    ins = [dev(a) for a in arrs] + [dev(off), dev(idx if len(idx) else np.zeros(1, np.int32))]
    nan = lambda: [torch.full((n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(7)]
    ref, new = nan(), nan()
    ws = torch.empty(P.petar_short_range_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    P.petar_short_range_force(*ins, n, w.G, w.r_in_over_r_out, ref[0:3], ref[3:6], ref[6], ws)
    P.petar_short_range_force_noalloc(*ins, n, w.G, w.r_in_over_r_out, new[0:3], new[3:6], new[6])
    torch.cuda.synchronize()
    return [v.cpu().numpy() for v in ref], [v.cpu().numpy() for v in new], off


def _assert_same(ref, new):
    for v in ref + new:
        assert np.all(np.isfinite(v))                      # every entry was written by both
    for lo in (0, 3):                                      # acceleration, jerk: vector error over vector norm
        den = np.sqrt(ref[lo] ** 2 + ref[lo + 1] ** 2 + ref[lo + 2] ** 2)
        err = np.sqrt(sum((new[lo + k] - ref[lo + k]) ** 2 for k in range(3)))
        assert np.all(err[den == 0] == 0)
        assert np.all(err[den > 0] <= TOL * den[den > 0])
    assert np.all(np.abs(new[6] - ref[6]) <= TOL * np.abs(ref[6]))


def test_noalloc_matches_workspace_path_on_two_calls_in_a_row():
    w = make_workload(1, velocities=True)                  # N = 4096 Plummer sphere
    # call 1: four times the radius => rows of > 32 entries in the core, so the shared long-row queue is in use
    ref, new, off = _both_paths(w, w.N, 4.0 * w.r_out)
    assert np.diff(off).max() > 32 and (ref[6] != 0).sum() > 1000
    _assert_same(ref, new)
    # call 2, straight after: fewer particles, the configured radii, short rows only; the array holds call 1's leftovers
    ref2, new2, off2 = _both_paths(w, 3001, w.r_out)
    assert 0 < np.diff(off2).max() <= 32 and (ref2[6] != 0).sum() > 100
    _assert_same(ref2, new2)


def test_noalloc_refuses_sizes_beyond_its_array():
    import torch
    import paper_2006_16560_b200 as P
    t = torch.zeros(8, dtype=torch.float64, device="cuda")
    off = torch.zeros(9, dtype=torch.int64, device="cuda")
    idx = torch.zeros(1, dtype=torch.int32, device="cuda")
    with pytest.raises(P.PetarError) as e:
        P.petar_short_range_force_noalloc(t, t, t, t, t, t, t, t, off, idx, P.SHORT_RANGE_NOALLOC_MAX_N + 1, 1.0, 0.1,
                                          (t, None, None), (None, None, None), None)
    assert e.value.code == -6 and "capacity" in str(e.value)
    # at the size of the arrays given the same call goes through
    P.petar_short_range_force_noalloc(t, t, t, t, t, t, t + 1.0, t + 1.0, off, idx, 8, 1.0, 0.1, (t.clone(), None, None), (None, None, None), None)
    torch.cuda.synchronize()
