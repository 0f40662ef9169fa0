"""GPU parity of SURVEY.md 8(f) rank 3 through the C-ABI: kick, artificial particles (tidal-tensor measure points,
centre-of-mass point, pseudoparticles of Eq. 38) and the tidal-tensor fit (Table 1), against the numpy oracle."""
import numpy as np
import pytest

from oracle import artificial as A
from workloads import make_workload

pytestmark = pytest.mark.gpu


def _P():
    import paper_2006_16560_b200 as P
    return P


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _binaries(w):
    """Member pairs of the generator's binaries: mutually nearest, bound pairs (found with numpy, not the library)."""
    import oracle
    off, idx = oracle.neighbors_direct(w.x, w.y, w.z, np.full(w.N, 2.1e-3))
    pairs = []
    for i in range(w.N):
        for j in idx[off[i]:off[i + 1]]:
            if i < j:
                d = np.array([w.x[j] - w.x[i], w.y[j] - w.y[i], w.z[j] - w.z[i]])
                v = np.array([w.vx[j] - w.vx[i], w.vy[j] - w.vy[i], w.vz[j] - w.vz[i]])
                if 2 / np.linalg.norm(d) - v.dot(v) / (w.m[i] + w.m[j]) > 1 / 2e-3:
                    pairs.append((i, j))
    return np.array(pairs, dtype=np.int32)


def test_kick_bit_exact():
    import torch
    P = _P()
    rng = np.random.default_rng(0)
    n = 100003
    v = [rng.normal(size=n) for _ in range(3)]; a = [rng.normal(size=n) for _ in range(3)]
    dv = [_dev(q) for q in v]; da = [_dev(q) for q in a]
    P.petar_kick(*dv, *da, 2.0 ** -11, n)
    for k in range(3):
        assert np.array_equal(dv[k].cpu().numpy(), A.kick(v[k], a[k], 2.0 ** -11))
    P.petar_kick(*dv, *da, 0.5, 0)                                   # N = 0
    with pytest.raises(P.PetarError):
        P.petar_kick(None, None, None, None, None, None, 0.5, 10)


@pytest.mark.parametrize("order", [2, 3])
def test_artificial_particles_and_tidal_fit(order):
    import torch
    P = _P()
    w = make_workload(2, N=20000, velocities=True)
    pairs = _binaries(w)
    nb = len(pairs)
    assert nb > 3000
    # a few degenerate pairs as well: an unbound pair (two singles far apart) and a pair listed in reverse order
    pairs = np.concatenate([pairs, [[0, w.N - 1]], pairs[:1, ::-1]]).astype(np.int32)
    nb = len(pairs)
    na = P.art_count(order)
    ins = [_dev(q) for q in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m)]
    out = [torch.empty(nb * na, dtype=torch.float64, device="cuda") for _ in range(4)]
    elem = torch.empty(nb * 8, dtype=torch.float64, device="cuda")
    tt_scale = 2.0
    P.petar_artificial_particles(*ins, _dev(pairs), nb, w.G, order, tt_scale, *out, elem)
    gx, gy, gz, gm = (o.cpu().numpy().reshape(nb, na) for o in out)
    el = elem.cpu().numpy().reshape(nb, 8)
    n_bound = 0
    for b in range(nb):
        i, j = pairs[b]
        art = A.artificial_particles([w.x[i], w.y[i], w.z[i]], [w.vx[i], w.vy[i], w.vz[i]], w.m[i],
                                     [w.x[j], w.y[j], w.z[j]], [w.vx[j], w.vy[j], w.vz[j]], w.m[j], w.G, order, tt_scale)
        assert bool(el[b, 6]) == art["bound"]
        assert np.array_equal(gm[b], art["mass"])
        g = np.stack([gx[b], gy[b], gz[b]], axis=1)
        scale = art["a"] if art["bound"] else 1.0
        # positions relative to the centre of mass, on the scale of the orbit (the frame vectors of a nearly circular
        # orbit are the least well conditioned quantity: e enters through a cancellation of order 1e-16 / e)
        tol = 1e-9 if (not art["bound"] or art["e"] > 1e-3) else 1e-6
        assert np.max(np.abs(g - art["pos"])) < tol * scale + 1e-15 * np.abs(art["cm"]).max(), (b, art["e"])
        if art["bound"]:
            n_bound += 1
            assert el[b, 0] == pytest.approx(art["a"], rel=1e-10) and el[b, 1] == pytest.approx(art["e"], abs=1e-9)
            assert el[b, 2] == pytest.approx(art["d_c"], rel=1e-10)
    assert n_bound >= nb - 1 and not bool(el[nb - 2, 6])
    # tidal fit: accelerations of a smooth external field (three distant point masses) at the artificial particles
    src = np.array([[3.0, -2.0, 1.5], [-4.0, 0.5, 2.0], [0.3, 5.0, -3.0]]); ms = np.array([2.5, 1.0, 4.0])

    def field(p):
        d = src[None, :, :] - p[:, None, :]
        return np.sum(ms[None, :, None] * d / np.linalg.norm(d, axis=2, keepdims=True) ** 3, axis=1)

    pos = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)
    acc = field(pos)
    nc = 6 if order == 2 else 16
    T = torch.empty(nb * nc, dtype=torch.float64, device="cuda")
    P.petar_tidal_tensor_fit(_dev(acc[:, 0]), _dev(acc[:, 1]), _dev(acc[:, 2]), elem, nb, order, T)
    Tg = T.cpu().numpy().reshape(nb, nc)
    ntt = na - 4
    acc = acc.reshape(nb, na, 3)
    for b in list(range(0, nb, 97)) + [nb - 2, nb - 1]:
        if el[b, 2] > 0:
            To = A.tidal_fit(order, el[b, 2], acc[b, :ntt], acc[b, ntt])
            # A' = A(r_k) - A(r_cm) cancels to ~d_c/R of A: compare on the scale |A| / d_c (and / d_c^2)
            sc = np.linalg.norm(acc[b, ntt]) / el[b, 2]
            assert np.max(np.abs(Tg[b, :6] - To[:6])) < 1e-9 * sc
            if order == 3:
                assert np.max(np.abs(Tg[b, 6:] - To[6:])) < 1e-9 * sc / el[b, 2]
        else:
            assert np.all(Tg[b] == 0)
    with pytest.raises(P.PetarError):
        P.petar_artificial_particles(*ins, _dev(pairs), nb, w.G, 4, tt_scale, *out, elem)


def test_artificial_particles_through_the_long_range_force():
    """The pipeline of PAPER.md Fig. 2 steps 3-4: artificial particles appended to the particle set (members of those
    binaries massless in the tree), long-range force of the extended set against the oracle (1e-5), tidal tensors fitted
    from the measured accelerations."""
    import torch
    import oracle
    from workloads.generators import changeover_radii
    P = _P()
    w = make_workload(2, N=20011, velocities=True)
    pairs = w.meta["pairs"][:400].copy()
    nb, order = len(pairs), 2
    na = P.art_count(order)
    ins = [_dev(q) for q in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m)]
    out = [torch.empty(nb * na, dtype=torch.float64, device="cuda") for _ in range(4)]
    elem = torch.empty(nb * 8, dtype=torch.float64, device="cuda")
    P.petar_artificial_particles(*ins, _dev(pairs), nb, w.G, order, 2.0, *out, elem)
    ax_, ay_, az_, am_ = (o.cpu().numpy() for o in out)
    m_tree = w.m.copy(); m_tree[pairs.ravel()] = 0.0                 # their mass is carried by the pseudoparticles
    x = np.concatenate([w.x, ax_]); y = np.concatenate([w.y, ay_]); z = np.concatenate([w.z, az_]); m = np.concatenate([m_tree, am_])
    assert m.sum() == pytest.approx(w.m.sum(), rel=1e-12)
    r_out = np.concatenate([w.r_out, np.maximum(changeover_radii(np.concatenate([w.m, am_]), w.r_out_ref)[w.N:], w.r_out_ref)])
    n = len(x)
    params = P.PetarParams.from_workload(w)
    t = P.Tree(n, params)
    t.upload(x, y, z, m, r_out)
    t.build()
    t.force()
    T = oracle.OracleTree(x, y, z, m, r_out, oracle.OracleParams.from_workload(w))
    a = T.force()
    g = [v.cpu().numpy() for v in (t.acc_x, t.acc_y, t.acc_z, t.pot)]
    den = np.sqrt(a[0] ** 2 + a[1] ** 2 + a[2] ** 2)
    err = np.sqrt(sum((g[k] - a[k]) ** 2 for k in range(3))) / den
    assert err.max() < 1e-5 and np.max(np.abs(g[3] - a[3]) / np.abs(a[3])) < 1e-5
    assert P.petar_tree_status(t.handle) == 0
    # tidal tensors from the measured accelerations (the artificial particles are the last nb * na entries)
    Tt = torch.empty(nb * 6, dtype=torch.float64, device="cuda")
    P.petar_tidal_tensor_fit(t.acc_x[w.N:], t.acc_y[w.N:], t.acc_z[w.N:], elem, nb, order, Tt)
    Tg = Tt.cpu().numpy().reshape(nb, 6)
    el = elem.cpu().numpy().reshape(nb, 8)
    acc_o = np.stack([a[0][w.N:], a[1][w.N:], a[2][w.N:]], axis=1).reshape(nb, na, 3)
    rel = []
    for b in range(nb):
        To = A.tidal_fit(order, el[b, 2], acc_o[b, :4], acc_o[b, 4])
        rel.append(np.linalg.norm(Tg[b] - To) / np.linalg.norm(To))
    # (the long-range field is not harmonic inside the changeover radius of the binary's own pseudoparticles, so no
    # trace condition holds.)  The measured differences A(r_k) - A(r_cm) are ~d_c/R of the fp32-accurate accelerations: percent-level agreement
    assert np.median(rel) < 0.05
    t.close()


def test_orbit_sampling():
    import torch
    P = _P()
    w = make_workload(2, N=20000, velocities=True)
    pairs = np.concatenate([w.meta["pairs"][:3000], [[0, w.N - 1]]]).astype(np.int32)       # + one unbound pair
    nb, ns = len(pairs), 8
    ins = [_dev(q) for q in (w.x, w.y, w.z, w.vx, w.vy, w.vz, w.m)]
    out = [torch.empty(nb * 2 * ns, dtype=torch.float64, device="cuda") for _ in range(4)]
    P.petar_orbit_sampling(*ins, _dev(pairs), nb, w.G, ns, *out)
    gx, gy, gz, gm = (o.cpu().numpy().reshape(nb, 2 * ns) for o in out)
    for b in range(0, nb, 13):
        i, j = pairs[b]
        x1 = np.array([w.x[i], w.y[i], w.z[i]]); x2 = np.array([w.x[j], w.y[j], w.z[j]])
        v1 = np.array([w.vx[i], w.vy[i], w.vz[i]]); v2 = np.array([w.vx[j], w.vy[j], w.vz[j]])
        el = A.kepler_elements(x2 - x1, v2 - v1, w.G * (w.m[i] + w.m[j]))
        cm = (w.m[i] * x1 + w.m[j] * x2) / (w.m[i] + w.m[j])
        assert el["bound"]
        pos, mass = A.orbit_sampling(w.m[i], w.m[j], el["a"], el["e"], el["P"], el["Q"], cm, ns)
        g = np.stack([gx[b], gy[b], gz[b]], axis=1)
        tol = 1e-9 if el["e"] > 1e-3 else 1e-6
        assert np.max(np.abs(g - pos)) < tol * el["a"] + 1e-15 * np.abs(cm).max()
        assert np.allclose(gm[b], mass, rtol=1e-12)
    # every binary keeps its mass; the unbound pair sits at its centre of mass
    assert np.allclose(gm.sum(axis=1), w.m[pairs[:, 0]] + w.m[pairs[:, 1]], rtol=1e-13)
    b = nb - 1
    cm = (w.m[0] * np.array([w.x[0], w.y[0], w.z[0]]) + w.m[-1] * np.array([w.x[-1], w.y[-1], w.z[-1]])) / (w.m[0] + w.m[-1])
    assert np.allclose(np.stack([gx[b], gy[b], gz[b]], axis=1), cm)
    with pytest.raises(P.PetarError):
        P.petar_orbit_sampling(*ins, _dev(pairs), nb, w.G, 0, *out)
