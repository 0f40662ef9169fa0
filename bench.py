#!/usr/bin/env python
"""bench.py -- long-range P3T force step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 3]

One "step" = the whole hot path on one batch of synthetic input:
petar_tree_build + petar_long_range_force + petar_neighbor_list (count phase and fill phase).
Workload: BASELINE.json configs[2] (N = 1,048,576 Plummer sphere, Kroupa IMF, 100 % binaries,
r_out = 0.003, theta = 0.3, quadrupole), the configuration the metric is quoted on.

Prints ONE JSON line (rank 0).  `value` = long-range interactions per second of the whole job,
interactions = sum over i-groups of n_i * (n_ep + n_sp) as counted by the walk (rule O7),
inputs resident in HBM.  `e2e` = the same metric through the C-ABI with HOST buffers (pinned
host inputs copied in, accelerations/potentials/neighbour lists copied out, every step).
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
Multi-GPU: the path is single-GPU by design ("replicas only"): N ranks run N
independent replicas, no data-path collective; value = total interactions / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOP_NEWTON, FLOP_CUT, FLOP_QUAD = 20, 49, 53      # fixed flops-per-interaction convention
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the force kernels, from the committed `ncu --set full` capture of
# THIS round's build at config 3 (profiles/ncu_r02_force.md).  Emitted only for that configuration; any other run reports null.
TRAFFIC_NCU = {"capture": "profiles/ncu_r03_force.md", "config": 3, "k_force_units_tc": 131.9e6, "k_force_units": 44.6e6, "k_force": 1231.2e6, "stage": 176.5e6}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--N", type=int, default=None, help="override the particle count (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-groups", type=int, default=40000, help="i-groups in the oracle's timed sample")
    ap.add_argument("--theta-sweep", action="store_true",
                    help="BASELINE.json configs[3]: after the headline run, sweep theta over 0.2, 0.3, 0.5, 0.7 (interactions/s and "
                         "RMS force error against the direct long-range sum on a 4096-particle subsample, oracle on the host)")
    return ap.parse_args()


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except Exception:
                continue
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for nme, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_oracle_sample(w, n_groups_sample: int, seed: int = 1):
    """Times the oracle as it stands on a bounded sample: full tree build + walk + force of sampled i-groups."""
    import oracle
    op = oracle.OracleParams.from_workload(w)
    t0 = time.perf_counter()
    T = oracle.OracleTree(w.x, w.y, w.z, w.m, w.r_out, op)
    t_build = time.perf_counter() - t0
    ng = T.n_groups
    sel = np.sort(np.random.default_rng(seed).choice(ng, size=min(n_groups_sample, ng), replace=False)).astype(np.int64)
    t0 = time.perf_counter()
    T.force(sel)
    t_force = time.perf_counter() - t0
    # interactions of the sample, counted exactly by the oracle's own (untimed) count walk: sum over the sampled groups of
    # n_i * (n_ep + n_sp), rule O7
    oc, _, _ = T.walk_counts()
    n_int = int((oc[sel, 0] * (oc[sel, 1] + oc[sel, 2])).sum())
    return dict(value=n_int / t_force, unit="interactions/s", cores=oracle.num_threads(), kind="oracle",
                sample=f"fp64 oracle (oracle/petar_oracle.c, OpenMP): tree build of all N={w.N} particles ({t_build:.2f} s, untimed in value) "
                       f"+ walk and force of {len(sel)} of {ng} i-groups ({t_force:.2f} s, {n_int} interactions, counted exactly)",
                seconds=t_force, build_seconds=t_build)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make_workload
    w = make_workload(args.config, N=args.N)
    vals = []
    per_step = max(50, args.cpu_groups // max(1, args.steps + args.warmup))
    base = None
    for s in range(args.warmup + args.steps):
        r = cpu_oracle_sample(w, per_step, seed=s)
        if s >= args.warmup:
            vals.append(r)
        base = r
    v = float(np.mean([r["value"] for r in vals]))
    ms = float(np.mean([r["seconds"] for r in vals])) * 1e3
    out = dict(metric="long-range interactions/sec", value=v, unit="interactions/s", n_gpus=args.gpus, steps=args.steps,
               warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
               data="synthetic", impl="reference",
               config={"workload": f"BASELINE.json configs[{args.config - 1}] (N={w.N}); each step = oracle walk+force of "
                                   f"{per_step} sampled i-groups on the host CPU"},
               cpu_baseline=dict(value=v, unit="interactions/s", cores=base["cores"], kind="oracle", sample=base["sample"]),
               e2e=dict(value=v, unit="interactions/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(out), flush=True)


def aggregate_ranks(ms_step: float, e2e_ms: float, interactions: float, dist=None, device="cpu"):
    """Whole-job figures of N independent replicas: time = MAX over ranks, interactions = SUM over ranks
    (tests/test_multi_rank.py runs this very function on two gloo ranks)."""
    if dist is not None:
        import torch
        t = torch.tensor([ms_step, e2e_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step, e2e_ms = float(t[0]), float(t[1])
        s = torch.tensor([interactions], dtype=torch.float64, device=device)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
        interactions = float(s[0])
    return ms_step, e2e_ms, interactions


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import paper_2006_16560_b200 as P
    from workloads import make_workload

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU path)")
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist_.init_process_group("nccl", device_id=dev)
        dist = dist_
    W = max(3, args.warmup)
    K = args.steps
    cfg = args.config
    # weak scaling: every rank holds its own replica of the workload (different seed per rank)
    from workloads.generators import SEED_BASE
    w = make_workload(cfg, N=args.N, seed=SEED_BASE + cfg + 1000 * rank if rank else None)
    N = w.N
    params = P.PetarParams.from_workload(w)
    P.petar_set_profiling(True)
    tree = P.Tree(N, params, device=dev)
    stream = torch.cuda.current_stream()
    # pinned host inputs (e2e) and their device copies (device-resident measurement)
    host_in = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (w.x, w.y, w.z, w.m, w.r_out)]
    dev_in = [torch.empty(N, dtype=torch.float64, device=dev) for _ in range(5)]
    for d, h in zip(dev_in, host_in):
        d.copy_(h, non_blocking=True)
    tree.inputs = tuple(dev_in) + (None,)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step_device(capacity_holder):
        tree.build(stream)
        P.petar_long_range_force(tree.handle, tree.acc_x, tree.acc_y, tree.acc_z, tree.pot, False, stream)
        P.petar_neighbor_list(tree.handle, tree.offsets, None, 0, None, stream)                  # count + scan
        P.petar_neighbor_list(tree.handle, tree.offsets, capacity_holder[0], capacity_holder[0].numel(), tree.nb_status, stream)

    # one untimed pass to size the neighbour index buffer (two-phase output) and to read the counters
    tree.build(stream)
    counts = P.petar_long_range_force(tree.handle, tree.acc_x, tree.acc_y, tree.acc_z, tree.pot, True, stream)
    off, idx = tree.neighbors(stream)
    nb_total = int(off[-1].item())
    cap = [torch.empty(int(nb_total * 1.1) + 1024, dtype=torch.int32, device=dev)]
    n_inter = counts.n_epep + counts.n_epsp
    quad = params.multipole >= 2
    flop_sp = FLOP_QUAD if quad else FLOP_NEWTON
    flops_units = flop_sp * counts.n_epsp_common                      # phase A: k_force_units_tc + k_force_units (super-group-wide cells)
    flops_near = FLOP_CUT * counts.n_epep_near                        # k_force_near: the pairs inside the changeover radius
    flops_groups = (FLOP_NEWTON * (counts.n_epep - counts.n_epep_near)
                    + flop_sp * (counts.n_epsp - counts.n_epsp_common))  # phase B: k_force (the groups' own lists, Newtonian pairs + cells)
    flops_step = flops_units + flops_near + flops_groups

    for _ in range(W):
        flush.fill_(1)
        step_device(cap)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    sampler = ClockSampler(local); sampler.start()
    launches0 = P.petar_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    stage_sum = {k: 0.0 for k in P.STAGE_NAMES}
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    for k in range(K):
        flush.fill_(k & 255)                     # L2 flush between timed iterations (outside the events)
        ev[k][0].record(stream)
        step_device(cap)
        ev[k][1].record(stream)
        ev[k][1].synchronize()
        st = P.petar_stage_times(tree.handle)
        for name, v in st.items():
            stage_sum[name] += v
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    launches = P.petar_launch_count() - launches0
    clocks = sampler.stop()
    if dist: dist.barrier()
    ms_total = sum(a.elapsed_time(b) for a, b in ev)
    status = P.petar_tree_status(tree.handle)

    # ---- the same work with the calls in the other order (neighbour count first): the per-group walk then runs ALONE before the
    #      force kernels instead of beside force phase A, which gives every kernel's duration without the overlap (not part of `value`)
    stage_seq = {k: 0.0 for k in P.STAGE_NAMES}
    seq_ms = 0.0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for rep in range(3):
        flush.fill_(rep)
        e0.record(stream)
        tree.build(stream)
        P.petar_neighbor_list(tree.handle, tree.offsets, None, 0, None, stream)
        P.petar_long_range_force(tree.handle, tree.acc_x, tree.acc_y, tree.acc_z, tree.pot, False, stream)
        P.petar_neighbor_list(tree.handle, tree.offsets, cap[0], cap[0].numel(), tree.nb_status, stream)
        e1.record(stream); e1.synchronize()
        seq_ms += e0.elapsed_time(e1) / 3
        for name, v in P.petar_stage_times(tree.handle).items():
            stage_seq[name] += v / 3

    # ---- e2e: HOST buffers through the C-ABI, copies inside the timed region ---------------------------
    host_out = [torch.empty(N, dtype=torch.float64).pin_memory() for _ in range(4)]
    host_off = torch.empty(N + 1, dtype=torch.int64).pin_memory()
    host_idx = torch.empty(cap[0].numel(), dtype=torch.int32).pin_memory()
    e2e_ms, d2h_bytes = 0.0, 0

    copy_stream = torch.cuda.Stream(device=dev)
    ev_force = torch.cuda.Event()

    def step_e2e():
        """Host buffers in, host buffers out.  The caller overlaps what the asynchronous C-ABI lets it overlap: the
        accelerations travel back on a second stream while the neighbour lists are built."""
        nonlocal d2h_bytes
        for d, h in zip(dev_in, host_in):
            d.copy_(h, non_blocking=True)
        tree.build(stream)
        P.petar_long_range_force(tree.handle, tree.acc_x, tree.acc_y, tree.acc_z, tree.pot, False, stream)
        ev_force.record(stream)
        with torch.cuda.stream(copy_stream):
            copy_stream.wait_event(ev_force)
            for h, d in zip(host_out, (tree.acc_x, tree.acc_y, tree.acc_z, tree.pot)):
                h.copy_(d, non_blocking=True)
        P.petar_neighbor_list(tree.handle, tree.offsets, None, 0, None, stream)
        total = int(tree.offsets[-1].item())                 # the caller reads the total, then asks for the rows
        if total > cap[0].numel():
            cap[0] = torch.empty(int(total * 1.1), dtype=torch.int32, device=dev)
        P.petar_neighbor_list(tree.handle, tree.offsets, cap[0], cap[0].numel(), tree.nb_status, stream)
        host_off.copy_(tree.offsets, non_blocking=True)
        host_idx[:total].copy_(cap[0][:total], non_blocking=True)
        stream.synchronize()
        copy_stream.synchronize()
        d2h_bytes = 4 * 8 * N + 8 * (N + 1) + 4 * total + 8

    step_e2e()
    torch.cuda.synchronize()
    Ke = K
    if dist: dist.barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        step_e2e()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / Ke
    h2d_bytes = 5 * 8 * N

    # ---- SURVEY 8(f) ranks 1-2, timed after the headline region (not part of `value`) -----------------------
    # Eq. 24 radii -> tree with r_search -> two-stage orbit-dependent neighbour list -> clusters
    next_rows = None
    if world == 1:
        wv = make_workload(cfg, N=args.N, velocities=True)
        vdev = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (wv.vx, wv.vy, wv.vz)]
        rs_dev = torch.empty(N, dtype=torch.float64, device=dev)
        label = torch.empty(N, dtype=torch.int32, device=dev); ncl = torch.zeros(1, dtype=torch.int64, device=dev)
        coff = torch.zeros(N + 1, dtype=torch.int64, device=dev); mem = torch.empty(N, dtype=torch.int32, device=dev)
        cws = torch.empty(P.petar_clusters_workspace_bytes(N), dtype=torch.uint8, device=dev)
        tree.inputs = tuple(dev_in) + (rs_dev,)
        sws = torch.empty(P.petar_short_range_workspace_bytes(N), dtype=torch.uint8, device=dev)
        sr_out = [torch.empty(N, dtype=torch.float64, device=dev) for _ in range(7)]
        evn = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
        acc = np.zeros(5)
        reps = max(3, min(K, 5))
        for rep in range(reps + 1):
            flush.fill_(rep & 255)
            evn[0].record(stream)
            P.petar_search_radii(*vdev, dev_in[4], 3.0, wv.dt_L, N, rs_dev, stream)
            evn[1].record(stream)
            tree.build(stream)
            evn[2].record(stream)
            P.petar_neighbor_list_orbit(tree.handle, *vdev, 1.5, tree.offsets, None, 0, None, stream)
            tot_o = int(tree.offsets[-1].item())
            if tot_o > cap[0].numel():
                cap[0] = torch.empty(int(tot_o * 1.1), dtype=torch.int32, device=dev)
            P.petar_neighbor_list_orbit(tree.handle, *vdev, 1.5, tree.offsets, cap[0], cap[0].numel(), tree.nb_status, stream)
            evn[3].record(stream)
            P.petar_clusters(tree.offsets, cap[0], N, label, ncl, coff, mem, cws, stream)
            evn[4].record(stream)
            P.petar_short_range_force(*dev_in[:3], *vdev, dev_in[3], dev_in[4], tree.offsets, cap[0], N, params.G, params.r_in_over_r_out,
                                      sr_out[0:3], sr_out[3:6], sr_out[6], sws, stream)
            evn[5].record(stream)
            evn[5].synchronize()
            if rep:                                   # first repetition = warm-up
                acc += np.array([evn[i].elapsed_time(evn[i + 1]) for i in range(5)])
        acc /= reps
        n_cl = int(ncl.item())
        hbm = float(peaks()[0].get("hbm_gbs", 6545.6))
        cl_bytes = 8 * (N + 1) + 4 * tot_o + 4 * N + 4 * (12 + 12) * N + 8 * N + 4 * N      # CSR read, labels, 4 sort passes, offsets, members
        next_rows = {
            "workload": "same config with Plummer velocities + binary orbital motion, C_r = 3, C_V = 1.5, dt_L = %g" % wv.dt_L,
            "search_radii_ms": acc[0], "search_radii_gbs": 40.0 * N / (acc[0] * 1e-3) / 1e9 if acc[0] > 0 else None,
            "tree_build_with_r_search_ms": acc[1],
            "walk_plus_neighbor_list_orbit_ms": acc[2], "neighbours_orbit": tot_o,
            "clusters_ms": acc[3], "n_clusters": n_cl, "clusters_algorithmic_gbs": cl_bytes / (acc[3] * 1e-3) / 1e9 if acc[3] > 0 else None,
            "clusters_frac_of_hbm": cl_bytes / (acc[3] * 1e-3) / 1e9 / hbm if acc[3] > 0 else None,
            "short_range_force_ms": acc[4],
            "short_range_algorithmic_gbs": (240.0 * N + 8.0 * (N + 1) + 68.0 * tot_o) / (acc[4] * 1e-3) / 1e9 if acc[4] > 0 else None,
            "short_range_frac_of_hbm": (240.0 * N + 8.0 * (N + 1) + 68.0 * tot_o) / (acc[4] * 1e-3) / 1e9 / hbm if acc[4] > 0 else None,
        }
        # rank 3: kick, artificial particles of every binary (3rd-order measure points + pseudoparticles), tensor fit
        pairs = wv.meta["pairs"]
        nbin = int(pairs.shape[0])
        if nbin:
            na, nc = P.art_count(3), 16
            pd = torch.from_numpy(np.ascontiguousarray(pairs)).to(dev)
            art = [torch.empty(nbin * na, dtype=torch.float64, device=dev) for _ in range(4)]
            elem = torch.empty(nbin * 8, dtype=torch.float64, device=dev)
            Tt = torch.empty(nbin * nc, dtype=torch.float64, device=dev)
            vk = [v.clone() for v in vdev]
            ev3 = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            acc3 = np.zeros(3)
            for rep in range(reps + 1):
                flush.fill_(rep & 255)
                ev3[0].record(stream)
                P.petar_kick(*vk, tree.acc_x, tree.acc_y, tree.acc_z, 0.5 * wv.dt_L, N, stream)
                ev3[1].record(stream)
                P.petar_artificial_particles(*dev_in[:3], *vdev, dev_in[3], pd, nbin, params.G, 3, 2.0, *art, elem, stream)
                ev3[2].record(stream)
                P.petar_tidal_tensor_fit(art[0], art[1], art[2], elem, nbin, 3, Tt, stream)      # (positions stand in for accelerations: timing only)
                ev3[3].record(stream)
                ev3[3].synchronize()
                if rep:
                    acc3 += np.array([ev3[i].elapsed_time(ev3[i + 1]) for i in range(3)])
            acc3 /= reps
            next_rows.update({
                "kick_ms": acc3[0], "kick_gbs": 72.0 * N / (acc3[0] * 1e-3) / 1e9,
                "n_binaries": nbin, "artificial_particles_ms": acc3[1],
                "artificial_particles_gbs": nbin * (2 * 56.0 + 8 + na * 32.0 + 64.0) / (acc3[1] * 1e-3) / 1e9,
                "tidal_tensor_fit_ms": acc3[2], "tidal_tensor_fit_gbs": nbin * (9 * 24.0 + 64.0 + nc * 8.0) / (acc3[2] * 1e-3) / 1e9,
            })
        tree.inputs = tuple(dev_in) + (None,)

    # ---- theta sweep (config 4 of BASELINE.json): interactions/s and RMS error vs the DEFINITION -----------------
    theta_sweep = None
    if args.theta_sweep and world == 1:
        import oracle
        tg = np.sort(np.random.default_rng(44).choice(N, size=min(4096, N), replace=False)).astype(np.int64)
        dref = oracle.direct(w.x, w.y, w.z, w.m, w.r_out, oracle.OracleParams.from_workload(w), "long", targets=tg)
        dn = np.sqrt(dref[0] ** 2 + dref[1] ** 2 + dref[2] ** 2)
        theta_sweep = []
        for th in (0.2, 0.3, 0.5, 0.7):
            pt = P.PetarParams.from_workload(w, theta=th)
            tt = P.Tree(N, pt, device=dev)
            tt.inputs = tuple(dev_in) + (None,)
            tt.build(stream)
            cth = P.petar_long_range_force(tt.handle, tt.acc_x, tt.acc_y, tt.acc_z, tt.pot, True, stream)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ms_th = 0.0
            for rep in range(3):
                flush.fill_(rep)
                a0.record(stream)
                tt.build(stream)
                P.petar_long_range_force(tt.handle, tt.acc_x, tt.acc_y, tt.acc_z, tt.pot, False, stream)
                a1.record(stream); a1.synchronize()
                ms_th += a0.elapsed_time(a1) / 3
            g = [v[torch.from_numpy(tg).to(dev)].cpu().numpy() for v in (tt.acc_x, tt.acc_y, tt.acc_z)]
            rel = np.sqrt(sum((g[k] - dref[k]) ** 2 for k in range(3))) / dn
            theta_sweep.append(dict(theta=th, interactions=int(cth.n_epep + cth.n_epsp), build_plus_force_ms=ms_th,
                                    interactions_per_s=(cth.n_epep + cth.n_epsp) / (ms_th * 1e-3),
                                    rms_rel_force_error_vs_direct_sum=float(np.sqrt(np.mean(rel ** 2))), targets=int(len(tg))))
            tt.close()

    # ---- FP32 peak probe (FFMA only), timed alone ------------------------------------------------------
    scratch = torch.zeros(2, dtype=torch.float32, device=dev)
    P.petar_probe_fp32(20000, scratch, stream)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream); fl = P.petar_probe_fp32(400000, scratch, stream); b.record(stream); b.synchronize()
    probe_tflops = fl / (a.elapsed_time(b) * 1e-3) / 1e12
    pk, pk_kind = peaks()
    sm_max = float(pk.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    nominal_fp32 = 2 * 128 * n_sm * sm_max * 1e6 / 1e12

    # ---- aggregate over ranks --------------------------------------------------------------------------
    # headline time per step: the MEDIAN of the K per-step CUDA-event times; the mean is kept beside it
    step_ms = sorted(a.elapsed_time(b) for a, b in ev)
    ms_median = step_ms[K // 2] if K % 2 else 0.5 * (step_ms[K // 2 - 1] + step_ms[K // 2])
    ms_mean = ms_total / K
    ms_step, e2e_ms, tot_inter = aggregate_ranks(ms_median, e2e_ms, float(n_inter), dist, dev)
    value = tot_inter / (ms_step * 1e-3)
    e2e_value = tot_inter / (e2e_ms * 1e-3)

    stage_ms = {k: v / K for k, v in stage_sum.items()}
    # HBM-side stages: algorithmic bytes per particle against the measured copy bandwidth
    hbm_peak = float(pk.get("hbm_gbs", 6545.6))
    # keys 36 B, sort ~200 B (8 + 8 x 24), gather 84 B per particle, S4-S6 (tree + moments + groups) ~100 B together
    stage_bytes = {"bbox_keys": (36.0, ("bbox_keys",)), "sort": (200.0, ("sort",)), "gather": (84.0, ("gather",)),
                   "tree_moments_groups": (100.0, ("tree", "moments", "groups"))}
    hbm_stages = {}
    for name, (bpp, parts) in stage_bytes.items():
        ms_st = sum(stage_ms.get(q, 0.0) for q in parts)
        if ms_st > 0.0:
            gbs = bpp * N / (ms_st * 1e-3) / 1e9
            hbm_stages[name] = dict(ms=ms_st, bytes_per_particle=bpp, achieved_gbs=gbs, frac_of_hbm=gbs / hbm_peak)
    # k_force (phase B): PETAR_STAGE_FORCE is an event pair around the single k_force launch, on the stream it is launched on, inside
    # the timed region (nothing runs beside it: the side stream has been joined).  Phase A is a two-stream STAGE (unit table +
    # k_force_units_tc on the caller's stream; k_walk, k_force_units, k_force_near beside them on the library's side stream) and is
    # called a stage here; its kernels' time without the walk beside them is `ms_alone` (the sequential call order timed after the
    # headline region).  The 53 flops per quadrupole interaction are counted wherever they are executed (tensor or CUDA cores).
    phase_a = "stage force_units (unit table + k_force_units_tc | k_walk + k_force_units + k_force_near)" if quad else \
              "stage force_units (unit table | k_walk + k_force_units + k_force_near)"
    kern = [dict(kernel="k_force", timed="event pair around the single launch, in the timed region", ms=stage_ms["force"],
                 ms_alone=stage_seq["force"], flops_per_launch=float(flops_groups)),
            dict(kernel=phase_a, timed="event pair around a two-stream stage; ms_alone = the same kernels without k_walk beside them",
                 ms=stage_ms["force_units"], ms_alone=stage_seq["force_units"], flops_per_launch=float(flops_units),
                 note="k_force_near's changeover pairs (flops_k_force_near) are credited to neither entry: that kernel runs inside "
                      "this stage in the timed region and outside every stage in the sequential order")]
    for kd in kern:
        kd["frac_alone"] = kd["flops_per_launch"] / (kd["ms_alone"] * 1e-3) / 1e12 / nominal_fp32 if kd["ms_alone"] > 0 else 0.0
        kd["achieved"] = kd["flops_per_launch"] / (kd["ms"] * 1e-3) / 1e12 if kd["ms"] > 0 else 0.0
        kd["frac"] = kd["achieved"] / nominal_fp32
        kd["share_of_step"] = kd["ms"] / ms_step
    dom = max(kern, key=lambda kd: kd["ms_alone"])            # the dominant kernel: by its own duration, not by an overlapped stage's
    force_ms = stage_ms["force_units"] + stage_ms["force"]
    achieved_both = flops_step / (force_ms * 1e-3) / 1e12

    if rank == 0:
        out = dict(
            metric="long-range interactions/sec", value=value, unit="interactions/s", n_gpus=world, steps=K, warmup=W,
            ms_per_step=ms_step, ms_per_step_mean=ms_mean, ms_per_step_min=step_ms[0], ms_per_step_max=step_ms[-1], higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
            config={"workload": f"BASELINE.json configs[{cfg - 1}]: N={N} Plummer (Henon units), "
                                f"{w.meta['masses']} masses, {2 * w.meta['n_pairs']} stars in binaries, r_out_ref={w.r_out_ref}, "
                                f"theta={w.theta}, multipole={params.multipole}, leaf<=8, group<=64",
                    "step": "petar_tree_build + petar_long_range_force + petar_neighbor_list (count phase + fill phase)",
                    "l2": "256 MB buffer written between timed iterations (L2 flush), outside the per-step CUDA events",
                    "interactions_per_step": int(n_inter), "n_epep": int(counts.n_epep), "n_epsp": int(counts.n_epsp),
                    "n_epep_changeover": int(counts.n_epep_near), "n_epsp_common": int(counts.n_epsp_common),
                    "n_refined": int(counts.n_refined), "neighbours": nb_total, "n_groups": int(counts.n_groups),
                    "n_nodes": int(counts.n_nodes), "status": status, "multi_gpu": "replicas only (no data-path collective)"},
            stage_ms=stage_ms,
            stage_ms_sequential=dict(stage_seq, step=seq_ms,
                                     note="calls in the order build, neighbour count, force, neighbour fill: the per-group walk runs alone; "
                                          "kernel durations without the overlap (3 repetitions after the timed region)"),
            stage_note="the per-group walk (stage walk) runs on the library's side stream BESIDE force phase A (stage force_units): the two "
                       "stage times overlap and each is longer than when run alone",
            hbm_stages=dict(peak_gbs=hbm_peak, note="keys / sort / tree stages: algorithmic bytes over stage time; at N = 2^20 the working "
                            "set (12-116 MB) sits in the 126 MB L2 and the stages are launch- and latency-bound, the fraction of HBM "
                            "bandwidth only means something at --config 5 (N = 10^7)", stages=hbm_stages),
            e2e=dict(value=e2e_value, unit="interactions/s", ms_per_step=e2e_ms, h2d_bytes_per_step=h2d_bytes,
                     d2h_bytes_per_step=d2h_bytes, steps=Ke),
            gpu_launches=int(launches),
            clocks=clocks,
            roofline=dict(bound="alu", kernel=dom["kernel"], achieved=dom["achieved"], peak=nominal_fp32, unit="TFLOP/s",
                          frac=dom["frac"],
                          traffic=TRAFFIC_NCU.get(dom["kernel"].split()[0]) if (cfg == TRAFFIC_NCU["config"] and args.N is None) else None,
                          traffic_source=TRAFFIC_NCU["capture"],
                          peak_kind=f"nominal CUDA-core FP32: 2 x 128 lanes x {n_sm} SMs x {sm_max:.0f} MHz (sm_max_mhz of MEASURED_PEAKS.json, {pk_kind})",
                          peak_measured_ffma_probe=probe_tflops, frac_of_probe=dom["achieved"] / probe_tflops,
                          flops_convention=f"{FLOP_NEWTON}/{FLOP_CUT}/{FLOP_QUAD} flops per Newtonian / changeover / quadrupole interaction",
                          flops_per_launch=dom["flops_per_launch"], kernel_ms=dom["ms"], kernel_share_of_step=dom["share_of_step"],
                          flops_k_force_near=float(flops_near), force_kernels=kern, both_force_kernels=dict(ms=force_ms, achieved=achieved_both, frac=achieved_both / nominal_fp32,
                                                                      share_of_step=force_ms / ms_step),
                          hbm_peak_gbs=pk.get("hbm_gbs")),
            wall_s_timed_region=t_wall,
        )
        if next_rows is not None:
            out["next_rows"] = next_rows
        if theta_sweep is not None:
            out["theta_sweep"] = theta_sweep
        if not args.no_cpu_baseline and world == 1:
            import oracle
            cb = cpu_oracle_sample(w, args.cpu_groups)
            out["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
            ncores = oracle.num_threads()
            oracle.set_num_threads(1)                      # the same oracle on ONE core, on a 16 times smaller sample
            c1 = cpu_oracle_sample(w, max(50, args.cpu_groups // 16), seed=2)
            oracle.set_num_threads(ncores)
            out["cpu_baseline"]["single_thread_value"] = c1["value"]
            out["cpu_baseline"]["single_thread_sample"] = c1["sample"]
        print(json.dumps(out), flush=True)
    if dist:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
