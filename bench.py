#!/usr/bin/env python
"""Benchmark of the FMM cell-to-cell interaction step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg5|cfg3|cfg2] [--theta 0.5] [--ncell 256]

A "step" is one pass of the whole hot path over one batch: stage the sources (set_moments), the
interaction kernel (interact), store/copy the expansions (get_expansions).  Default workload is
config 5 (256^3 cells = 32768 sub-grids, two-polytrope binary, theta = 0.5, correction on), the
configuration BASELINE.json's metric is quoted on.  Prints ONE JSON line (rank 0).

N > 1 (torchrun): every rank runs an independent problem of the same shape (its own seed) --
the path shards by sub-problem with no data-path collective ("scaling": "weak"); timing is the
max over ranks between barriers.

--impl reference times the CPU oracle (oracle/, test infrastructure) on the host cores on a
bounded sample of the same workload; it is a deliberately plain program, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fmm_cell_interactions_per_s"
UNIT = "interactions/s"
FP64_LANES_PER_SM = 64        # FP64 FMA lanes per SM per clock on B200 (37.2 TFLOP/s at 148 SMs x 1965 MHz)
# flops per interaction the ROUND-1 kernel executed on the general multipole path (kind 0), for continuity with r01's frac:
# the round-2 kernel evaluates the same formula in fewer operations
ROUND1_FLOPS = {0: 224}


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def make_workload(name, theta, ncell, seed):
    import fmm_inputs as fi
    if name == "cfg5":
        w = fi.config5(seed=seed, theta=theta, ncell=ncell or 256)
    elif name == "cfg3":
        w = fi.config3(seed=seed, theta=theta, ncell=ncell or 128)
    elif name == "cfg2":
        w = fi.config2(seed=seed, theta=theta, ncell=ncell or 32)
    elif name == "cfg4":
        w = fi.config4(seed=seed, theta=theta, ncell=ncell or 128)
    else:
        raise SystemExit("unknown workload " + name)
    return w


def sample_regions(ncell, nregions, edge=16):
    """Stratified, deterministic sample of edge^3-cell regions (8 sub-grids each): corners,
    faces and interior of the lattice of regions."""
    m = ncell // edge
    picks = []
    i = 0
    while len(picks) < min(nregions, m ** 3):
        # low-discrepancy walk over the region lattice (includes (0,0,0) and boundary regions)
        a = (i * 7) % m
        b = (i * 11 + i // m) % m
        c = (i * 13 + i // (m * m) + (i // 3)) % m
        if (a, b, c) not in picks:
            picks.append((a, b, c))
        i += 1
    return [((a * edge, b * edge, c * edge), ((a + 1) * edge, (b + 1) * edge, (c + 1) * edge)) for a, b, c in picks]


def oracle_sample(w, theta, nregions, first=0):
    """Time the oracle, as it stands, on regions first .. first+nregions-1 of the stratified sample.
    Returns (interactions, seconds, threads, regions)."""
    import oracle
    regions = sample_regions(w.n[0], first + nregions)[first:]
    oracle.lib()
    t0 = time.perf_counter()
    total = 0
    for lo, hi in regions:
        if w.com_off is None:      # monopole workload (cfg 4)
            _, cnt = oracle.interact_monopole(w.n, w.h, theta, w.moments[0], lo, hi)
        else:
            _, _, cnt = oracle.interact_multipole(w.n, w.h, theta, w.moments, w.com_off, lo, hi, True)
        total += cnt
    return total, time.perf_counter() - t0, oracle.num_threads(), len(regions)


def oracle_sample_bounded(w, theta, target_s, pilot=4):
    """A sample sized for about target_s seconds of oracle work: a short pilot fixes the region count."""
    c0, s0, _, n0 = oracle_sample(w, theta, pilot)
    per_region = max(s0 / n0, 1e-6)
    m = (w.n[0] // 16) ** 3
    nreg = int(max(pilot, min(m - pilot, target_s / per_region)))
    return oracle_sample(w, theta, nreg, first=pilot if nreg + pilot <= m else 0)


def aggregate_over_ranks(ms_local, units_local, dist=None, device=None):
    """Whole-job numbers from per-rank ones: time = MAX over ranks, units = SUM over ranks
    (every rank works on its own problem; there is no data-path collective)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), int(units_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([int(units_local)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows[-3:]]
        sm, smax, power, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
                power.append(float(f[2]))
            except ValueError:
                continue
            for nme, val in zip(names, f[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    rank = env_int("RANK", 0)
    if rank != 0:
        return
    w = make_workload(args.workload, args.theta, args.ncell, args.seed)
    for _ in range(args.warmup):
        oracle_sample(w, args.theta, 1)
    tot, secs, nreg = 0, 0.0, 0
    threads = 1
    for _ in range(args.steps):
        c, s, threads, nr = oracle_sample_bounded(w, args.theta, args.ref_seconds)
        tot += c
        secs += s
        nreg = nr
    value = tot / secs
    sample = "%d regions of 16^3 cells (%d sub-grids) per step of %s" % (nreg, 8 * nreg, w.name)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s theta=%g correction=on" % (w.name, args.theta), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_solve(args):
    """--workload solve: the complete uniform-grid solve (octo_fmm_solver_*, NEXT f1) on the paper's uniform-sphere
    problem (section 3.4); a step = one solve (all levels); interactions = ordered pairs over all levels."""
    import numpy as np
    import torch
    import fmm_inputs as fi
    import oracle
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200 import build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = env_int("LOCAL_RANK", 0)
    if env_int("WORLD_SIZE", 1) > 1:
        raise SystemExit("bench.py --workload solve is a single-GPU line")
    torch.cuda.set_device(local)
    build.build()
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    n = args.ncell or 256
    h, mass, phi, r = fi.uniform_sphere(n)
    s = p.OctoFMMSolver(n, h, args.theta, True, device=local, stream=stream, two_rhs=True)
    n_int = s.interaction_count()
    levels, launches = s.num_levels()
    m_d = torch.from_numpy(mass).to(dev)
    out = torch.empty((4, n, n, n), dtype=torch.float64, device=dev)
    for _ in range(max(args.warmup, 3)):
        s.solve(m_d, out)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev0.record(stream)
    for _ in range(args.steps):
        s.solve(m_d, out)
    ev1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop(t0, time.perf_counter())
    ms = ev0.elapsed_time(ev1) / args.steps
    if s.status() != p.OK:
        raise SystemExit("bench.py: device reported status %d" % s.status())
    eps = np.abs(out[0].cpu().numpy() - phi) / np.abs(phi)
    # the second right-hand side (f2, L81-83) on the same tree and centres, timed beside the solve (not part of `value`):
    # d(mass)/dt of a rigid drift of the sphere along x, u . grad(rho) by central differences
    dm_d = (torch.roll(m_d, 1, 2) - torch.roll(m_d, -1, 2)) * (0.5 / h)
    out2 = torch.empty((n, n, n), dtype=torch.float64, device=dev)
    s.solve_rhs2(dm_d, out2)
    torch.cuda.synchronize()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record(stream)
    for _ in range(args.steps):
        s.solve_rhs2(dm_d, out2)
    ev3.record(stream)
    torch.cuda.synchronize()
    rhs2_ms = ev2.elapsed_time(ev3) / args.steps
    # both right-hand sides in one call (octo_fmm_solver_solve2): default, and with the fused kernel on every level
    both_ms = {}
    for fused in (0, 1):
        s.set_option("f2_fused", fused)
        s.solve2(m_d, dm_d, out, out2)
        torch.cuda.synchronize()
        ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev4.record(stream)
        for _ in range(args.steps):
            s.solve2(m_d, dm_d, out, out2)
        ev5.record(stream)
        torch.cuda.synchronize()
        both_ms[fused] = ev4.elapsed_time(ev5) / args.steps
    # like for like: the same two variants with the DIRECT kernel on every level (two launches vs one fused launch)
    s.set_option("kernel", 1)
    for fused in (0, 1):
        s.set_option("f2_fused", fused)
        s.solve2(m_d, dm_d, out, out2)
        torch.cuda.synchronize()
        ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev4.record(stream)
        for _ in range(args.steps):
            s.solve2(m_d, dm_d, out, out2)
        ev5.record(stream)
        torch.cuda.synchronize()
        both_ms[2 + fused] = ev4.elapsed_time(ev5) / args.steps
    s.set_option("kernel", 0)
    s.set_option("f2_fused", 0)
    s.solve(m_d, out)
    torch.cuda.synchronize()
    # end to end through the host-buffer entry point
    nb = p.octo_fmm_solver_host_scratch_bytes(s.cfg)
    scratch = torch.empty(nb, dtype=torch.uint8, device=dev)
    m_h = torch.from_numpy(mass).pin_memory()
    o_h = torch.empty((4, n, n, n), dtype=torch.float64).pin_memory()
    p.octo_fmm_solver_solve_host(s.handle, m_h, o_h, scratch, nb)
    t0 = time.perf_counter()
    for _ in range(max(args.e2e_steps, 1)):
        p.octo_fmm_solver_solve_host(s.handle, m_h, o_h, scratch, nb)
    e2e_ms = 1e3 * (time.perf_counter() - t0) / max(args.e2e_steps, 1)
    # the oracle's complete solve on the host cores, on the 64^3 version of the same problem
    nref = 64
    hr, mr, _, _ = fi.uniform_sphere(nref)
    oracle.lib()
    t0 = time.perf_counter()
    oracle.solve(nref, hr, args.theta, mr, True)
    t_ref = time.perf_counter() - t0
    cnt_ref = oracle.interact_monopole_leaf((nref, nref, nref), hr, args.theta, mr)[1]
    m = nref // 2
    while m >= 2:
        cnt_ref += oracle.interaction_count((m, m, m), args.theta)
        m //= 2
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sm_count * FP64_LANES_PER_SM * 2 * 1965.0e6 / 1e12
    leaf_int = s.leaf_interaction_count()
    f_multi = p.octo_fmm_flops_per_interaction_path(p.MULTIPOLE, True, False)[0]   # the solver's levels have no dipoles
    flops = float(f_multi) * (n_int - leaf_int) + 8.0 * leaf_int
    line = {"metric": METRIC, "value": n_int / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "complete solve, uniform sphere (paper 3.4), %d^3 leaf cells, theta=%g, correction on" % (n, args.theta),
                       "interactions_per_step": n_int, "leaf_interactions": leaf_int, "multipole_levels": levels,
                       "cells_per_s": n ** 3 / (ms * 1e-3), "l2": "arrays of the fine levels larger than L2",
                       "residual_vs_analytic": {"max": float(eps.max()), "mean": float(eps.mean())}},
            "roofline": {"bound": "alu", "kernel": "whole solve (m2l_staged_kernel at the n/2 level dominates)",
                         "achieved": flops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                         "frac": flops / (ms * 1e-3) / 1e12 / peak, "traffic": None},
            "cpu_baseline": {"value": cnt_ref / t_ref, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": "oracle.solve of the same problem at %d^3 (%d interactions) in %.1f s" % (nref, cnt_ref, t_ref)},
            "e2e": {"value": n_int / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(mass.nbytes),
                    "d2h_bytes_per_step": int(o_h.numel() * 8), "ms_per_step": e2e_ms},
            "second_rhs": {"ms_per_solve": rhs2_ms, "value": n_int / (rhs2_ms * 1e-3), "unit": UNIT,
                           "note": "octo_fmm_solver_solve_rhs2: d(phi)/dt from d(mass)/dt on the same tree and centres, "
                                   "correction off, dipole terms on; timed beside the solve, not part of value"},
            "two_rhs_one_call": {"ms_solve_plus_rhs2_separately": ms + rhs2_ms, "ms_solve2": both_ms[0],
                                 "ms_solve2_fused_on_every_level": both_ms[1],
                                 "ms_solve2_direct_kernels_two_launches_per_level": both_ms[2],
                                 "ms_solve2_direct_kernels_fused": both_ms[3],
                                 "note": "octo_fmm_solver_solve2: one upward and one downward pass for both right-hand sides; the "
                                         "fused kernel (shared list walk, separation, 1/r, radial factors) runs on the "
                                         "one-warp-per-cell levels by default and, for this measurement, on every level "
                                         "(m2l_direct2_kernel instead of two launches of the slab-fed kernel)"},
            "clocks": clocks, "gpu_launches": launches * args.steps}
    print(json.dumps(line))
    s.close()


def run_tree(args):
    """--workload tree: the solve on an ADAPTIVE oct-tree of 8^3 sub-grids (octo_fmm_tree_*, NEXT f3) on the two-star
    field of cfg 3/5 refined around the stars (the paper's density-based refinement, Eq. 34-35): 64^3 base
    cells, 3 levels, 256^3-equivalent inside the stars.  A step = one solve over all levels; interactions = ordered
    pairs of all kinds (multipole pairs, leaf-leaf point-mass pairs, point-mass pairs across refinement boundaries)."""
    import numpy as np
    import torch
    import fmm_inputs as fi
    import oracle
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200 import build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = env_int("LOCAL_RANK", 0)
    if env_int("WORLD_SIZE", 1) > 1:
        raise SystemExit("bench.py --workload tree is a single-GPU line")
    torch.cuda.set_device(local)
    build.build()
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    if args.workload == "tree9":
        # the paper's production depth (9 levels, L684): every level a window of a few sub-grids around one star
        n0, depth = args.ncell or 16, 9
        boxes, kinds, masses = fi.nested_tree(n0, depth, reach=2.6)     # 1.8 M leaf cells: the paper's "2 - 8 M cells" (L916)
        h0 = 1.0 / n0
        what = "9-level tree around one star (windows of <= %d cells per axis on every level; %d^3 lattice at the bottom)" % (
            max(max(b[3:]) for b in boxes[1:]), n0 << 8)
    else:
        n0, depth = args.ncell or 64, 3
        dense = fi.star_tree(n0, depth)
        boxes = fi.tree_boxes(dense)
        kinds, masses = fi.crop_tree(dense, boxes)
        h0 = dense.h0
        what = "two-star field refined around the stars, %d^3 base cells, %d levels (%d^3-equivalent)" % (n0, depth, n0 << (depth - 1))
        del dense
    t = p.OctoFMMTree(n0, h0, args.theta, kinds, True, device=local, stream=stream, box=boxes)
    mass = [torch.from_numpy(m).to(dev) for m in masses]
    out = t.empty_out()
    cnt, _ = t.interaction_counts(mass, out)
    n_int = cnt["m2l"] + cnt["p2p"] + cnt["cross"]
    launches = t.launches()
    leaves = [int((k == fi.TREE_LEAF).sum()) for k in kinds]
    for _ in range(max(args.warmup, 3)):
        t.solve(mass, out)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev0.record(stream)
    for _ in range(args.steps):
        t.solve(mass, out)
    ev1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop(t0, time.perf_counter())
    ms = ev0.elapsed_time(ev1) / args.steps
    if t.status() != p.OK:
        raise SystemExit("bench.py: device reported status %d" % t.status())
    # conservation on the timed result (L125, L127): sum of m g and of x x m g over the leaves of all levels
    F = torch.zeros(3, dtype=torch.float64, device=dev)
    Fa = torch.zeros((), dtype=torch.float64, device=dev)
    for l in range(depth):
        mg = mass[l][None] * out[l][1:4] * torch.from_numpy(kinds[l] == fi.TREE_LEAF).to(dev)[None]
        F += mg.sum(dim=(1, 2, 3))
        Fa += mg.abs().sum()
    net_force = float(F.abs().max() / Fa)
    # the second right-hand side (L81-83) on the same tree and centres, timed beside the solve (not part of `value`)
    dm = [m * (2.0 * torch.rand(m.shape, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(7 + l)) - 1.0)
          for l, m in enumerate(mass)]
    dphi = t.solve_rhs2(dm)
    torch.cuda.synchronize()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record(stream)
    for _ in range(args.steps):
        t.solve_rhs2(dm, dphi)
    ev3.record(stream)
    torch.cuda.synchronize()
    rhs2_ms = ev2.elapsed_time(ev3) / args.steps
    t.solve(mass, out)
    torch.cuda.synchronize()
    # end to end through the host-buffer entry point (pinned host arrays, every level)
    nb = p.octo_fmm_tree_host_scratch_bytes(t.handle)
    scratch = torch.empty(nb, dtype=torch.uint8, device=dev)
    m_h = [torch.from_numpy(m).pin_memory() for m in masses]
    o_h = [torch.empty((4,) + t.shape[l], dtype=torch.float64).pin_memory() for l in range(depth)]
    p.octo_fmm_tree_solve_host(t.handle, m_h, o_h, scratch, nb)
    t0 = time.perf_counter()
    for _ in range(max(args.e2e_steps, 1)):
        p.octo_fmm_tree_solve_host(t.handle, m_h, o_h, scratch, nb)
    e2e_ms = 1e3 * (time.perf_counter() - t0) / max(args.e2e_steps, 1)
    h2d = sum(int(m.numel() * 8) for m, k in zip(m_h, kinds) if (k == fi.TREE_LEAF).any())
    d2h = sum(int(o.numel() * 8) for o in o_h)
    same = all(bool(torch.equal(o_h[l], out[l].cpu())) for l in range(depth))
    # the oracle's tree solve on the host cores: the same tree for the 9-level workload, the same refinement pattern one
    # octave down (n0 / 2) for the two-star field
    oracle.lib()
    if args.workload == "tree9":
        o_n0, o_h0, o_kinds, o_masses, o_boxes = n0, h0, kinds, masses, boxes
        o_what = "oracle.solve_tree of the same tree"
    else:
        small = fi.star_tree(max(n0 // 2, 16), depth)
        o_boxes = fi.tree_boxes(small)
        o_kinds, o_masses = fi.crop_tree(small, o_boxes)
        o_n0, o_h0 = small.n0, small.h0
        o_what = "oracle.solve_tree of the same pattern at %d^3 base cells" % small.n0
    t0 = time.perf_counter()
    _, cref = oracle.solve_tree(o_n0, o_h0, args.theta, o_kinds, o_masses, True, box=o_boxes)
    t_ref = time.perf_counter() - t0
    cnt_ref = cref["m2l"] + cref["p2p"] + cref["cross"]
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sm_count * FP64_LANES_PER_SM * 2 * 1965.0e6 / 1e12
    f_multi = p.octo_fmm_flops_per_interaction_path(p.MULTIPOLE, True, False)[0]   # centre-of-mass expansions: no dipoles
    flops = float(f_multi) * cnt["m2l"] + 8.0 * (cnt["p2p"] + cnt["cross"])
    line = {"metric": METRIC, "value": n_int / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "adaptive-tree solve, %s, theta=%g, correction on" % (what, args.theta),
                       "interactions_per_step": n_int, "pairs": cnt, "leaf_cells_per_level": leaves,
                       "boxes": [list(b) for b in boxes],
                       "leaf_cells_per_s": sum(leaves) / (ms * 1e-3),
                       "l2": "arrays of the fine levels larger than L2", "net_force_over_sum_abs_force": net_force,
                       "host_entry_bit_identical": same},
            "roofline": {"bound": "alu", "kernel": "whole solve (m2l_staged_kernel<.,L2L,TREE> and p2p_monopole_dmma_kernel over tile lists)",
                         "achieved": flops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                         "frac": flops / (ms * 1e-3) / 1e12 / peak, "traffic": None,
                         "note": "useful flops only: %d per multipole pair, 8 per point-mass pair; pairs the kernels mask "
                                 "(two leaves in a brick of the multipole step) are executed but not counted" % f_multi},
            "cpu_baseline": {"value": cnt_ref / t_ref, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": "%s (%d interactions) in %.1f s" % (o_what, cnt_ref, t_ref)},
            "e2e": {"value": n_int / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms},
            "second_rhs": {"ms_per_solve": rhs2_ms, "note": "octo_fmm_tree_solve_rhs2: d(phi)/dt from d(mass)/dt on the same tree "
                                                            "and centres, correction off, dipole terms on; not part of value"},
            "clocks": clocks, "gpu_launches": launches * args.steps}
    print(json.dumps(line))
    t.close()


def run_coupled(args):
    """--coupled: ONE problem sharded over the ranks (z-slabs of a grid of ncell x ncell x (ncell * N) cells, rank r owns
    slab r) with one halo exchange of boundary layers per step (paper_2101_08226_b200/sharded.py).
    Opt-in: the default N > 1 arm runs independent problems.  A step = halo exchange (in place, straight into the
    persistent extended arrays) + staging + interaction."""
    import torch
    import torch.distributed as dist
    world, rank, local = env_int("WORLD_SIZE", 1), env_int("RANK", 0), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log lets the driver count ranks
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2101_08226_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_2101_08226_b200 as p
    from paper_2101_08226_b200.sharded import HALO, PeerShardedLevel, ShardedLevel
    w = make_workload(args.workload, args.theta, args.ncell, args.seed + rank)     # rank r's slab of the tall domain
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    peer = args.halo == "peer"
    if peer:       # no exchange: the kernel reads the neighbours' staged layers through peer memory (CUDA IPC)
        lvl = PeerShardedLevel(w.n, w.h, args.theta, True, rank=rank, world=world, device=local, stream=stream)
        own_m = torch.from_numpy(w.moments).to(dev)
        own_c = torch.from_numpy(w.com_off).to(dev)
    else:
        lvl = ShardedLevel(w.n, w.h, args.theta, True, rank=rank, world=world, device=local, stream=stream)
        own_m, own_c = lvl.moments, lvl.com_off
        own_m.copy_(torch.from_numpy(w.moments))               # the producer writes into the owned views, once
        own_c.copy_(torch.from_numpy(w.com_off))
    lvl.fmm.set_option("dipole_terms", 1)
    L = torch.empty((20,) + lvl.fmm.out_shape, dtype=torch.float64, device=dev)
    Lc = torch.empty((3,) + lvl.fmm.out_shape, dtype=torch.float64, device=dev)
    lvl.fmm.bind_outputs(L, Lc)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if peer:
            lvl.step(own_m, own_c, L, Lc)
        else:
            lvl.step(None, None, L, Lc)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    clocks = sampler.stop(t0, time.perf_counter()) if rank == 0 else None
    if lvl.fmm.status() != p.OK:
        raise SystemExit("bench.py: device reported status %d" % lvl.fmm.status())
    n_int = lvl.interaction_count()
    ms, units = aggregate_over_ranks(ev0.elapsed_time(ev1), n_int * args.steps, dist if world > 1 else None, dev)
    # end to end: the rank's slab from pinned host memory into the owned views, the step, the expansions back
    m_h, c_h = torch.from_numpy(w.moments).pin_memory(), torch.from_numpy(w.com_off).pin_memory()
    L_h = torch.empty(L.shape, dtype=torch.float64).pin_memory()
    e2e_steps = max(args.e2e_steps, 1)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        own_m.copy_(m_h, non_blocking=True)
        own_c.copy_(c_h, non_blocking=True)
        step()
        L_h.copy_(L, non_blocking=True)
        torch.cuda.synchronize()
    barrier()
    e2e_ms_local = 1e3 * (time.perf_counter() - t0)
    e2e_ms, e2e_units = aggregate_over_ranks(e2e_ms_local, n_int * e2e_steps, dist if world > 1 else None, dev)
    if rank == 0:
        flops_per, instr_per = p.octo_fmm_flops_per_interaction(p.MULTIPOLE, True)
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        peak = world * sm_count * FP64_LANES_PER_SM * 2 * 1965.0e6 / 1e12
        achieved = flops_per * units / (ms * 1e-3) / 1e12
        c, s, threads, nr = oracle_sample_bounded(w, args.theta, args.ref_seconds)
        print(json.dumps({"metric": METRIC, "value": units / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": "%s stacked in z: %d x %d x %d cells, theta=%g, correction on" % (
                              w.name, w.n[0], w.n[1], w.n[2] * world, args.theta),
                              "parallelism": ("z-slabs, no exchange: the kernel's TMA loads read the neighbours' staged layers "
                                              "through peer memory (CUDA IPC); two host barriers per step") if peer else (
                                             "z-slabs, one in-place halo exchange per step (%d bytes sent by this rank, "
                                             "%d layers of 23 doubles per cell per neighbour)" % (lvl.halo_bytes_sent, HALO)),
                              "l2": "inputs larger than L2" if w.moments.nbytes > 126e6 else "inputs smaller than L2"},
                          "roofline": {"bound": "alu", "kernel": "m2l_staged_kernel<correction> on every rank (step incl. exchange and staging)",
                                       "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None},
                          "cpu_baseline": {"value": c / s, "unit": UNIT, "cores": threads, "kind": "oracle",
                                           "sample": "%d regions of 16^3 cells (%d interactions) of rank 0's slab in %.1f s" % (nr, c, s)},
                          "e2e": {"value": e2e_units / (e2e_ms * 1e-3), "unit": UNIT,
                                  "h2d_bytes_per_step": int(world * (m_h.numel() + c_h.numel()) * 8),
                                  "d2h_bytes_per_step": int(world * L_h.numel() * 8), "ms_per_step": e2e_ms / e2e_steps},
                          "clocks": clocks, "gpu_launches": 2 * args.steps * world}))
    lvl.close()
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    world = env_int("WORLD_SIZE", 1)
    rank = env_int("RANK", 0)
    local = env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2101_08226_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_2101_08226_b200 as p

    # independent problem per rank (weak scaling): same shape, own seed
    w = make_workload(args.workload, args.theta, args.ncell, args.seed + rank)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    multi = w.com_off is not None          # cfg 4 is the monopole (leaf) variant
    kind = p.MULTIPOLE if multi else p.MONOPOLE
    f = p.OctoFMM(w.n, w.h, args.theta, kind, True, device=local, stream=stream)
    n_int = f.interaction_count()
    info = f.launch_info()
    flops_per, instr_per = p.octo_fmm_flops_per_interaction(kind, True)

    mom = torch.from_numpy(w.moments).to(dev)
    com = torch.from_numpy(w.com_off).to(dev) if multi else None
    ncoef = 20 if multi else 4
    L = torch.empty((ncoef,) + f.out_shape, dtype=torch.float64, device=dev)
    Lc = torch.empty((3,) + f.out_shape, dtype=torch.float64, device=dev) if multi else None

    f.bind_outputs(L, Lc)          # interact() writes the expansions straight into the caller's buffers
    if multi:
        # The headline is the GENERAL path (all 27 dipole terms evaluated) although these
        # centre-of-mass inputs would let the library leave them out; its default path is measured after the timed
        # region and reported beside it as "com_fast_path".
        f.set_option("dipole_terms", 1)

    def step():
        f.set_moments(mom, com)
        f.interact()
        f.get_expansions(L, Lc)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- timed region: device-resident inputs ----
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_begin = time.perf_counter()
    # inputs + outputs smaller than L2 (cfg 4): flush L2 between the timed steps by writing 256 MB, and time every
    # step with its own pair of events so that the flush is not counted
    flush = (mom.numel() + L.numel()) * 8 < 256e6
    l2_scratch = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if flush else None
    sev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ev0.record(stream)
    for i in range(args.steps):
        if flush:
            l2_scratch.fill_(i & 1)
        sev[i][0].record(stream)
        f.set_moments(mom, com)
        kev[i][0].record(stream)
        f.interact()
        kev[i][1].record(stream)
        f.get_expansions(L, Lc)
        sev[i][1].record(stream)
    ev1.record(stream)
    barrier()
    t_end = time.perf_counter()
    clocks = sampler.stop(t_begin, t_end)
    ms_total = sum(a.elapsed_time(b) for a, b in sev) if flush else ev0.elapsed_time(ev1)
    kernel_ms = sum(a.elapsed_time(b) for a, b in kev) / args.steps
    if f.status() != p.OK:
        raise SystemExit("bench.py: device reported status %d" % f.status())
    ms_total, units = aggregate_over_ranks(ms_total, n_int * args.steps, dist if world > 1 else None, dev)
    ms_per_step = ms_total / args.steps
    value = units / (ms_total * 1e-3)

    # ---- end to end through the host-buffer entry point (H2D + step + D2H inside the timed region) ----
    e2e = None
    if args.e2e_steps > 0:
        nb = p.octo_fmm_host_scratch_bytes(f.cfg)
        scratch = torch.empty(nb, dtype=torch.uint8, device=dev)
        mom_h = torch.from_numpy(w.moments).pin_memory()
        com_h = torch.from_numpy(w.com_off).pin_memory() if multi else None
        L_h = torch.empty((ncoef,) + f.out_shape, dtype=torch.float64).pin_memory()
        # the step's result is L (20 coefficients with the correction folded in, BASELINE.json cfg 1); the correction
        # alone (Lcorr) is an optional diagnostic of the API and is not copied back
        Lc_h = None
        p.octo_fmm_run_host(f.handle, mom_h, com_h, L_h, Lc_h, scratch, nb)       # warm-up
        barrier()
        t0 = time.perf_counter()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(args.e2e_steps):
            p.octo_fmm_run_host(f.handle, mom_h, com_h, L_h, Lc_h, scratch, nb)
        b.record(stream)
        barrier()
        e2e_ms = max(a.elapsed_time(b), 1e3 * (time.perf_counter() - t0))
        e2e_ms, e2e_units = aggregate_over_ranks(e2e_ms, n_int * args.e2e_steps, dist if world > 1 else None, dev)
        e2e = {"value": e2e_units / (e2e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(mom_h.numel() * 8 + (com_h.numel() * 8 if multi else 0)),
               "d2h_bytes_per_step": int(L_h.numel() * 8),
               "steps": args.e2e_steps, "ms_per_step": e2e_ms / args.e2e_steps,
               "checksum_L0": float(L_h[0].sum())}
        del scratch, mom_h, com_h, L_h, Lc_h

    # ---- the library's default path on these inputs (dipole terms left out after the device-side check) ----
    fast = None
    if multi:
        f.set_option("dipole_terms", 0)
        f.set_moments(mom, com)
        used = f.dipole_terms_used()
        for _ in range(2):
            f.interact()
        fa, fb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        fa.record(stream)
        for _ in range(3):
            f.interact()
        fb.record(stream)
        torch.cuda.synchronize()
        fast_ms = fa.elapsed_time(fb) / 3
        ff, fi_ = p.octo_fmm_flops_per_interaction_path(kind, True, used)
        fast = {"dipole_terms_evaluated": bool(used), "kernel_ms": fast_ms, "interactions_per_s": n_int / (fast_ms * 1e-3),
                "flops_per_interaction": ff, "fp64_instr_per_interaction": fi_,
                "achieved_tflops": ff * n_int / (fast_ms * 1e-3) / 1e12,
                "note": "every |M1_i| <= 4e-16 |M| h (checked on the device at staging): the 27 dipole terms contribute "
                        "nothing and are not evaluated; results agree with the general path to round-off"}
        f.set_option("dipole_terms", 1)

    # ---- one level of an adaptive mesh (f3): half of the sub-grids are leaves (point masses), seeded; the near-field
    #      pairs with a leaf on either side are taken at this level.  Measured beside the step, not part of `value`. ----
    mixed = None
    if multi and rank == 0 and w.n[0] % 8 == 0:
        g = torch.Generator(device="cpu").manual_seed(args.seed)
        sub = (torch.rand(tuple(v // 8 for v in w.n[::-1]), generator=g) < 0.5).to(dev)
        leaf = sub.repeat_interleave(8, 0).repeat_interleave(8, 1).repeat_interleave(8, 2).to(torch.uint8).contiguous()
        keep = (leaf == 0).to(torch.float64)
        mom_m = mom.clone()
        mom_m[1:] *= keep
        com_m = com * keep
        f.set_moments(mom_m, com_m)
        f.set_option("mixed_count", 1)
        f.interact_mixed(leaf)
        pairs = f.mixed_interaction_count()
        f.set_option("mixed_count", 0)
        ma, mb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ma.record(stream)
        for _ in range(3):
            f.interact_mixed(leaf)
        mb.record(stream)
        torch.cuda.synchronize()
        mixed_ms = ma.elapsed_time(mb) / 3
        mixed = {"leaf_fraction_of_subgrids": float(sub.double().mean()), "kernel_ms": mixed_ms, "interactions": pairs,
                 "near_field_interactions": pairs - n_int, "interactions_per_s": pairs / (mixed_ms * 1e-3),
                 "note": "octo_fmm_interact_mixed: one pass of the slab-fed kernel over the Eq. 15 list + the near field (a pair "
                         "that is not well separated counts if it has a leaf on either side); timed beside the step, not part "
                         "of value"}
        del mom_m, com_m, leaf, keep
        f.set_moments(mom, com)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the interaction kernel), FP64 ALU bound ----
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak_tflops = sm_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    probe_scratch = torch.empty(8 << 20, dtype=torch.uint8, device=dev)
    probe = p.octo_fmm_fp64_peak_probe(local, stream.cuda_stream, probe_scratch, 40000)
    issue_peak = sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    issue_probe = {name: p.octo_fmm_fp64_issue_probe(local, stream.cuda_stream, probe_scratch, mode) / issue_peak
                   for mode, name in ((0, "dfma_three_fresh_registers"), (1, "dfma_operand_reuse"), (2, "dmul"))}
    bytes_per_cell = (23 + 23) * 8 if multi else (1 + 4) * 8      # algorithmic: inputs read once, outputs written once
    achieved = flops_per * n_int / (kernel_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "m2l_staged_kernel<correction>" if multi else "p2p_monopole_dmma_kernel", "achieved": achieved, "peak": peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                "peak_source": "derived: %d SMs x %d FP64 FMA lanes x 2 x %.0f MHz (sm_max_mhz of %s)" % (
                    sm_count, FP64_LANES_PER_SM, sm_max_mhz, "MEASURED_PEAKS.json" if peaks else "nvidia-smi"),
                "peak_measured_dfma": probe["flops_per_s"] / 1e12,
                "frac_of_measured_dfma": achieved / (probe["flops_per_s"] / 1e12),
                "flops_per_interaction": flops_per, "fp64_instr_per_interaction": instr_per,
                "flops_note": "flops_per_interaction = what the kernel executes per pair (counted in its SASS); round 1 executed "
                              "224 for the same formula, so frac_at_round1_operation_count is the figure comparable with r01's 0.607",
                "round1_flops_per_interaction": ROUND1_FLOPS.get(kind),
                "frac_at_round1_operation_count": (ROUND1_FLOPS[kind] * n_int / (kernel_ms * 1e-3) / 1e12 / peak_tflops
                                                   if kind in ROUND1_FLOPS else None),
                "fp64_pipe_issue_frac": (instr_per * n_int / (kernel_ms * 1e-3)) / (sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6),
                "fp64_issue_probe_frac_of_issue_peak": issue_probe,
                "kernel_ms": kernel_ms, "interactions_per_launch": n_int,
                "traffic": traffic_bytes(args.workload, int(w.n[0]), args.theta, p.octo_fmm_version()),
                "kernel_version": p.octo_fmm_version(),
                "algorithmic_bytes": int(bytes_per_cell * w.moments[0].size),
                "hbm_gbs_at_algorithmic_bytes": bytes_per_cell * w.moments[0].size / (kernel_ms * 1e-3) / 1e9,
                "hbm_peak_gbs": peaks.get("hbm_gbs")}

    # ---- the oracle timed beside it on this box's host cores (bounded sample) ----
    c, s, threads, nr = oracle_sample_bounded(w, args.theta, args.ref_seconds)
    cpu_baseline = {"value": c / s, "unit": UNIT, "cores": threads, "kind": "oracle",
                    "sample": "%d regions of 16^3 cells (%d sub-grids, %d interactions) of %s in %.1f s" % (
                        nr, 8 * nr, c, w.name, s)}
    # "(i) single thread, (ii) OpenMP over sub-grids on all cores": the same oracle on ONE thread, on the
    # first regions of the same stratified sample (about a quarter of the time budget)
    import oracle
    oracle.lib().fmm_oracle_set_num_threads(1)
    n1 = max(1, int(nr * (args.ref_seconds / 4.0) / max(s, 1e-9) / max(threads, 1)))
    c1, s1, _, _ = oracle_sample(w, args.theta, min(n1, nr))
    oracle.lib().fmm_oracle_set_num_threads(threads)
    cpu_baseline["single_thread"] = {"value": c1 / s1, "unit": UNIT, "cores": 1,
                                     "sample": "%d regions of 16^3 cells (%d interactions) in %.1f s" % (min(n1, nr), c1, s1)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s theta=%g %s (%d^3 cells, %d sub-grids of 8^3)" % (
                w.name, args.theta, "correction=on" if multi else "monopole", w.n[0], (w.n[0] // 8) ** 3),
                "interactions_per_step": n_int, "l2": ("inputs (%.2f GB) larger than L2" % (mom.numel() * 8 / 1e9)) if mom.numel() * 8 > 126e6 else
                ("inputs + outputs (%.3f GB) vs 126 MB L2; 256 MB scratch written between timed steps" % (
                    (mom.numel() + L.numel()) * 8 / 1e9)),
                "launch": info, "parallelism": "independent problem per GPU" if world > 1 else "single GPU"},
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "clocks": clocks,
            "gpu_launches": 2 * args.steps}
    if fast is not None:
        fast["frac_of_peak"] = fast["achieved_tflops"] / peak_tflops
        line["com_fast_path"] = fast
    if mixed is not None:
        line["mixed_level"] = mixed
    print(json.dumps(line))
    f.close()
    if world > 1:
        dist.destroy_process_group()


def traffic_bytes(workload, ncell, theta, version):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the tracked table
    profiles/traffic.csv (one row per `ncu --set full` capture; the raw export each row comes from is named in it).
    A row counts only if it was captured with THIS build of the kernels (version string of octo_fmm_version()):
    a stale capture yields None, not a wrong number."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(path, newline="") as fh:
            for row in csv.DictReader(r for r in fh if not r.startswith("#")):
                if (row["version"] == version and row["workload"] == workload and int(row["ncell"]) == int(ncell)
                        and abs(float(row["theta"]) - float(theta)) < 1e-12):
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except (OSError, KeyError, ValueError):
        return None
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--theta", type=float, default=0.5)
    ap.add_argument("--ncell", type=int, default=0)
    ap.add_argument("--seed", type=int, default=20210108)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--coupled", action="store_true",
                    help="N > 1: ONE problem in z-slabs with a halo exchange per step instead of independent problems")
    ap.add_argument("--halo", default="exchange", choices=["exchange", "peer"],
                    help="with --coupled: how a rank gets its neighbours' boundary layers")
    ap.add_argument("--ref-seconds", type=float, default=12.0,
                    help="CPU seconds of oracle work per cpu_baseline sample / per --impl reference step")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "solve":
        run_solve(args)
    elif args.workload in ("tree", "tree9"):
        run_tree(args)
    elif args.coupled:
        run_coupled(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
