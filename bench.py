#!/usr/bin/env python
"""bench.py -- throughput of the LOC hot path (one ALI iteration = loc_simulate + loc_solve) on synthetic clouds.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1|C2|C2H|C3|C3H|C4|C5] [--impl reference]

One "step" is one pass of the whole hot path (ray tracing of all directions / rays for all traced transitions, then
the per-cell statistical-equilibrium solve) over one synthetic model.  Prints ONE JSON line (rank 0).
section 8 for the definitions of the metric, the roofline and the CPU baseline.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "ray-cell-channel updates/sec per ALI iteration"
UNIT = "updates/s"
VALUE_KIND = "active updates: channels within 5 sigma of the line centre x traced transitions x ray-cell steps (DESIGN.md 8.1)"
DEFAULT_WORKLOAD = "C5"
CONFIG_ITERATIONS = {"C1": 20, "C2": 50, "C2H": 50, "C3": 10, "C3H": 10, "C4": 10, "C5": 5}  # BASELINE.json configs: ALI iterations of a run

# ---- roofline constants -----------------------------------------------------------------------------
N_SM = 148
# DRAM bytes read + written by one launch of the dominant kernel, from the committed `ncu --set full` captures
# (profiles/r2_summary.md, profiles/r1_sim1d_C2.md); workloads without a capture report null
NCU_TRAFFIC_BYTES = {"C2": (24.3e6, "profiles/r1_sim1d_C2.md"), "C3": (19.08e9 + 7.87e9, "profiles/r2_summary.md"),
                     "C4": (904.1e9 + 298.6e9, "profiles/r2_summary.md"), "C5": (816.6e9 + 142.8e9, "profiles/r2_summary.md")}
FP32_LANES_PER_SM_CLK = 128  # 4 sub-partitions x 1 warp instruction / clk
MUFU_PER_SM_CLK = 16


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


# ---- workloads --------------------------------------------------------------------------------------------------------
def make_workload(name: str):
    """returns (model description, human description).  Seeded synthetic stand-ins for the paper's test models
    (DESIGN.md section 4); the paper's own inputs are not available."""
    import loc_workloads as W
    if name == "C1":
        return W.shell_config(1), "C1: 1D, 64 log shells, 64 rays, 64 channels, 5-level rotor (4 transitions)"
    if name == "C2":
        return W.shell_config(2), "C2: 1D, 1000 log shells, 4000 rays, 256 channels, 10-level rotor (9 transitions)"
    if name == "C2H":  # C2 with a three-component hyperfine structure on J = 1-0 (LTE between the components)
        m = W.shell_config(2)
        m.species.hfs = {0: (np.array([-1.0e5, 0.05e5, 0.7e5]), np.array([0.2, 0.5, 0.3]))}
        m.name = "C2H"
        return m, "C2H: C2 with hyperfine structure on J = 1-0: components at -1.0, +0.05, +0.7 km/s with weights 0.2, 0.5, 0.3"
    if name == "C3H":  # the cost of the masked (hyperfine) path of k_sim3d on record at C3 size
        m = W.cloud_config(3)
        m.species.hfs = {0: (np.array([-1.0e5, 0.05e5, 0.7e5]), np.array([0.2, 0.5, 0.3]))}
        m.name = "C3H"
        return m, "C3H: C3 with hyperfine structure on J = 1-0 (components at -1.0, +0.05, +0.7 km/s, weights 0.2, 0.5, 0.3): every step takes the masked round"
    if name == "C3":
        return W.cloud_config(3), "C3: Cartesian 128^3, 48 directions, 128 channels, 10-level rotor (9 transitions)"
    if name == "C4":
        return W.cloud_config(4), "C4: octree root 64^3 + 3 levels (~30M leaves), 48 directions, 128 channels, 9 transitions"
    if name == "C5":
        return W.cloud_config(5), "C5: octree root 256^3 + 2 levels (~200M leaves), 12 directions, 256 channels, 3 transitions"
    if name.startswith("T"):  # tiny variants for tests of bench.py itself: T3 = 16^3 Cartesian, T4 = small octree
        if name == "T1":
            return W.shell_config(1, ns=32), "T1: 1D test model"
        if name == "T3":
            return W.cloud_config(3, nroot=16, nchannel=64, nside=1), "T3: Cartesian 16^3 test model"
        return W.cloud_config(4, nroot=8, nlev=3, nchannel=64, nside=1), "T4: octree 8^3 + 2 levels test model"
    raise SystemExit(f"unknown workload {name}")


def nominal_updates(steps: int, nch: int, nt: int) -> float:
    return float(steps) * nch * nt


# ---- clocks -----------------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._halt.wait(0.2)

    def stop(self):
        self._halt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        reasons = []
        for i, nm in enumerate(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")):
            if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows):
                reasons.append(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


# ---- CPU oracle sample (cpu_baseline / --impl reference) --------------------------------------------------------------
_KB_OVER_AMU = 1.380649e-16 / 1.66053906660e-24


def _union_count(cc, hw, nch, offs):
    """channels of [0, nch) within hw of any of the centres cc + offs (offs ascending; arrays over steps)"""
    tot = 0.0
    prev_hi = None
    for o in offs:
        lo = np.maximum(0, np.ceil(cc + o - hw))
        hi = np.minimum(nch - 1, np.floor(cc + o + hw))
        if prev_hi is not None:
            lo = np.maximum(lo, prev_hi + 1)
        tot += float(np.maximum(0, hi - lo + 1).sum())
        prev_hi = hi if prev_hi is None else np.maximum(prev_hi, hi)
    return tot


def active_channels_per_cell(m, d=None):
    """the counting rule of the metric: number of channels with |v_c - v_0| <= 5 sigma for one ray
    step through each cell, for propagation direction d (3D) or for mu = 1 (1D: an upper bound is not needed -- the 1D arm
    counts per step, see oracle_sample).  float64 numpy; the library counts the same rule per step in float32."""
    dv = 2.0 * m.band_half / m.nchannel
    sig = np.sqrt(np.asarray(m.sigma, np.float64) ** 2 + (_KB_OVER_AMU / m.species.mass_amu if m.species.mass_amu > 0 else 0.0)
                  * np.asarray(m.tkin, np.float64))
    v0 = -(np.asarray(m.vx, np.float64) * d[0] + np.asarray(m.vy, np.float64) * d[1] + np.asarray(m.vz, np.float64) * d[2])
    cc = v0 / dv + 0.5 * (m.nchannel - 1)
    hw = 5.0 * sig / dv
    return np.maximum(0, np.minimum(m.nchannel - 1, np.floor(cc + hw)) - np.maximum(0, np.ceil(cc - hw)) + 1)


_GEOM_CACHE = {}


def oracle_sample(m, budget_updates=6e9, keep=False):
    """Runs the float64 oracle, as it stands, on a bounded sample of the workload: the ray tracing (all channels) of as
    many transitions of direction 0 as fit the update budget -- or, when even one transition of one direction is more than
    twice the budget (C5), of every k-th line of the root lattice of direction 0 -- plus the solve over all cells.
    Returns a dict: nominal / active updates done, seconds, threads, description (and the oracle's result with keep=True)."""
    import oracle as O
    ncores = os.cpu_count() or 1
    O.set_threads(ncores)
    sp = O.OSpecies(m.species)
    nch = m.nchannel
    dv = 2.0 * m.band_half / nch
    dens, tk, ab = (np.asarray(x, np.float64) for x in (m.density, m.tkin, m.abundance))
    if hasattr(m, "child"):
        allsel = np.arange(sp.ntrans, dtype=np.int32) if getattr(m, "sel", None) is None else np.asarray(m.sel, np.int32)
        key = id(m)
        if key not in _GEOM_CACHE:  # the geometry pass is not part of the timed sample
            _GEOM_CACHE[key] = int(O.sim_3d(sp, m, None, geom_only=True, dirs=m.dirs[0])["visits"].sum())
        steps_dir = _GEOM_CACHE[key]
        per_trans = max(1.0, float(steps_dir) * nch)
        pops = O.lte(sp, dens, tk, ab)
        if per_trans <= 2.0 * budget_updates:
            nt, stride = max(1, min(len(allsel), int(budget_updates // per_trans))), 1
            desc = f"direction 0 of {len(m.dirs)}, transitions {list(map(int, allsel[:nt]))}, all {nch} channels, all cells; then the solve"
        else:
            nt, stride = 1, int(math.ceil(per_trans / budget_updates))
            desc = (f"direction 0 of {len(m.dirs)}, transition {int(allsel[0])}, every {stride}-th line of the root lattice (rays born in "
                    f"refined regions not traced), all {nch} channels; then the solve over all cells")
        sel = allsel[:nt]
        # the solve of the step is sampled in the same proportion as its ray tracing: every k-th cell
        k = max(1, int(round(len(m.dirs) * len(allsel) * stride / nt)))
        desc = desc.replace("then the solve over all cells", "then the solve").replace("then the solve", f"then the solve of every {k}-th cell (the same fraction of the step)")
        t0 = time.perf_counter()
        r = O.sim_3d(sp, m, pops, sel, dirs=m.dirs[0], root_stride=stride)
        ps = np.ascontiguousarray(pops[::k])
        O.solve(sp, dens[::k], tk[::k], ab[::k], r["veff"][::k], sel, np.ascontiguousarray(r["P"][:, ::k]), np.ascontiguousarray(r["LAM"][:, ::k]),
                dv, m.t_bg, ps)
        dt = time.perf_counter() - t0
        steps = int(r["visits"].sum())
        act = float((r["visits"] * active_channels_per_cell(m, m.dirs[0])).sum()) * nt
        threads = ncores  # rays are distributed over OpenMP threads
    else:
        pops = O.lte(sp, dens, tk, ab)
        sel = np.arange(sp.ntrans, dtype=np.int32)
        nt = len(sel)
        nray = len(m.ray_p)
        steps_all = sum(2 * (len(m.r_out) - 1 - int(np.searchsorted(m.r_out, p, side="right"))) + 1 for p in m.ray_p)
        frac = min(1.0, budget_updates / 8 / max(1.0, nominal_updates(steps_all, nch, len(sel))))  # 1D oracle is serial
        if frac < 1.0:
            import copy
            kept = np.arange(0, nray, max(1, int(round(1 / frac))))
            ms = copy.copy(m)
            ms.ray_p, ms.ray_w = m.ray_p[kept], m.ray_w[kept]
        else:
            kept, ms = np.arange(nray), m
        k = max(1, int(round(nray / len(kept))))
        t0 = time.perf_counter()
        r = O.sim_1d(sp, ms, pops, sel)
        ps = np.ascontiguousarray(pops[::k])
        O.solve(sp, dens[::k], tk[::k], ab[::k], r["veff"][::k], sel, np.ascontiguousarray(r["P"][:, ::k]), np.ascontiguousarray(r["LAM"][:, ::k]),
                dv, m.t_bg, ps)
        dt = time.perf_counter() - t0
        steps = int(r["visits"].sum())
        # 1D: the Doppler shift of a step is -v_r mu with the entry cosine of the step (oracle's path table)
        sig = np.sqrt(np.asarray(m.sigma, np.float64) ** 2 + (_KB_OVER_AMU / m.species.mass_amu if m.species.mass_amu > 0 else 0.0)
                      * np.asarray(m.tkin, np.float64))
        vr = np.asarray(m.vrad, np.float64)
        act = 0.0
        hfs = getattr(m.species, "hfs", None) or {}
        for p_ in ms.ray_p:
            sh, _, mu = O.path_1d(m.r_out, float(p_))
            cc = -vr[sh] * mu / dv + 0.5 * (nch - 1)
            hw = 5.0 * sig[sh] / dv
            for t in sel:  # a transition's active channels: within 5 sigma of any of its hyperfine components
                offs = np.sort(np.asarray(hfs[int(t)][0], np.float64) / dv) if int(t) in hfs else np.zeros(1)
                act += _union_count(cc, hw, nch, offs)
        desc = f"{len(kept)} of {nray} rays, all {len(sel)} transitions, all {nch} channels; then the solve of every {k}-th shell (the same fraction of the step)"
        threads = 1  # the 1D ray loop of the oracle is serial
    out = {"nominal": nominal_updates(steps, nch, nt), "active": act, "seconds": dt, "threads": threads, "desc": desc}
    if keep:
        out.update(result=r, sel=sel)
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    m, desc = make_workload(args.workload)
    import oracle as O
    O.build()
    times, last = [], None
    for i in range(args.warmup + args.steps):
        last = oracle_sample(m, budget_updates=args.ref_budget)
        if i >= args.warmup:
            times.append(last["seconds"])
    t = float(np.mean(times))
    val = last["active"] / t
    out = {"impl": "reference", "metric": METRIC, "value": val, "value_kind": VALUE_KIND, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic", "nominal_updates_per_s": last["nominal"] / t,
           "config": {"workload": desc, "sample": last["desc"]},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": last["threads"], "kind": "oracle", "sample": last["desc"]},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ---- multi-process plumbing (replicas only: DESIGN.md section 9) -----------------------------------------------------
def max_over_ranks(values, device="cpu"):
    """max over the ranks of a list of floats (device-timed seconds); identity when torch.distributed is not initialised"""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(updates_per_rank_step: float, steps: int, world: int, seconds: float) -> float:
    """`value` of the JSON line: units all ranks processed / max-over-ranks time (weak scaling: every rank runs a replica)"""
    return world * updates_per_rank_step * steps / seconds


# ---- full-size parity on a direction subset (SURVEY 8d parity protocol (b)) -----------------------------------
def default_parity_dirs(dirs):
    """direction 0 plus the first axis-aligned direction whose main component is negative (zero slopes: the T = 0 branches of
    the lattice arithmetic; mirrored main axis)"""
    d = np.asarray(dirs, np.float64)
    out = [0]
    for i in range(len(d)):
        a = np.abs(d[i])
        k = int(np.argmax(a))
        if d[i, k] < 0 and np.all(np.rint(np.delete(a, k) / a[k] * 2 ** 20) == 0) and i not in out:
            out.append(i)
            break
    return out


def parity_leg(g, m, dirs_idx, ntrans=1, map_patch=0):
    """The oracle traces directions `dirs_idx` of the FULL model for the first `ntrans` traced transitions from LTE
    populations (its own, rounded to float32: the input of both sides); the library does the same with
    loc_set_directions(those directions).  Compared per cell: visit counts and integer path sums bit-exact, SJ within 1e-4
    relative, ESC within 1e-4 of (ESC + 3e-3) -- the rules of tests/parity.py and tests/test_gpu_3d.py.  Leaves the model
    with the subset as its directions (call last)."""
    import oracle as O
    import torch
    O.set_threads(os.cpu_count() or 1)
    sp = O.OSpecies(m.species)
    allsel = np.arange(sp.ntrans, dtype=np.int32) if getattr(m, "sel", None) is None else np.asarray(m.sel, np.int32)
    sel = np.ascontiguousarray(allsel[:ntrans])
    nch = m.nchannel
    dv = 2.0 * m.band_half / nch
    p64 = O.lte(sp, m.density, m.tkin, m.abundance)          # [ncell][NL]
    p32 = np.ascontiguousarray(p64.T.astype(np.float32))     # level-major, float32: the common input
    p64[...] = p32.T
    is3d = hasattr(m, "child")
    leaf = (np.asarray(m.child) < 0) if is3d else np.ones(len(m.density), bool)
    # the library first: all compared transitions in one pass over the direction subset
    if is3d:
        dsub = np.ascontiguousarray(np.asarray(m.dirs, np.float64)[list(dirs_idx)])
        g.set_directions(dsub)
    g.set_populations(p32)
    g.simulate(sel, geometry_counters=True)
    sj, esc = g.counters()
    sj, esc = sj.cpu().numpy(), esc.cpu().numpy()
    vis, pz = g.geometry_counters()
    vis, pz = vis.cpu().numpy().astype(np.int64), pz.cpu().numpy().astype(np.int64)
    # the oracle keeps one donor spectrum [transitions][channels] of float64 per refined cell while it traces a direction
    # (C5: 25.8 M refined cells x 256 channels = 53 GB per transition), so the transitions go through it in groups that keep
    # that store below ~60 GB: one at a time on C5, all at once on the small workloads
    nref = int((~leaf).sum()) if is3d else 0
    per_trans = max(1, nref) * nch * 8
    group = int(max(1, min(len(sel), 60e9 // per_trans)))
    cvel = 2.99792458e10
    worst_sj, worst_esc, t_or, nsteps_ref = 0.0, 0.0, 0.0, 0
    visits_equal, path_equal = True, (True if is3d else None)
    for k0 in range(0, len(sel), group):
        sub = np.ascontiguousarray(sel[k0:k0 + group])
        t0 = time.perf_counter()
        ref = O.sim_3d(sp, m, p64, sub, dirs=dsub) if is3d else O.sim_1d(sp, m, p64, sub)
        t_or += time.perf_counter() - t0
        if k0 == 0:
            nsteps_ref = int(ref["visits"].sum())
            visits_equal = bool(np.array_equal(vis, ref["visits"]))
            if is3d:
                path_equal = bool(np.array_equal(pz, ref["pathz"]))
        for j, t in enumerate(sub):
            k = k0 + j
            sj_o = cvel ** 3 * ref["P"][j] / (8.0 * np.pi * sp.freq(int(t)) ** 3 * dv * ref["veff"])
            esc_o = 1.0 - ref["LAM"][j]
            worst_sj = max(worst_sj, float((np.abs(sj[leaf, k] - sj_o[leaf]) / np.maximum(np.abs(sj_o[leaf]), 1e-300)).max()))
            worst_esc = max(worst_esc, float((np.abs(esc[leaf, k] - esc_o[leaf]) / (np.abs(esc_o[leaf]) + 3e-3)).max()))
        del ref
    del sj, esc, vis, pz
    ok = visits_equal and (path_equal is not False) and worst_sj < 1e-4 and worst_esc < 1e-4
    map_par = None
    if is3d and map_patch > 0:
        # S10 at full size: the cube bench.py times (one pixel per finest cell along +z), computed in full by the
        # library from the same float32 LTE populations; its corner patch (two map edges) against orc_spectra_3d, channel by
        # channel at the tolerance of tests/test_gpu_spectra.py
        nfine, pix = int(m.nx) << (int(m.nlev) - 1), (1 << 20) >> (int(m.nlev) - 1)
        npt = min(int(map_patch), nfine)
        ix0, iy0 = 0, nfine - npt
        zdir = np.array([0.0, 0.0, 1.0])
        tm = int(sel[0])
        cube = g.spectra(tm, nfine, nfine, dir=zdir, aff=np.array([pix // 2, pix // 2, pix, 0, 0, pix], np.int64))
        ta = cube[iy0:iy0 + npt, ix0:ix0 + npt, :].cpu().numpy().astype(np.float64)
        del cube
        t1 = time.perf_counter()
        rm = O.spectra_3d(sp, m, p64, tm, zdir, npt, npt, np.array([pix // 2 + ix0 * pix, pix // 2 + iy0 * pix, pix, 0, 0, pix], np.int64))
        tol = 1e-3 * np.abs(rm) + 2e-5 * np.max(np.abs(rm))
        worst = float(np.max(np.abs(ta - rm) / tol))
        map_par = {"pixels": [npt, npt], "origin": [ix0, iy0], "of_map": [nfine, nfine], "channels": int(nch), "transition": tm,
                   "peak_K": float(np.max(np.abs(rm))), "max_err_over_tol": worst, "tol": "1e-3 |T_A| + 2e-5 max|T_A| per channel",
                   "passed": bool(worst <= 1.0 and np.max(np.abs(rm)) > 0), "oracle_seconds": time.perf_counter() - t1}
        ok = ok and map_par["passed"]
    del p64
    return {"map": map_par, "workload": m.name, "directions": [int(d) for d in dirs_idx] if is3d else None, "transitions": [int(t) for t in sel],
            "cells": int(leaf.sum()), "ray_cell_steps": nsteps_ref, "visits_equal": visits_equal,
            "path_sums_equal": path_equal, "max_rel_sj": worst_sj, "max_esc_err": worst_esc, "tol": 1e-4, "passed": bool(ok),
            "oracle_seconds": t_or, "oracle_transitions_per_pass": group,
            "note": "per-cell counters of the first simulate from LTE; oracle float64, all channels, no cut-off"}


# ---- own arm ------------------------------------------------------------------------------------------------------------
def roofline(stats_geom, nt, t_sim_s, hbm_gbs, sm_mhz, peak_kind):
    """T_roof = max(bytes / HBM, MUFU ops / MUFU rate, FP32 instructions / issue rate) for the simulation
    kernel; `achieved`/`peak` are quoted for the binding resource."""
    steps = stats_geom["steps"]
    u_active = float(stats_geom["active_updates"])
    byt = float(steps) * (8 + 16 + 24 * nt)
    mufu = u_active * (1.0 + 1.0 / nt)
    fp32 = u_active * (8.0 + 4.0 / nt)
    clk = sm_mhz * 1e6
    t_hbm = byt / (hbm_gbs * 1e9)
    t_mufu = mufu / (N_SM * MUFU_PER_SM_CLK * clk)
    t_fp32 = fp32 / (N_SM * FP32_LANES_PER_SM_CLK * clk)
    t_roof = max(t_hbm, t_mufu, t_fp32)
    if t_roof == t_hbm:
        r = {"bound": "hbm", "achieved": byt / t_sim_s / 1e9, "peak": hbm_gbs, "unit": "GB/s"}
    elif t_roof == t_mufu:
        r = {"bound": "alu", "achieved": mufu / t_sim_s / 1e12, "peak": N_SM * MUFU_PER_SM_CLK * clk / 1e12, "unit": "TMUFU/s"}
    else:
        r = {"bound": "alu", "achieved": fp32 / t_sim_s / 1e12, "peak": N_SM * FP32_LANES_PER_SM_CLK * clk / 1e12,
             "unit": "Tinstr/s (FP32-pipe lane instructions)"}
    r["frac"] = t_roof / t_sim_s
    tr = NCU_TRAFFIC_BYTES.get(stats_geom.get("workload"))
    r["traffic"] = tr[0] if tr else None  # not measured in this run: from the committed ncu capture named next
    r["traffic_from_profile"] = tr[1] if tr else None
    r.update({"kernel": "k_sim3d" if stats_geom.get("is3d") else "k_sim1d_w", "peak_source": peak_kind + " HBM copy; ALU peaks derived at sm_max clock",
              "algorithmic_bytes_per_launch": byt, "active_updates_per_launch": u_active, "hbm_gbs_achieved": byt / t_sim_s / 1e9,
              "hbm_frac": t_hbm / t_sim_s, "mufu_frac": t_mufu / t_sim_s, "fp32_frac": t_fp32 / t_sim_s,
              "t_kernel_ms": 1e3 * t_sim_s})
    return r


def run_own(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the LOC library has no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2009_12609_b200 import LocModel

    t_gen = time.perf_counter()
    m, desc = make_workload(args.workload)
    t_gen = time.perf_counter() - t_gen
    is3d = hasattr(m, "child")
    # fingerprint of the realisation (the C4/C5 inputs come from a float32 torch FFT whose rounding depends on the
    # backend): numbers of two runs are on the same model only if this matches
    import hashlib
    hh = hashlib.blake2b(digest_size=8)
    for a in ([m.child] if is3d else [m.r_out]) + [m.density]:
        hh.update(np.ascontiguousarray(a).view(np.uint8).reshape(-1))
    input_hash = hh.hexdigest()
    sel = None if getattr(m, "sel", None) is None else m.sel
    nt = len(m.species.upper) if sel is None else len(sel)
    g = LocModel(m, device=f"cuda:{local}", ntrans_sim=nt)
    for kv in args.option:  # loc_set_option(key, value) for A/B measurements; recorded in config.options
        k, v = kv.split("=")
        g.set_option(int(k), float(v))
    g.init_lte()
    # one untimed pass with the geometry counters: step and active-channel counts of this workload
    g.simulate(sel, geometry_counters=True)
    sg = g.stats()
    sg["is3d"] = is3d
    sg["workload"] = args.workload
    g.init_lte()
    g.simulate(sel)  # remember the selection for loc_iterate
    g.solve()
    g.init_lte()
    steps_per_iter = sg["steps"]
    u_nom = nominal_updates(steps_per_iter, m.nchannel, nt)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        g.iterate(1)
    sampler = ClockSampler(local)
    sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    ev_all = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    l0 = g.stats()["kernel_launches"]
    barrier()
    ev_all[0].record()  # ONE pair around the K steps: the host synchronisation of every loc_solve (its scalar) is inside
    for k in range(args.steps):
        ev[k][0].record()
        g.simulate()
        ev[k][1].record()
        g.solve()
        ev[k][2].record()
    ev_all[1].record()
    barrier()
    clocks = sampler.stop()
    launches = g.stats()["kernel_launches"] - l0
    t_sim = sum(e[0].elapsed_time(e[1]) for e in ev) * 1e-3
    t_solve = sum(e[1].elapsed_time(e[2]) for e in ev) * 1e-3
    t_all = ev_all[0].elapsed_time(ev_all[1]) * 1e-3
    t_all, t_sim, t_solve = max_over_ranks([t_all, t_sim, t_solve], device=f"cuda:{local}")
    u_act = float(sg["active_updates"])
    value = whole_job_value(u_act, args.steps, world, t_all)
    # the same throughput with the one-off path set-up (loc_set_directions) spread over the ALI iterations the config names
    n_cfg = CONFIG_ITERATIONS.get(args.workload, args.steps)
    value_setup = world * u_act * n_cfg / (1e-3 * sg["setup_ms"] + n_cfg * t_all / args.steps)

    # ---- end to end: host buffers -> device -> one ALI iteration -> populations back to the host ----
    names = ["density", "tkin", "sigma", "abundance"] + (["vx", "vy", "vz"] if is3d else ["vx"])
    src = {"density": m.density, "tkin": m.tkin, "sigma": m.sigma, "abundance": m.abundance,
           "vx": m.vx if is3d else m.vrad}
    if is3d:
        src.update(vy=m.vy, vz=m.vz)
    host = {k: torch.from_numpy(np.ascontiguousarray(src[k], np.float32)).pin_memory() for k in names}
    g.init_lte()
    host_pops = g.pops.cpu().pin_memory()
    host_out = torch.empty_like(host_pops).pin_memory()
    h2d = sum(t.numel() * 4 for t in host.values()) + host_pops.numel() * 4
    d2h = host_out.numel() * 4
    from paper_2009_12609_b200 import binding as B

    # the caller's side of the public API, pipelined as a user would: the device-to-host read of step k's result runs on a
    # second stream (its own copy engine) while step k + 1's inputs come in; every step still copies all its inputs from
    # pinned host memory and its result back, and the timed region ends only when the last result has arrived
    side = torch.cuda.Stream(device=local)
    out_dev = torch.empty_like(g.pops)

    def e2e_step():
        g.update_cells(**host)
        g.pops.copy_(host_pops, non_blocking=True)
        B.loc_set_populations(g.h, g.pops)
        g.iterate(1)
        torch.cuda.current_stream().wait_stream(side)  # (the previous result has left out_dev)
        out_dev.copy_(g.pops, non_blocking=True)
        done = torch.cuda.Event()
        done.record()
        side.wait_event(done)
        with torch.cuda.stream(side):
            host_out.copy_(out_dev, non_blocking=True)

    e2e_step()
    torch.cuda.current_stream().wait_stream(side)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(args.steps, 5))
    barrier()
    e0.record()
    for _ in range(n_e2e):
        e2e_step()
    torch.cuda.current_stream().wait_stream(side)  # the last result is on the host before the clock stops
    e1.record()
    barrier()
    (t_e2e,) = max_over_ranks([e0.elapsed_time(e1) * 1e-3], device=f"cuda:{local}")
    e2e_val = whole_job_value(u_act, n_e2e, world, t_e2e)
    del host, host_pops, host_out, out_dev  # 24 GB of pinned memory at C5: returned before the oracle runs
    if hasattr(torch._C, "_host_emptyCache"):
        torch._C._host_emptyCache()  # (torch caches freed pinned blocks; the oracle legs need the host memory)

    # ---- S10: spectral cube of the first traced line along +z, one pixel per finest cell (C5: 1024 x 1024 x
    #      256 channels), and its line-area map; after the iterations above, timed apart from `value` ----
    map_info = None
    if is3d and not args.no_map:
        nfine = int(m.nx) << (int(m.nlev) - 1)
        pix = (1 << 20) >> (int(m.nlev) - 1)
        aff = np.array([pix // 2, pix // 2, pix, 0, 0, pix], np.int64)
        zdir = np.array([0.0, 0.0, 1.0])
        t0 = int(sel[0]) if sel is not None else 0
        cube = g.spectra(t0, nfine, nfine, dir=zdir, aff=aff)
        wmap = g.line_area(cube)
        me = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        nrep = 3
        barrier()
        me[0].record()
        for _ in range(nrep):
            B.loc_spectra(g.h, t0, cube, nfine, nfine, zdir, aff, None)
        me[1].record()
        for _ in range(nrep):
            B.loc_line_area(g.h, cube, nfine * nfine, wmap)
        me[2].record()
        barrier()
        t_map, t_area = max_over_ranks([me[0].elapsed_time(me[1]) * 1e-3 / nrep, me[1].elapsed_time(me[2]) * 1e-3 / nrep],
                                       device=f"cuda:{local}")
        # roofline of k_spectra3d (DESIGN 8.2).  Along +z a pixel of the finest grid crosses every leaf of
        # its column once: steps = sum over leaves of 4^(finest level - level).  Per step and active channel (the 5-sigma rule of
        # the metric) the kernel needs two ex2 (profile, 1 - e^-tau) on the MUFU pipe: 16 per SM and clock.
        lvl = np.asarray(m.level, np.int64)
        leafm = np.asarray(m.child) < 0
        cover = np.left_shift(1, 2 * (int(m.nlev) - 1 - lvl[leafm]))
        act = active_channels_per_cell(m, zdir)[leafm]
        map_steps = int(cover.sum())
        map_active = float((cover * act).sum())
        del lvl, leafm, cover, act
        area_bytes = float(nfine) * nfine * (4 * m.nchannel + 4)
        map_info = {"pixels": [nfine, nfine], "channels": int(m.nchannel), "transition": t0, "ms_spectra": 1e3 * t_map,
                    "ms_line_area": 1e3 * t_area, "line_area_gbs": area_bytes / t_area / 1e9,
                    "cube_bytes": int(cube.numel() * 4), "w_mean_K_kms": float(wmap.mean()),
                    "los_steps": map_steps, "active_updates": map_active}
        del cube, wmap

    parity = None
    if rank == 0 and world == 1 and not args.no_parity:
        import oracle as O
        O.build()
        pdirs = [int(x) for x in args.parity_dirs.split(",")] if args.parity_dirs else (default_parity_dirs(m.dirs) if is3d else [0])
        parity = parity_leg(g, m, pdirs, ntrans=min(args.parity_trans, nt), map_patch=args.parity_map)

    if rank == 0:
        hbm, sm_max, kind = load_peaks()
        if map_info is not None:
            map_info["line_area_hbm_frac"] = map_info["line_area_gbs"] / hbm
            mufu_peak = N_SM * MUFU_PER_SM_CLK * sm_max * 1e6  # ex2 per second
            mufu_ach = 2.0 * map_info["active_updates"] / (1e-3 * map_info["ms_spectra"])
            map_info["roofline"] = {"kernel": "k_spectra3d", "bound": "alu", "resource": "MUFU ex2: 2 per active channel and step",
                                    "achieved": mufu_ach / 1e12, "peak": mufu_peak / 1e12, "unit": "Tex2/s", "frac": mufu_ach / mufu_peak,
                                    "hbm_frac_of_cube_write": map_info["cube_bytes"] / (1e-3 * map_info["ms_spectra"]) / 1e9 / hbm,
                                    "traffic": None}
        roof = roofline(sg, nt, t_sim / args.steps, hbm, sm_max, kind)
        cpu = None
        if world == 1 and not args.no_cpu:
            import oracle as O
            O.build()
            smp = oracle_sample(m, budget_updates=args.ref_budget)
            cpu = {"value": smp["active"] / smp["seconds"], "unit": UNIT, "cores": smp["threads"], "kind": "oracle", "sample": smp["desc"],
                   "seconds": smp["seconds"], "nominal_updates_per_s": smp["nominal"] / smp["seconds"]}
        out = {"metric": METRIC, "value": value, "value_kind": VALUE_KIND, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
               "ms_per_step": 1e3 * t_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f32", "data": "synthetic",
               "config": {"workload": desc, "cells": int(g.ncell), "ray_cell_steps_per_iteration": int(steps_per_iter),
                          "channels": int(m.nchannel), "transitions_traced": int(nt), "parallelism": "replicas" if world > 1 else "single GPU",
                          "updates": "value = active updates (5-sigma rule) / s; nominal = steps x channels x transitions (what a code without a profile cut-off evaluates)",
                          "l2": "inputs larger than L2 (no flush)" if is3d and g.ncell > 1_000_000 else "working set fits L2 (model is small); no flush: the data is re-read from L2 by design",
                          "setup_ms_once": sg["setup_ms"], "input_generation_s": t_gen, "options": args.option,
                          "input_hash": input_hash, "iterations_of_config": n_cfg},
               "value_incl_setup": value_setup,
               "nominal_updates_per_s": whole_job_value(u_nom, args.steps, world, t_all),
               "ms_simulate": 1e3 * t_sim / args.steps, "ms_solve": 1e3 * t_solve / args.steps,
               "clocks": clocks, "roofline": roof,
               "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
               "gpu_launches": int(launches)}
        if cpu is not None:
            out["cpu_baseline"] = cpu
        if map_info is not None:
            out["map"] = map_info
        if parity is not None:
            out["parity"] = parity
        print(json.dumps(out), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()
    if parity is not None and not parity["passed"]:
        raise SystemExit("bench.py: full-size parity against the oracle FAILED: " + json.dumps(parity))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--ref-budget", type=float, default=6e9, help="nominal updates per oracle sample (about 10-30 s of CPU)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-parity", action="store_true", help="skip the full-size parity leg (oracle vs library on a direction subset)")
    ap.add_argument("--parity-dirs", default=None,
                    help="comma-separated direction indices of the parity leg (3D); default: direction 0 plus the first direction "
                         "with zero slopes and a negative main component (axis-aligned, mirrored main axis)")
    ap.add_argument("--parity-trans", type=int, default=3, help="traced transitions compared in the parity leg (at most those traced)")
    ap.add_argument("--parity-map", type=int, default=64, help="edge of the corner patch of the spectral cube compared with the oracle (0 = none)")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=VALUE", help="loc_set_option before the run (A/B measurements)")
    ap.add_argument("--no-map", action="store_true", help="skip the spectral-cube / line-area leg of the 3D workloads")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
