#!/usr/bin/env python
"""bench.py -- one JSON line for the W-VEG sampling hot path on B200 (contract: DESIGN.md section 9).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload all|c1|c2|c3|c4|c5] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input:
gs_preprocess -> gs_build_accel -> gs_sample_fwd (fused MSE) -> gs_sample_bwd.
The headline (`value`, `ms_per_step`, `roofline`, `e2e`, `cpu_baseline`) is the LARGEST single-GPU configuration of
BASELINE.json, configs[4] (C5: 8,388,608 Gaussians, 2^24-point batches of the shell-and-fragments point set, LBVH
rebuilt every step).  With the default `--workload all` the same figures for configs[1] (C2), configs[2] (C3) and
configs[3] (C4, plus its forward-only decode rate) are printed beside it under `workloads`; `--workload cN` times that
configuration alone.  `value` = query points per second (whole job), inputs resident in HBM; `e2e` = the same through
gs_step_host with pinned HOST buffers (H2D/D2H inside the timed region).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TAU = 0.01
HEADLINE = "c5"
# algorithmic FP32-pipe lane-instructions per HIT pair: canonical predicate + weight + accumulate
INSTR_FWD = 19.0
INSTR_BWD = 40.0
# plain-ALU peak: 148 SMs x 128 FP32 lanes x 1.965 GHz (B200_PROFILING.md unit counts / max SM clock)
ALU_PEAK_TINSTR = 148 * 128 * 1.965e9 / 1e12
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")
MIN_TIMED_S = 0.3   # secondary workloads repeat their step until the timed region is at least this long


def _code_only(text: str) -> str:
    """C / CUDA source without comments and blank lines: what the compiler sees."""
    import re
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    text = re.sub(r"//[^\n]*", "", text)
    return "\n".join(ln.rstrip() for ln in text.splitlines() if ln.strip())


def csrc_sha16() -> str:
    """Identity of the kernels this run executes: sha256 over the CODE (comments stripped) of csrc/* and include/gs.h, so
    that a stale ncu capture in profiles/traffic.json reads null and a comment edit does not (the GPU box has no .git)."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2607_01164_b200", "csrc")
    for f in sorted(os.listdir(d)) + ["../../include/gs.h"]:
        with open(os.path.join(d, f), "r", encoding="utf-8", errors="replace") as fh:
            h.update(f.encode() + b"\0" + _code_only(fh.read()).encode())
    return h.hexdigest()[:16]


def load_traffic():
    """dram read + write bytes per launch from an `ncu --set full` capture, valid only for the build they were taken from
    (profiles/traffic.json is written by `bench.py --record-traffic`, keyed by the csrc hash)."""
    try:
        t = json.load(open(TRAFFIC_JSON))
    except (OSError, ValueError):
        return {}, "no profiles/traffic.json"
    if t.get("csrc_sha16") != csrc_sha16():
        return {}, f"profiles/traffic.json is of another build ({t.get('csrc_sha16')} != {csrc_sha16()})"
    return t.get("kernels", {}), t.get("source", "profiles/traffic.json")


def record_traffic(csv_path: str, workload: str, source: str):
    """Parse `ncu -i X.ncu-rep --page raw --csv` (one row per captured launch) and store dram bytes per launch."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    hdr = rows[0]
    ci = {h: i for i, h in enumerate(hdr)}
    units = rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc = {}
    for r in rows[2:]:
        name = r[ci["Kernel Name"]]
        head = name.split("(")[0]
        if any(t in head for t in ("k_grid_fwd<1", "k_grid_fwd<(bool)1", "k_points_fwd<1", "k_points_fwd<(bool)1")):
            continue   # the forward's debug instance (ID sets / counters): launched once outside the timed region
        short = name.split("(")[0].split("::")[-1].split("<")[0].replace("void ", "").strip()
        tot = 0.0
        for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            tot += float(r[ci[m]].replace(",", "")) * scale[units[ci[m]]]
        acc.setdefault(short, []).append(tot)
    try:
        t = json.load(open(TRAFFIC_JSON))
    except (OSError, ValueError):
        t = {}
    if t.get("csrc_sha16") != csrc_sha16():
        t = {"csrc_sha16": csrc_sha16(), "kernels": {}, "source": source}
    for k, v in acc.items():
        t["kernels"][f"{workload}/{k}"] = {"bytes": sum(v) / len(v), "launches": len(v), "source": source}
    json.dump(t, open(TRAFFIC_JSON, "w"), indent=1, sort_keys=True)
    print(json.dumps(t, indent=1))


# ------------------------------------------------------------------------------------------------------------------
# workloads (BASELINE.json configs; the recipes are in DESIGN.md section 4)
# ------------------------------------------------------------------------------------------------------------------
def make_workload(name: str):
    from paper_2607_01164_b200 import inputs
    if name == "c1":
        grid = inputs.c1_grid(32)
        g = inputs.c1_gaussians(seed=0, n=1024)
        rng = np.random.default_rng(1)
        return dict(name=name, kind="grid", g=g, grid=grid, target=rng.uniform(0, 1, grid.num_points).astype(np.float32), domain=None,
                    desc="C1 tiny structured 32^3, 1024 Gaussians (BASELINE.json configs[0])")
    if name == "c2":
        grid = inputs.c2_grid(256)
        g = inputs.c2_gaussians(seed=2, n_grid=256, n=262144)
        return dict(name=name, kind="grid", g=g, grid=grid, target=inputs.c2_target(grid), domain=None,
                    desc="C2 structured 256^3 Marschner-Lobb, 262144 Gaussians, whole grid per step (BASELINE.json configs[1])")
    if name == "c3":
        xyz_all, t_all = inputs.c3_points(seed=3, p=2_000_000)
        g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=1_048_576)
        batches = []
        for b in range(4):   # a fresh batch (without replacement) per step, cycling through 4 resident ones
            idx = inputs.batch_indices(3, b, len(xyz_all), 1 << 20)
            batches.append((np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])))
        return dict(name=name, kind="points", g=g, batches=batches, domain=inputs.points_domain(xyz_all),
                    desc="C3 unstructured, 2^20-point batches (4 distinct, one per step) of 2M mixture points, 1048576 Gaussians, "
                         "LBVH rebuilt per step (BASELINE.json configs[2])")
    if name == "c4":
        field = inputs.c4_field(seed=4)
        g = inputs.c4_gaussians(seed=4, n_grid=1024, n=4_194_304, field=field)
        full = inputs.c4_grid(1024)
        grid = full.batch((48, 48, 48), (16, 16, 16))
        return dict(name=name, kind="grid", g=g, grid=grid, full=full, target=inputs.c4_target(grid, field), domain=None,
                    decode_blocks=[(16 * x, 16 * y, 16 * z) for z in range(4) for y in range(4) for x in range(4)],
                    desc="C4 structured 1024^3 turbulence field, 4194304 Gaussians (5% 20:1 needles), one 128^3 brick-aligned batch "
                         "per step (BASELINE.json configs[3])")
    if name == "c5":
        xyz_all, t_all = inputs.c5_points(seed=5)   # the whole 200,000,000-point set (2.4 GB of positions; drawn by a thread pool)
        g = inputs.c5_gaussians(xyz_all, t_all)
        batches = []
        for b in range(2):
            idx = inputs.batch_indices(5, b, len(xyz_all), 1 << 24)
            batches.append((np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])))
        return dict(name=name, kind="points", g=g, batches=batches, domain=inputs.points_domain(xyz_all), decode_xyz=xyz_all,
                    desc="C5 unstructured shell-and-fragments, 2^24-point batches (2 distinct, alternating) drawn without replacement from the "
                         "200,000,000-point set, 8388608 Gaussians centred on points of that set, LBVH rebuilt per step (BASELINE.json configs[4])")
    raise SystemExit(f"unknown workload {name}")


def shard_workload(wl, rank: int, world: int):
    """This rank's share of every batch of the workload (host arrays; no GPU needed): a z-slab of the grid's bricks
    (dist.shard_bricks) or a contiguous slice of each point batch (dist.shard_points).  Returns ([{grid | xyz, target}],
    P_total); the list is empty for a rank whose slab is empty.  Every rank holds the SAME model."""
    from paper_2607_01164_b200 import dist as gsdist
    if wl["kind"] == "grid":
        grid = wl["grid"]
        P_total = grid.num_points
        lo, cnt = gsdist.shard_bricks(grid.brick_cnt, rank, world)
        if cnt[2] <= 0:
            return [], P_total
        sub = grid.batch(tuple(a + b for a, b in zip(grid.brick_lo, lo)), cnt)
        bd = grid.batch_dims
        z0 = 8 * lo[2]
        t = np.asarray(wl["target"]).reshape(bd[2], bd[1], bd[0])[z0:z0 + sub.batch_dims[2]]
        return [dict(grid=sub, target=np.ascontiguousarray(t).ravel())], P_total
    P_total = len(wl["batches"][0][0])
    a, b = gsdist.shard_points(P_total, rank, world)
    return [dict(xyz=np.ascontiguousarray(x[a:b]), target=np.ascontiguousarray(t[a:b])) for x, t in wl["batches"]], P_total


# point queries: which acceleration mode each configuration runs in by default (the measured winner)
POINTS_MODE_DEFAULT = {"c3": "gather", "c5": "gather"}


def points_mode(wl, args):
    if wl["kind"] != "points":
        return None
    return POINTS_MODE_DEFAULT.get(wl["name"], "gather") if args.points_accel == "default" else args.points_accel


def config_of(wl) -> dict:
    """The `config` object: identical in the `ours` and the `reference` arm (no measured quantity in it)."""
    P = wl["grid"].num_points if wl["kind"] == "grid" else len(wl["batches"][0][0])
    return {"workload": wl["desc"], "points_per_step": int(P), "gaussians": int(wl["g"].n),
            "step": "preprocess+build_accel+fwd(MSE)+bwd",
            "l2": "per-step working set (records, lists, per-sample arrays) exceeds the 126 MB L2 for C2-C5; no flush"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe), one sample per 20 ms."""

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20", "-i",
                                          str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def wait_first(self, timeout: float = 5.0):
        """nvidia-smi takes a moment to attach to the driver: let that happen outside the timed region."""
        t0 = time.time()
        while self.proc and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.02)

    def window(self, w0, w1):
        """Clock record of the host-time window (w0, w1) of a timed region."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        rows = [r for t, r in self.rows if len(r) >= 7 and w0 <= t <= w1 + 0.05]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in the window"], "samples": 0}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows)}

    def stop(self):
        if self.proc:
            self.proc.terminate()


# ------------------------------------------------------------------------------------------------------------------
# the oracle on a bounded sample of a workload (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------------------------
def oracle_sample(wl):
    """(xyz, target, note): the bounded sample of the workload the oracle is timed on (whole grid for C1/C2,
    one 128^3 batch for C4, the first 2^17 / 2^20 points of a batch for C3 / C5; always against the whole model)."""
    from oracle import wveg_oracle as oracle
    g = wl["g"]
    if wl["kind"] == "grid":
        grid = wl["grid"]
        bd = grid.batch_dims
        return oracle.grid_points(grid), wl["target"], f"the step's whole {bd[0]}x{bd[1]}x{bd[2]} batch, all {g.n} Gaussians, fwd+MSE+bwd"
    n = {"c3": 1 << 17, "c5": 1 << 20}.get(wl["name"], 1 << 15)
    xyz, t = wl["batches"][0]
    n = min(n, len(xyz))
    return xyz[:n], t[:n], f"first {n} points of a batch, all {g.n} Gaussians, fwd+MSE+bwd"


def oracle_step(wl, xyz, target):
    from oracle import wveg_oracle as oracle
    g = wl["g"]
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    return len(xyz)


def run_reference(args):
    """The oracle, as it stands, on the box's host cores: every step is the cpu_baseline sample of the headline workload."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import wveg_oracle as oracle
    oracle.build()
    name = HEADLINE if args.workload == "all" else args.workload
    wl = make_workload(name)
    xyz, target, note = oracle_sample(wl)
    for _ in range(min(args.warmup, 1)):   # the oracle has no caches to warm beyond the page cache: one pass at most
        oracle_step(wl, xyz, target)
    t0 = time.perf_counter()
    pts = 0
    for _ in range(args.steps):
        pts += oracle_step(wl, xyz, target)
    dt = time.perf_counter() - t0
    val = pts / dt
    line = {"impl": "reference", "metric": "query_points_per_s_fwd_bwd", "value": val, "unit": "points/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_of(wl),
            "cpu_baseline": {"value": val, "unit": "points/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": note},
            "e2e": {"value": val, "unit": "points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------------------
def measure(wl, args, sampler, world, rank, headline: bool):
    """Times one workload: K steps (device-resident), the e2e leg through gs_step_host, decode legs where the config has
    one.  Returns the workload's result dict."""
    import torch
    import torch.distributed as dist
    from paper_2607_01164_b200 import api, dist as gsdist

    g = wl["g"]
    ctx = api.Context()
    mode = points_mode(wl, args)
    if mode is not None:
        ctx.gs_set_option(api.OPT_POINTS_ACCEL, api.POINTS_SCATTER if mode == "scatter" else api.POINTS_GATHER)
    if args.no_hit_masks:
        ctx.gs_set_option(api.OPT_BWD_HIT_MASKS, 0)   # A/B: the point backward evaluates every cull-list entry (gs.h)
    if wl["kind"] == "grid" and not args.sync_build:
        ctx.gs_set_option(api.OPT_ASYNC_BUILD, 1)   # steady-state builds without a host round trip (gs.h)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    gd = [dev(a) for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    # ---- this rank's share of the samples: same model everywhere, bricks / points are sharded
    shards, P_total = shard_workload(wl, rank, world)
    keep = [dev(s_["xyz"]) if wl["kind"] == "points" else None for s_ in shards]
    queries = [api.grid_query(s_["grid"]) if wl["kind"] == "grid" else api.points_query(x) for s_, x in zip(shards, keep)]
    tgt = [dev(s_["target"]) for s_ in shards]
    P = api.query_num_points(queries[0]) if queries else 0
    phi = torch.empty(max(P, 1), device="cuda")
    I = torch.empty(max(P, 1), device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    grads = ctx.alloc_grads(g.n, flat=True)
    if world > 1:
        ctx.gs_set_sample_count(P_total)   # the loss mean runs over the samples of ALL ranks

    it = [0]

    def step():
        k = it[0] % max(len(queries), 1)
        it[0] += 1
        loss.zero_()
        ctx.gs_preprocess(*gd, domain=wl["domain"], tau=TAU)
        if queries:
            q = queries[k]
            ctx.gs_build_accel(q)
            ctx.gs_sample_fwd(q, phi, I, target=tgt[k], loss=loss)  # fused MSE: keeps the backward coefficients
            ctx.gs_sample_bwd(q, None, None, None, grads)           # dL_dphi = NULL: backward of that fused loss
        else:
            for v in grads.values():
                v.zero_()
        if world > 1:
            gsdist.allreduce_grads(grads, loss)   # ONE collective on the flat gradient buffer (+ the loss scalar)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    barrier()
    # hit / tested pair counts of this workload (outside the timed region; first batch)
    tested = hits = 0
    if queries:
        ctx.gs_build_accel(queries[0])
        _, _, _, tested, hits = ctx.debug_point_sets(queries[0])
    ctx.profile_read()
    ctx.profile_enable(True)
    for _ in range(2):
        step()
    barrier()
    ctx.profile_read()
    # K steps exactly for the headline; a secondary workload repeats until its timed region is long enough for clock samples
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); step(); e1.record(); barrier()
    est_ms = max(e0.elapsed_time(e1), 1e-3)
    steps = args.steps if headline else max(args.steps, int(math.ceil(1e3 * MIN_TIMED_S / est_ms)))
    ctx.profile_read()
    w0 = time.time()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    barrier()
    w1 = time.time()
    ms_total = e0.elapsed_time(e1)
    stage_ms, stage_calls, launches = ctx.profile_read()
    ctx.profile_enable(False)
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / steps
    out = {"config": config_of(wl), "points_accel": mode, "async_build": bool(wl["kind"] == "grid" and not args.sync_build), "steps": steps, "ms_per_step": ms_step, "value": P_total / (ms_step * 1e-3), "unit": "points/s",
           "gpu_launches": launches, "clocks": sampler.window(w0, w1) if rank == 0 else None,
           "hit_pairs": hits, "tested_pairs": tested, "cull_efficiency": hits / tested if tested else None}
    per = {k: (stage_ms[k] / stage_calls[k] if stage_calls[k] else 0.0) for k in stage_ms}
    out["stage_ms"] = per
    # ---- roofline of the sampling kernels (this rank's share of the work): per kernel (a) the algorithmic FP32-pipe
    #      lane-instructions of its HIT pairs at the ALU issue peak and (b) its compulsory bytes at the measured HBM copy bandwidth;
    #      the larger of the two times is the bound, frac = that time / the measured launch time
    traffic, tsrc = load_traffic()
    pts = wl["kind"] == "points"
    kpre = "k_points_" if pts else "k_grid_"
    hbm_gbs = _peaks().get("hbm_gbs") or 6547.0
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if _peaks().get("hbm_gbs") else "fallback 6547 GB/s (B200_PROFILING.md)"
    alu_peak = ALU_PEAK_TINSTR   # replaced by the FFMA rate measured in this run for the headline (see below)
    # Gaussians whose record a launch must read: the whole model for a point batch, the Gaussians that overlap the batch for a grid one
    Ng = g.n if pts else int(ctx.gs_status_query().get("grid_touched", g.n))
    # compulsory bytes per launch, term by term
    recipe = {
        "fwd": {"per_point": (4 + 8) + ((12 + 4) if pts else 0), "per_gaussian": 64,
                "terms": "per point: 4 B target + 8 B (Phi, I) written" + (" + 12 B xyz + 4 B order" if pts else "") + "; per Gaussian: 64 B record"
                         + ("" if pts else "; + 4 B per (brick, Gaussian) list entry")},
        "bwd": {"per_point": 16 + ((12 + 4) if pts else 0), "per_gaussian": 64 + 2 * 48,
                "terms": "per point: 16 B (Phi, I, dL/dPhi, dL/dI or the packed coefficients)" + (" + 12 B xyz + 4 B order" if pts else "")
                         + "; per Gaussian: 64 B record + 48 B accumulator row read and written"
                         + ("" if pts else "; + 4 B per (brick, Gaussian) list entry")},
        "cull": {"per_point": 16, "per_gaussian": 128,
                 "terms": "per point: 16 B of the sorted copy; per Gaussian: 64 B traversal node + 64 B record (the lists themselves are scratch, not compulsory)"},
    }
    list_bytes = 0 if pts else 4 * int(ctx.gs_status_query().get("grid_pairs", 0))
    kernels = {}
    names = (("fwd", INSTR_FWD), ("bwd", INSTR_BWD)) + ((("cull", None),) if pts and per.get("cull", 0.0) > 0 else ())
    for nm, instr in names:
        ms = per[nm]
        rb = recipe[nm]
        nbytes = P * rb["per_point"] + Ng * rb["per_gaussian"] + (list_bytes if nm != "cull" else 0)
        alu_ms = hits * instr / (alu_peak * 1e12) * 1e3 if instr else None
        hbm_ms = nbytes / (hbm_gbs * 1e9) * 1e3
        bound = "alu" if (alu_ms is not None and alu_ms >= hbm_ms) else "hbm"
        bound_ms = alu_ms if bound == "alu" else hbm_ms
        ach = hits * instr / (ms * 1e-3) / 1e12 if (ms > 0 and instr) else None
        kname = kpre + nm + ("_masked" if (pts and nm == "bwd" and not args.no_hit_masks and mode != "scatter") else "")
        tr = traffic.get(f"{wl['name']}/{kname}")
        # the ALU figure over the pairs the kernel actually EVALUATES (how busy the pipes are; frac_alu / issue_frac = cull efficiency)
        # (not for a backward that drops the entries without a hit, GS_OPT_BWD_HIT_MASKS: it evaluates fewer pairs than `tested`)
        issue = tested * instr / (ms * 1e-3) / 1e12 / alu_peak if (ms > 0 and pts and instr and (nm == "fwd" or args.no_hit_masks)) else None
        kernels[nm] = {"kernel": kname, "launch_ms": ms, "alu_ms": alu_ms, "hbm_ms": hbm_ms, "bound": bound,
                       "frac": bound_ms / ms if ms > 0 else None, "frac_alu": (alu_ms / ms if (ms > 0 and alu_ms is not None) else None),
                       "frac_hbm": hbm_ms / ms if ms > 0 else None, "achieved": ach, "achieved_gbs": nbytes / (ms * 1e-3) / 1e9 if ms > 0 else None,
                       "issue_frac": issue, "algorithmic_lane_instr": hits * instr if instr else None, "algorithmic_bytes": nbytes,
                       "bytes_recipe": rb["terms"], "traffic": tr["bytes"] if tr else None, "traffic_source": tr["source"] if tr else tsrc}
    dom = "fwd" if per["fwd"] >= per["bwd"] else "bwd"
    kd = kernels[dom]
    fb_ms = per["fwd"] + per["bwd_pack"] + per["bwd"]
    samp_ms = fb_ms + (per.get("cull", 0.0) if pts else 0.0)
    both_alu_ms = hits * (INSTR_FWD + INSTR_BWD) / (alu_peak * 1e12) * 1e3
    both_hbm_ms = kernels["fwd"]["hbm_ms"] + kernels["bwd"]["hbm_ms"]
    both_ms = max(both_alu_ms, both_hbm_ms)
    out["roofline"] = {
        "bound": kd["bound"], "kernel": kd["kernel"],
        "achieved": kd["achieved"] if kd["bound"] == "alu" else kd["achieved_gbs"],
        "peak": alu_peak if kd["bound"] == "alu" else hbm_gbs,
        "unit": "T FP32 lane-instr/s (algorithmic: hit pairs x 19 fwd / x 40 bwd)" if kd["bound"] == "alu" else "GB/s",
        "frac": kd["frac"], "traffic": kd["traffic"], "traffic_unit": "bytes per launch (dram read + write, ncu --set full)",
        "traffic_source": kd["traffic_source"], "launch_ms": kd["launch_ms"], "kernels": kernels,
        "fwd_bwd_frac": both_ms / fb_ms if fb_ms > 0 else None,
        "sampling_frac": both_ms / samp_ms if samp_ms > 0 else None,   # cull + fwd + bwd: the traversal is half of S5
        "step_frac": both_ms / ms_step,
        "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src, "alu_peak_nominal": ALU_PEAK_TINSTR,
        "peak_source": "148 SM x 128 lanes x 1.965 GHz (B200_PROFILING.md unit counts and max SM clock)"}
    out["rates"] = {"fwd_points_per_s": P / (per["fwd"] * 1e-3) if per["fwd"] else None,
                    "fwd_gaussian_evals_per_s": hits / (per["fwd"] * 1e-3) if per["fwd"] else None,
                    "fwd_bwd_gaussian_evals_per_s": hits / (ms_step * 1e-3)}

    # ---- forward-only decode legs (configs[3]: 64 consecutive 128^3 batches; configs[4]: the 40M draw in 2^24 chunks)
    if world == 1 and wl.get("decode_blocks"):
        blocks = wl["decode_blocks"]
        qs = [api.grid_query(wl["full"].batch(lo, (16, 16, 16))) for lo in blocks]
        Pb = api.query_num_points(qs[0])
        phis = torch.empty(len(qs) * Pb, device="cuda")   # every batch writes its own output: real HBM writes, not L2 hits
        Is = torch.empty(len(qs) * Pb, device="cuda")
        ctx.gs_preprocess(*gd, tau=TAU)

        views = [(q, phis[k * Pb:(k + 1) * Pb], Is[k * Pb:(k + 1) * Pb]) for k, q in enumerate(qs)]

        def decode():
            for q, p_, i_ in views:
                ctx.gs_build_accel(q)
                ctx.gs_sample_fwd(q, p_, i_)
        decode(); barrier()
        reps = max(1, int(math.ceil(1e3 * MIN_TIMED_S / (0.2 * len(qs)))))
        ctx.profile_read(); ctx.profile_enable(True)
        e0.record()
        for _ in range(reps):
            decode()
        e1.record(); barrier()
        sm, sc, _ = ctx.profile_read(); ctx.profile_enable(False)
        ms_b = e0.elapsed_time(e1) / (reps * len(qs))
        fwd_ms = sm["fwd"] / max(sc["fwd"], 1)
        peaks = _peaks()
        hbm = peaks.get("hbm_gbs")
        out["decode"] = {"what": f"forward-only decode of {len(qs)} consecutive 128^3 batches (a 512^3 block), one gs_preprocess, "
                                 "gs_build_accel + gs_sample_fwd per batch, each batch writing its own Phi/I",
                         "batches": len(qs), "ms_per_batch": ms_b, "points_per_s": Pb / (ms_b * 1e-3),
                         "build_ms": sm["build"] / max(sc["build"], 1), "fwd_ms": fwd_ms,
                         "roofline": {"bound": "hbm", "kernel": "k_grid_fwd", "unit": "GB/s",
                                      "achieved": Pb * 8 / (fwd_ms * 1e-3) / 1e9 if fwd_ms else None, "peak": hbm,
                                      "frac": (Pb * 8 / (fwd_ms * 1e-3) / 1e9 / hbm) if (fwd_ms and hbm) else None,
                                      "algorithmic_bytes": "8 B written per sample (Phi, I); records and lists are L2-resident",
                                      "peak_source": "MEASURED_PEAKS.json hbm_gbs (burst copy)"}}
        # the same 512^3 block as ONE batch (brick-aligned batches may span up to 2048 voxels per axis): the per-batch figure above is
        # bound by the launch and tail latencies of ~6 small kernels per 128^3 batch, not by arithmetic or bandwidth
        lo0 = blocks[0]
        qb = api.grid_query(wl["full"].batch(lo0, (64, 64, 64)))
        Pbig = api.query_num_points(qb)
        if Pbig == len(qs) * Pb:
            ctx.gs_set_option(api.OPT_ASYNC_BUILD, 0)   # 64x the pairs of the batches before: size the pair list synchronously
            ctx.gs_build_accel(qb); ctx.gs_sample_fwd(qb, phis, Is); barrier()
            if not args.sync_build:
                ctx.gs_set_option(api.OPT_ASYNC_BUILD, 1)
            repb = 5
            ctx.profile_read(); ctx.profile_enable(True)
            e0.record()
            for _ in range(repb):
                ctx.gs_build_accel(qb)
                ctx.gs_sample_fwd(qb, phis, Is)
            e1.record(); barrier()
            smb, scb, _ = ctx.profile_read(); ctx.profile_enable(False)
            ms_big = e0.elapsed_time(e1) / repb
            fwd_big = smb["fwd"] / max(scb["fwd"], 1)
            out["decode"]["one_batch_512"] = {
                "what": "the same 512^3 block decoded as ONE brick-aligned batch (gs_build_accel + gs_sample_fwd)",
                "ms": ms_big, "points_per_s": Pbig / (ms_big * 1e-3), "build_ms": smb["build"] / max(scb["build"], 1), "fwd_ms": fwd_big,
                "fwd_hbm_frac": (Pbig * 8 / (fwd_big * 1e-3) / 1e9 / hbm) if (fwd_big and hbm) else None}
        # gs_decode_grid: the library's own batch decode -- the same batches dealt to worker contexts on their own streams, so that
        # the build of one batch runs beside the forward of another.  First the 512^3 block (output compared with the loop above),
        # then the FULL 1024^3 grid of configs[3] (512 batches of 128^3, 1.07e9 samples, 8.6 GB of output).
        chk = float(phis.double().sum().item())
        region = wl["full"].batch(blocks[0], (64, 64, 64))
        phis.zero_()
        ctx.gs_decode_grid(*gd, api.grid_query(region), (16, 16, 16), phis, Is, streams=4, tau=TAU)
        same = float(phis.double().sum().item()) == chk
        del phis, Is
        full_q = api.grid_query(wl["full"])
        Pfull = api.query_num_points(full_q)
        phif, If = torch.empty(Pfull, device="cuda"), torch.empty(Pfull, device="cuda")
        sweep = []
        for nstr in (1, 2, 4, 8):
            ctx.gs_decode_grid(*gd, full_q, (16, 16, 16), phif, If, streams=nstr, tau=TAU)   # warm: worker contexts, buffers
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.gs_decode_grid(*gd, full_q, (16, 16, 16), phif, If, streams=nstr, tau=TAU)   # returns when the decode is complete
            dt = time.perf_counter() - t0
            sweep.append({"streams": nstr, "ms_total": 1e3 * dt, "ms_per_batch": 1e3 * dt / 512, "points_per_s": Pfull / dt,
                          "hbm_write_frac": (Pfull * 8 / dt / 1e9 / hbm) if hbm else None})
        best = max(sweep, key=lambda r: r["points_per_s"])
        out["decode"]["full_grid"] = {"what": "gs_decode_grid over the whole 1024^3 grid of configs[3]: 512 batches of 128^3, forward only, host "
                                              "wall clock around the (synchronous) call, including the workers' gs_preprocess of the model",
                                      "points": Pfull, "best": best, "sweep": sweep, "block_512_same_output_as_one_context": same,
                                      "covered_fraction": float((If > TAU).float().mean().item())}
        del phif, If
    if world == 1 and wl.get("decode_xyz") is not None:
        allx = wl["decode_xyz"]
        chunk = 1 << 24
        # end to end first (it needs two chunk buffers only): the set stays in HOST memory, chunk k+1 is copied in on a copy
        # stream while chunk k is built and sampled, Phi / I of every chunk go back to the host
        e2e_decode = None
        if len(allx) > chunk:
            nck = (len(allx) + chunk - 1) // chunk
            cs = torch.cuda.Stream()
            xb = [torch.empty((chunk, 3), device="cuda") for _ in range(2)]
            pb = [torch.empty(chunk, device="cuda") for _ in range(2)]
            ib = [torch.empty(chunk, device="cuda") for _ in range(2)]
            hx = torch.from_numpy(allx)   # pageable host memory is pinned chunk by chunk (cudaHostRegister on 2.4 GB takes seconds)
            hx_pin = [torch.empty((chunk, 3), pin_memory=True) for _ in range(2)]
            hphi = torch.empty(len(allx), pin_memory=True)
            hI = torch.empty(len(allx), pin_memory=True)
            ready = [torch.cuda.Event() for _ in range(2)]
            freed = [torch.cuda.Event() for _ in range(2)]
            main = torch.cuda.current_stream()

            def stage(k):
                a = k * chunk
                n_ = min(chunk, len(allx) - a)
                hx_pin[k % 2][:n_].copy_(hx[a:a + n_])          # host memcpy into the pinned staging buffer
                with torch.cuda.stream(cs):
                    cs.wait_event(freed[k % 2])
                    xb[k % 2][:n_].copy_(hx_pin[k % 2][:n_], non_blocking=True)
                    ready[k % 2].record(cs)
                return n_

            def decode_e2e():
                ctx.gs_preprocess(*gd, domain=wl["domain"], tau=TAU)
                for e in freed:
                    e.record(main)
                n_next = stage(0)
                for k in range(nck):
                    n_ = n_next
                    main.wait_event(ready[k % 2])
                    q_ = api.points_query(xb[k % 2][:n_])
                    ctx.gs_build_accel(q_)
                    ctx.gs_sample_fwd(q_, pb[k % 2][:n_], ib[k % 2][:n_])
                    a = k * chunk
                    hphi[a:a + n_].copy_(pb[k % 2][:n_], non_blocking=True)
                    hI[a:a + n_].copy_(ib[k % 2][:n_], non_blocking=True)
                    freed[k % 2].record(main)
                    if k + 1 < nck:
                        n_next = stage(k + 1)   # the pinned staging buffer of chunk k+1 was last read by the copy of chunk k-1: done (build synchronised)
                torch.cuda.synchronize()

            decode_e2e()
            t0 = time.perf_counter(); decode_e2e(); dt_e2e = time.perf_counter() - t0
            e2e_decode = {"ms_total": 1e3 * dt_e2e, "points_per_s": len(allx) / dt_e2e, "h2d_bytes": int(allx.nbytes), "d2h_bytes": int(8 * len(allx)),
                          "what": "the same decode with the point set in host memory: per chunk a host copy into a pinned staging buffer, H2D on a copy "
                                  "stream overlapped with the previous chunk's build + forward, D2H of Phi / I; host wall clock, one gs_preprocess inside"}
            del xb, pb, ib, hx_pin, hphi, hI
        xs = [dev(allx[a:a + chunk]) for a in range(0, len(allx), chunk)]
        qs = [api.points_query(x) for x in xs]
        pp = [torch.empty(len(x), device="cuda") for x in xs]
        ii = [torch.empty(len(x), device="cuda") for x in xs]
        def decode():   # from scratch: gs_preprocess, then per chunk gs_build_accel (the first one builds the LBVH, the others reuse it) + forward
            ctx.gs_preprocess(*gd, domain=wl["domain"], tau=TAU)
            for q, p_, i_ in zip(qs, pp, ii):
                ctx.gs_build_accel(q)
                ctx.gs_sample_fwd(q, p_, i_)
        decode(); barrier()
        ctx.profile_read(); ctx.profile_enable(True)
        e0.record(); decode(); decode(); e1.record(); barrier()
        sm, sc, _ = ctx.profile_read(); ctx.profile_enable(False)
        ms_all = e0.elapsed_time(e1) / 2
        out["decode"] = {"end_to_end": e2e_decode,
                         "what": f"forward-only decode of ALL {len(allx)} points of the set in {len(qs)} chunks of <= 2^24 points (device-resident): one gs_preprocess "
                                 "(inside the timed region), then gs_build_accel (query sort + cull lists; the first chunk also builds the LBVH over "
                                 "the Gaussians, the others reuse it) + gs_sample_fwd per chunk",
                         "chunks": len(qs), "ms_total": ms_all, "points_per_s": len(allx) / (ms_all * 1e-3),
                         "build_ms_per_chunk": sm["build"] / max(sc["build"], 1), "fwd_ms_per_chunk": sm["fwd"] / max(sc["fwd"], 1)}
        del xs, qs, pp, ii

    # ---- the paper's own training step at this scale: raw parameters, a new random
    #      position in every cell per iteration, L1 + the false-negative term Eq. 4 fused into the forward, fused
    #      backward, Adam -- five C-ABI calls, no host arithmetic
    if world == 1 and wl["name"] == "c2":
        logit = lambda x: np.log(x / (1 - x))
        gdr = [dev(a) for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]   # the recipe updates its own copy of the model
        raw = dict(mean=gdr[0], raw_scale=dev(np.log(g.scale)), quat=gdr[2],
                   raw_opacity=dev(logit(np.clip(g.opacity.astype(np.float64), 1e-3, 1 - 1e-3)).astype(np.float32)),
                   raw_scalar=dev(logit(np.clip(g.scalar.astype(np.float64), 1e-3, 1 - 1e-3)).astype(np.float32)))
        m_d, v_d = torch.zeros(12 * g.n, device="cuda"), torch.zeros(12 * g.n, device="cuda")
        terms = torch.zeros(3, dtype=torch.float64, device="cuda")
        gr2 = ctx.alloc_grads(g.n)
        res = {}
        for label, jit in (("voxel_centres", False), ("jittered", True)):
            itr = [0]

            def rstep():
                itr[0] += 1
                qj = api.grid_query(wl["grid"], jitter_seed=itr[0] if jit else None)
                ctx.gs_preprocess(raw["mean"], gdr[1], raw["quat"], gdr[3], gdr[4], tau=TAU)
                ctx.gs_build_accel(qj)
                ctx.gs_sample_fwd_loss(qj, phi, I, tgt[0], kind=api.LOSS_L1, lambda_fn=0.5, eps_fn=0.5, loss_terms=terms)
                ctx.gs_sample_bwd(qj, None, None, None, gr2)
                ctx.gs_adam_step(raw, gr2, m_d, v_d, itr[0], scale_out=gdr[1], opacity_out=gdr[3], scalar_out=gdr[4])
            for _ in range(3):
                rstep()
            barrier()
            nrep = 100
            ctx.profile_read(); ctx.profile_enable(True)
            e0.record()
            for _ in range(nrep):
                rstep()
            e1.record(); barrier()
            smr, scr, _ = ctx.profile_read(); ctx.profile_enable(False)
            ms_r = e0.elapsed_time(e1) / nrep
            res[label] = {"ms_per_step": ms_r, "samples_per_s": P / (ms_r * 1e-3),
                          "stage_ms": {k: (smr[k] / scr[k] if scr[k] else 0.0) for k in smr}}
        out["paper_recipe"] = {"what": "preprocess + build_accel + gs_sample_fwd_loss (L1 + Eq. 4) + gs_sample_bwd (fused) + gs_adam_step on all "
                                       "samples of the grid, 100 consecutive steps of a model that is being updated", **res}
        del gdr, raw, m_d, v_d, gr2

    # ---- volume rendering through gs_render: 512 x 512 rays x 64 samples of the configs[2] model = one 2^24-sample chunk
    if world == 1 and wl["name"] == "c3":
        from paper_2607_01164_b200 import inputs
        lo, hi = wl["domain"]
        ctr = 0.5 * (np.asarray(lo, np.float64) + np.asarray(hi, np.float64))
        o_, d_, tr_ = inputs.camera_rays(512, 512, eye=tuple(ctr + np.array([1.6, -1.3, 1.1])), look_at=tuple(ctr), fov_y_deg=35.0,
                                         box=(tuple(float(x) for x in lo), tuple(float(x) for x in hi)))
        od, dd, td, tab = dev(o_), dev(d_), dev(tr_), dev(inputs.diverging_transfer(256, 30.0))
        rgba = torch.empty((len(o_), 4), device="cuda")
        ctx.gs_preprocess(*gd, domain=wl["domain"], tau=TAU)
        ctx.gs_render(od, dd, td, 64, tab, rgba); barrier()
        e0.record()
        for _ in range(3):
            ctx.gs_render(od, dd, td, 64, tab, rgba)
        e1.record(); barrier()
        ms_r = e0.elapsed_time(e1) / 3
        out["render"] = {"what": "gs_render: 512 x 512 rays x 64 samples per ray (1.68e7 samples, one chunk) of this model, emission-absorption, "
                                 "coverage as the domain test; includes the LBVH / query sort / cull of the sample positions",
                         "ms_per_frame": ms_r, "samples_per_s": len(o_) * 64 / (ms_r * 1e-3), "covered_pixels": int((rgba[:, 3] > 0).sum().item())}
        del od, dd, td, rgba

    # ---- e2e through the HOST-buffer entry point (pinned memory, copies inside the timed region)
    if world == 1:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        gh = dict(mean=pin(g.mean), scale=pin(g.scale), quat=pin(g.quat), opacity=pin(g.opacity), scalar=pin(g.scalar))
        if wl["kind"] == "grid":
            th, qh = pin(wl["target"]), api.grid_query(wl["grid"])
        else:
            th, qh = pin(wl["batches"][0][1]), api.points_query(pin(wl["batches"][0][0]))
        # the host-visible result of a training step is the loss and the gradients; the per-sample Phi / I stay on the
        # device (gs_step_host copies them back only when asked to)
        gr_h = dict(dmean=pin(np.empty((g.n, 3), np.float32)), dscale=pin(np.empty((g.n, 3), np.float32)),
                    dquat=pin(np.empty((g.n, 4), np.float32)), dopacity=pin(np.empty(g.n, np.float32)),
                    dscalar=pin(np.empty(g.n, np.float32)), err=pin(np.empty(g.n, np.float32)))
        h2d = g.n * 48 + P_total * 4 + (P_total * 12 if wl["kind"] == "points" else 0)
        d2h = 8 + g.n * 52
        for _ in range(2):
            ctx.gs_step_host(gh, qh, th, None, None, gr_h, domain=wl["domain"], tau=TAU)
        barrier()
        e2e_steps = max(2, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            ctx.gs_step_host(gh, qh, th, None, None, gr_h, domain=wl["domain"], tau=TAU)
        barrier()
        e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
        out["e2e"] = {"value": P_total / (e2e_ms * 1e-3), "unit": "points/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                      "ms_per_step": e2e_ms, "steps": e2e_steps,
                      "api": "gs_step_host (pinned host buffers): H2D model + target (+ points), D2H loss + 6 gradient tensors"}
    if headline and rank == 0:
        ffma_peak, ex2_peak, ffma2_peak = ctx.measure_alu_peaks()  # measured ALU denominators at the clocks of this run
        out["roofline"]["peak_measured"] = {"ffma_tinstr_s": ffma_peak / 1e12, "ffma2_tlaneop_s": ffma2_peak / 1e12,
                                            "mufu_ex2_tinstr_s": ex2_peak / 1e12,
                                            "how": "gs_measure_alu_peaks: register-only FMA / packed FMA / EX2 loops, CUDA events, this run"}
        # re-state the ALU side of every kernel against the FFMA rate measured in this run (the nominal figure stays beside it)
        if ffma_peak:
            scale = ALU_PEAK_TINSTR / (ffma_peak / 1e12)
            rf = out["roofline"]
            for kk in rf["kernels"].values():
                if kk["alu_ms"] is None:
                    continue
                kk["alu_ms"] *= scale
                kk["frac_alu"] = kk["alu_ms"] / kk["launch_ms"] if kk["launch_ms"] else None
                kk["issue_frac"] = kk["issue_frac"] * scale if kk["issue_frac"] is not None else None
                kk["bound"] = "alu" if kk["alu_ms"] >= kk["hbm_ms"] else "hbm"
                kk["frac"] = max(kk["alu_ms"], kk["hbm_ms"]) / kk["launch_ms"] if kk["launch_ms"] else None
            kd_ = rf["kernels"]["fwd" if rf["kernel"].endswith("fwd") else "bwd"]   # the slower of the two sampling kernels
            rf.update(bound=kd_["bound"], frac=kd_["frac"], peak=(ffma_peak / 1e12) if kd_["bound"] == "alu" else rf["hbm_peak_gbs"],
                      achieved=kd_["achieved"] if kd_["bound"] == "alu" else kd_["achieved_gbs"],
                      unit="T FP32 lane-instr/s (algorithmic: hit pairs x 19 fwd / x 40 bwd)" if kd_["bound"] == "alu" else "GB/s",
                      peak_source="FFMA lane-instr/s measured in this run (gs_measure_alu_peaks2); nominal 37.2 T beside it")
            f_, b_ = rf["kernels"]["fwd"], rf["kernels"]["bwd"]
            both = max(f_["alu_ms"] + b_["alu_ms"], f_["hbm_ms"] + b_["hbm_ms"])
            fbm = f_["launch_ms"] + b_["launch_ms"]
            cm = rf["kernels"].get("cull", {}).get("launch_ms", 0.0) or 0.0
            rf["fwd_bwd_frac"] = both / fbm if fbm else None
            rf["sampling_frac"] = both / (fbm + cm) if fbm else None
            rf["step_frac"] = both / out["ms_per_step"]
    ctx.close()
    del gd, phi, I, grads
    torch.cuda.empty_cache()
    return out


def _peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2607_01164_b200 import build as gs_build
    if not os.path.exists(gs_build.LIB):  # a fresh checkout: local rank 0 builds the library, the others wait for it
        if local == 0:
            gs_build.build()
        t_wait = time.time()
        while not os.path.exists(gs_build.LIB) and time.time() - t_wait < 600:
            time.sleep(0.5)
    torch.cuda.set_device(local % max(torch.cuda.device_count(), 1))
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # a scaling run prints its communicator / transport lines
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        # one rank per GPU over NCCL; GS_BENCH_BACKEND=gloo only exists to smoke-test this arm's code path where fewer GPUs than
        # ranks are available (two processes sharing one GPU; never a measurement)
        backend = os.environ.get("GS_BENCH_BACKEND", "nccl")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    names = ["c2", "c3", "c4", HEADLINE] if args.workload == "all" else [args.workload]
    head = names[-1]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first()
    results = {}
    for nm in names:
        wl = make_workload(nm)
        results[nm] = measure(wl, args, sampler, world, rank, headline=(nm == head))
        if rank == 0 and not args.no_cpu and world == 1:   # the oracle beside EVERY workload, on a bounded sample of each
            from oracle import wveg_oracle as oracle
            oracle.build()
            xyz, target, note = oracle_sample(wl)
            t0 = time.perf_counter()
            pts = oracle_step(wl, xyz, target)
            dt = time.perf_counter() - t0
            results[nm]["cpu_baseline"] = {"value": pts / dt, "unit": "points/s", "cores": oracle.num_threads(), "kind": "oracle",
                                           "sample": note, "seconds": dt}
        del wl
    sampler.stop()
    if rank == 0:
        r = results[head]
        line = {"metric": "query_points_per_s_fwd_bwd", "value": r["value"], "unit": "points/s", "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                "scaling": "strong" if world > 1 else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": r["config"], "clocks": r["clocks"], "gpu_launches": r["gpu_launches"], "e2e": r.get("e2e"),
                "stage_ms": r["stage_ms"], "roofline": r["roofline"], "csrc_sha16": csrc_sha16(),
                "extra": {"hit_pairs": r["hit_pairs"], "tested_pairs": r["tested_pairs"], "cull_efficiency": r["cull_efficiency"],
                          "rates": r["rates"], "decode": r.get("decode"), "render": r.get("render"), "paper_recipe": r.get("paper_recipe"),
                          "points_accel": r.get("points_accel"), "async_build": r.get("async_build"),
                          "hbm_peak_gbs_measured": _peaks().get("hbm_gbs")}}
        if "cpu_baseline" in r:
            line["cpu_baseline"] = r["cpu_baseline"]
        if len(names) > 1:
            line["workloads"] = {k: v for k, v in results.items() if k != head}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="all", choices=["all", "c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--sync-build", action="store_true", help="grid queries: keep the host round trip in gs_build_accel (GS_OPT_ASYNC_BUILD = 0)")
    ap.add_argument("--no-hit-masks", action="store_true", help="point queries: backward without the forward's hit masks (GS_OPT_BWD_HIT_MASKS = 0)")
    ap.add_argument("--points-accel", default="default", choices=["default", "gather", "scatter"],
                    help="point queries: gather = LBVH over the Gaussians (north_star); scatter = the paper's tree over the samples")
    ap.add_argument("--record-traffic", nargs=3, metavar=("NCU_RAW_CSV", "WORKLOAD", "SOURCE"),
                    help="store dram bytes per launch of an `ncu --page raw --csv` export in profiles/traffic.json")
    args = ap.parse_args()
    if args.record_traffic:
        record_traffic(*args.record_traffic)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
