#!/usr/bin/env python
"""bench.py -- one JSON line for the W-VEG sampling hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c1|c3] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input:
gs_preprocess -> gs_build_accel -> gs_sample_fwd (fused MSE) -> gs_sample_bwd.
Default workload = BASELINE.json configs[1] (C2): 256^3 Marschner-Lobb grid, 262,144 Gaussians, full-grid
forward+backward per step.  `value` = query points per second (whole job), inputs resident in HBM;
`e2e` = the same through gs_step_host with pinned HOST buffers (H2D/D2H inside the timed region).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TAU = 0.01
# algorithmic FP32-pipe lane-instructions per HIT pair: canonical predicate + weight + accumulate
INSTR_FWD = 19.0
INSTR_BWD = 40.0
# plain-ALU peak: 148 SMs x 128 FP32 lanes x 1.965 GHz (B200_PROFILING.md unit counts / max SM clock)
ALU_PEAK_TINSTR = 148 * 128 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures (bytes); a kernel
# that has no capture of the current build reports null
NCU_TRAFFIC = {
    ("c2", "k_grid_bwd"): (190.35e6 + 28.64e6, "profiles/r1_step6_c2_ncu_full.md"),
    ("c2", "k_grid_fwd"): (113.68e6 + 224.00e6, "profiles/r1_step6_c2_ncu_full.md"),
    ("c3", "k_points_bwd"): (536.48e6 + 65.86e6, "profiles/r1_step4_c3.md"),
}


def make_workload(name: str, rank: int = 0):
    from paper_2607_01164_b200 import inputs
    if name == "c2":
        grid = inputs.c2_grid(256)
        g = inputs.c2_gaussians(seed=2 + 1000 * rank, n_grid=256, n=262144)
        return dict(kind="grid", g=g, grid=grid, target=inputs.c2_target(grid), domain=None,
                    desc="C2 structured 256^3 Marschner-Lobb, 262144 Gaussians (BASELINE.json configs[1])")
    if name == "c1":
        grid = inputs.c1_grid(32)
        g = inputs.c1_gaussians(seed=0, n=1024)
        rng = np.random.default_rng(1)
        return dict(kind="grid", g=g, grid=grid, target=rng.uniform(0, 1, grid.num_points).astype(np.float32), domain=None,
                    desc="C1 tiny structured 32^3, 1024 Gaussians (BASELINE.json configs[0])")
    if name == "c3":
        xyz_all, t_all = inputs.c3_points(seed=3, p=2_000_000)
        g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=1_048_576)
        idx = inputs.batch_indices(3, rank, len(xyz_all), 1 << 20)
        return dict(kind="points", g=g, xyz=np.ascontiguousarray(xyz_all[idx]), target=np.ascontiguousarray(t_all[idx]),
                    domain=inputs.points_domain(xyz_all),
                    desc="C3 unstructured, 2^20-point batch of 2M, 1048576 Gaussians (BASELINE.json configs[2])")
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100", "-i",
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

    def stop(self, window=None):
        """window = (t0, t1) host times of the timed region: only samples taken inside it count (all, if none fell inside)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        allrows = [(t, r) for t, r in self.rows if len(r) >= 7]
        rows = [r for t, r in allrows if window is None or window[0] <= t <= window[1] + 0.1]
        if not rows:
            rows = [r for _, r in allrows]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows)}


def oracle_step(wl, sample_note: list, cap_bricks: int = 12, cap_points: int = 1 << 15):
    """One bounded-sample pass of the oracle (fwd + MSE + bwd).  Returns (points processed, hits)."""
    from oracle import wveg_oracle as oracle
    g = wl["g"]
    if wl["kind"] == "grid":
        grid = wl["grid"]
        nb = [min(c, cap_bricks) for c in grid.brick_cnt]  # a brick-aligned corner batch of the grid (12 -> 96^3)
        sub = grid.batch((0, 0, 0), tuple(nb))
        xyz = oracle.grid_points(sub)
        bd = sub.batch_dims
        full = np.asarray(wl["target"]).reshape(grid.batch_dims[2], grid.batch_dims[1], grid.batch_dims[0])
        target = np.ascontiguousarray(full[:bd[2], :bd[1], :bd[0]]).ravel()
        sample_note[:] = [f"{bd[0]}x{bd[1]}x{bd[2]} brick-aligned sub-grid, all {g.n} Gaussians, fwd+MSE+bwd"]
    else:
        n = min(len(wl["xyz"]), cap_points)
        xyz, target = wl["xyz"][:n], wl["target"][:n]
        sample_note[:] = [f"first {n} points of the batch, all {g.n} Gaussians, fwd+MSE+bwd"]
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    return len(xyz), int(fwd["count"].astype(np.int64).sum())


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import wveg_oracle as oracle
    oracle.build()
    wl = make_workload(args.workload)
    note = []
    # the per-step sample shrinks with the number of steps so that the whole run ends within a few minutes
    total = args.steps + args.warmup
    cap_bricks, cap_points = (12, 1 << 15) if total <= 250 else (6, 1 << 12) if total <= 1000 else (4, 1 << 10)
    for _ in range(args.warmup):
        oracle_step(wl, note, cap_bricks, cap_points)
    t0 = time.perf_counter()
    pts = 0
    for _ in range(args.steps):
        p, _h = oracle_step(wl, note, cap_bricks, cap_points)
        pts += p
    dt = time.perf_counter() - t0
    val = pts / dt
    line = {"impl": "reference", "metric": "query_points_per_s_fwd_bwd", "value": val, "unit": "points/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl["desc"], "sample": note[0]},
            "cpu_baseline": {"value": val, "unit": "points/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": note[0]},
            "e2e": {"value": val, "unit": "points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_01164_b200 import api

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
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    wl = make_workload(args.workload, rank)
    g = wl["g"]
    ctx = api.Context()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    gd = [dev(a) for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    if wl["kind"] == "grid":
        q = api.grid_query(wl["grid"])
    else:
        xyz_d = dev(wl["xyz"])
        q = api.points_query(xyz_d)
    P = api.query_num_points(q)
    target = dev(wl["target"])
    phi = torch.empty(P, device="cuda")
    I = torch.empty(P, device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    grads = ctx.alloc_grads(g.n)
    flat = None
    if world > 1:  # data-parallel exchange: one all-reduce of the gradients
        flat = torch.empty(g.n * 16, device="cuda")

    recipe = args.step == "recipe"
    cur_q = [q]  # the query the acceleration structure was last built for
    if recipe:  # the paper's training step: raw parameters, jitter, L1 + Eq. 4, Adam
        assert wl["kind"] == "grid", "--step recipe needs a grid workload"
        logit = lambda x: np.log(x / (1 - x))
        raw = dict(mean=gd[0], raw_scale=dev(np.log(g.scale)), quat=gd[2],
                   raw_opacity=dev(logit(np.clip(g.opacity.astype(np.float64), 1e-3, 1 - 1e-3)).astype(np.float32)),
                   raw_scalar=dev(logit(np.clip(g.scalar.astype(np.float64), 1e-3, 1 - 1e-3)).astype(np.float32)))
        m_d, v_d = torch.zeros(12 * g.n, device="cuda"), torch.zeros(12 * g.n, device="cuda")
        terms = torch.zeros(3, dtype=torch.float64, device="cuda")
        it = [0]

    def step():
        if recipe:
            it[0] += 1
            qj = api.grid_query(wl["grid"], jitter_seed=it[0])   # a new random position in every cell
            ctx.gs_preprocess(raw["mean"], gd[1], raw["quat"], gd[3], gd[4], tau=TAU)
            ctx.gs_build_accel(qj)
            cur_q[0] = qj
            ctx.gs_sample_fwd_loss(qj, phi, I, target, kind=api.LOSS_L1, lambda_fn=0.5, eps_fn=0.5, loss_terms=terms)
            ctx.gs_sample_bwd(qj, None, None, None, grads)
            ctx.gs_adam_step(raw, grads, m_d, v_d, it[0], scale_out=gd[1], opacity_out=gd[3], scalar_out=gd[4])
            return
        loss.zero_()
        ctx.gs_preprocess(*gd, domain=wl["domain"], tau=TAU)
        ctx.gs_build_accel(q)
        ctx.gs_sample_fwd(q, phi, I, target=target, loss=loss)  # fused MSE: keeps the backward coefficients
        ctx.gs_sample_bwd(q, None, None, None, grads)           # dL_dphi = NULL: backward of that fused loss
        if world > 1:
            from paper_2607_01164_b200 import dist as gsdist
            gsdist.allreduce_grads(grads, flat)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # hit / tested pair counts of this workload (outside the timed region)
    _, _, _, tested, hits = ctx.debug_point_sets(cur_q[0])
    ffma_peak, ex2_peak = ctx.measure_alu_peaks()  # measured ALU denominators at the clocks of this run
    ctx.profile_read()
    ctx.profile_enable(True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first()
    for _ in range(3):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    w1 = time.time()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop((w0, w1)) if rank == 0 else None
    stage_ms, stage_calls, launches = ctx.profile_read()
    ctx.profile_enable(False)
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    value = world * P / (ms_step * 1e-3)

    # ---- e2e through the HOST-buffer entry point (pinned memory, copies inside the timed region)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    gh = dict(mean=pin(g.mean), scale=pin(g.scale), quat=pin(g.quat), opacity=pin(g.opacity), scalar=pin(g.scalar))
    th = pin(wl["target"])
    qh = api.grid_query(wl["grid"]) if wl["kind"] == "grid" else api.points_query(pin(wl["xyz"]))
    # the host-visible result of a training step is the loss and the gradients; the per-sample Phi / I stay on the device
    # (gs_step_host copies them back only when asked to)
    phi_h, I_h = None, None
    gr_h = dict(dmean=pin(np.empty((g.n, 3), np.float32)), dscale=pin(np.empty((g.n, 3), np.float32)),
                dquat=pin(np.empty((g.n, 4), np.float32)), dopacity=pin(np.empty(g.n, np.float32)),
                dscalar=pin(np.empty(g.n, np.float32)), err=pin(np.empty(g.n, np.float32)))
    h2d = g.n * 48 + P * 4 + (P * 12 if wl["kind"] == "points" else 0)
    d2h = 8 + g.n * 52
    e2e_steps = max(2, min(args.steps, 10))
    for _ in range(2):
        ctx.gs_step_host(gh, qh, th, phi_h, I_h, gr_h, domain=wl["domain"], tau=TAU)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.gs_step_host(gh, qh, th, phi_h, I_h, gr_h, domain=wl["domain"], tau=TAU)
    barrier()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
    te = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = world * P / (float(te.item()) * 1e-3)

    if rank == 0:
        per = {k: (stage_ms[k] / stage_calls[k] if stage_calls[k] else 0.0) for k in stage_ms}
        dom_name, dom_ms, instr = ("fwd", per["fwd"], INSTR_FWD) if per["fwd"] >= per["bwd"] else ("bwd", per["bwd"], INSTR_BWD)
        achieved = hits * instr / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
        fb_ms = per["fwd"] + per["bwd_pack"] + per["bwd"] + per["finalize"]
        roof_fb = hits * (INSTR_FWD + INSTR_BWD) / (fb_ms * 1e-3) / 1e12 if fb_ms > 0 else 0.0
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        kernel = ("k_grid_" if wl["kind"] == "grid" else "k_points_") + dom_name
        traffic, traffic_src = NCU_TRAFFIC.get((args.workload, kernel), (None, None))
        line = {
            "metric": "query_points_per_s_fwd_bwd", "value": value, "unit": "points/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl["desc"], "points_per_step": P, "gaussians": g.n, "hit_pairs": hits, "tested_pairs": tested,
                       "l2": "working set per step (>600 MB of per-sample arrays) exceeds the 126 MB L2; no flush",
                       "step": "preprocess+build_accel+fwd(L1+FN, jittered samples)+bwd+adam" if recipe else "preprocess+build_accel+fwd(MSE)+bwd"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": "points/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": float(te.item()),
                    "api": "gs_step_host (pinned host buffers): H2D model + target (+ points), D2H loss + 6 gradient tensors"},
            "stage_ms": per,
            "extra": {"fwd_points_per_s": P / (per["fwd"] * 1e-3) if per["fwd"] else None,
                      "fwd_gaussian_evals_per_s": hits / (per["fwd"] * 1e-3) if per["fwd"] else None,
                      "fwd_bwd_gaussian_evals_per_s": hits / (fb_ms * 1e-3) if fb_ms else None,
                      "fwd_bwd_kernels_roofline_frac": roof_fb / ALU_PEAK_TINSTR,
                      "cull_efficiency": hits / tested if tested else None,
                      "hbm_peak_gbs_measured": peaks.get("hbm_gbs")},
            "roofline": {"bound": "alu", "kernel": kernel,
                         "achieved": achieved, "peak": ALU_PEAK_TINSTR, "unit": "T FP32 lane-instr/s (algorithmic: hit pairs x "
                         f"{instr:.0f} instr)", "frac": achieved / ALU_PEAK_TINSTR, "traffic": traffic,
                         "traffic_unit": "bytes per launch (dram read + write, ncu --set full)", "traffic_source": traffic_src,
                         "launch_ms": dom_ms,
                         "peak_source": "148 SM x 128 lanes x 1.965 GHz (B200_PROFILING.md unit counts and max SM clock)",
                         "peak_measured": {"ffma_tinstr_s": ffma_peak / 1e12, "mufu_ex2_tinstr_s": ex2_peak / 1e12,
                                           "how": "gs_measure_alu_peaks: register-only FMA / EX2 loops, CUDA events, this run"},
                         "frac_of_measured": achieved / (ffma_peak / 1e12) if ffma_peak else None},
        }
        if not args.no_cpu and world == 1:
            from oracle import wveg_oracle as oracle
            oracle.build()
            note = []
            t0 = time.perf_counter()
            pts, _h = oracle_step(wl, note, cap_bricks=32, cap_points=1 << 17)  # C2: the whole 256^3 grid (~10-20 s)
            dt = time.perf_counter() - t0
            line["cpu_baseline"] = {"value": pts / dt, "unit": "points/s", "cores": oracle.num_threads(), "kind": "oracle",
                                    "sample": note[0], "seconds": dt}
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--step", default="mse", choices=["mse", "recipe"],
                    help="mse: the north_star step (default); recipe: the paper's training step (jitter, L1 + Eq. 4, Adam)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
