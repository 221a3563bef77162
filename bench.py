#!/usr/bin/env python
"""bench.py -- candidate views scored per second (Hessian + information gain) on synthetic clutter scenes.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A STEP is one pass of the whole hot path over one batch: nbv_score_candidates() on the C candidate cameras of
the workload (S0' confidence, then S1..S6 per view -- S6 factors c_g H_T,g + Lambda itself, nothing is cached between
calls -- and S7 arg-max), against the training Hessian accumulated (untimed set-up) from the workload's training cameras.  The default workload is BASELINE.json
configs[2] (200,000 Gaussians, 20 objects, 1280x720, 20 training + 64 candidate cameras, RGB + depth): the
configuration north_star quotes its roofline target on.  Inputs are seeded and synthetic (paper_2602_08266_b200.synth).

`value`   : views/s with the Gaussians, H_T and all work buffers resident in HBM, device-timed per step.
`e2e`     : the same through nbv_score_candidates_host: host camera structs in, host scores + best index out,
            host<->device copies and the final synchronisation inside the timed region.
`roofline`: the dominant stage, its algorithmic work over its CUDA-event time.
`cpu_baseline`: the oracle (oracle/, as it stands) on the host cores, on a bounded sample of the same workload.
`--impl reference` times the oracle alone (this tier has no reference implementation).
N > 1 (torchrun): every rank holds a replica of the scene and scores its own C candidates (no collective on
the data path; weak scaling).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "candidate views scored/sec (Hessian + info gain)"
UNIT = "views/s"
FP32_LANES_PER_SM = 128

# EXECUTED binary32 work per unit, from hardware counters (FMA = 2 flop, a packed FFMA2 = 4):
#   flop = 2 ffma + 4 ffma2 + fmul + 2 fmul2 + fadd + 2 fadd2   (smsp__sass_thread_inst_executed_op_*_pred_on.sum)
# of one launch of each raster kernel, divided by the (pixel, list entry) evaluations of that launch (walked entries x 256).
# Both slot bodies are branch-free, so the executed work is proportional to the evaluations, composited or not; S4's
# per-entry moment assembly and reduction are amortised into its figure.  Source: FLOP_SOURCE (committed ncu pass).
FLOP_PER_EVAL = {"forward": 31.6, "backward": {3: 84.7, 4: 99.9}}
FLOP_SOURCE = "profiles/r2_ncu_flops_cfg2.md"
BYTES_PER_KEY = 8         # S2: a (supertile, depth rank) key must be written once and read once (4 + 4 B)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch (8 views) from the committed `ncu --set full` capture named
# in TRAFFIC_SOURCE; known for config 2 only (null elsewhere)
NCU_TRAFFIC_BYTES_PER_VIEW = {2: {"backward": 236.8e6 / 16, "forward": 158.2e6 / 16}}      # the capture is of a 16-view launch
TRAFFIC_SOURCE = "profiles/r2_ncu_raster_cfg2.md (ncu --set full of the first candidate batch; a stored figure, not measured by this run)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-sample-views", type=int, default=0, help="oracle sample size (0 = automatic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--concurrency", type=int, default=0, help="views in flight (0 = library default)")
    ap.add_argument("--no-selection", action="store_true", help="skip the greedy / fused-output timings (SURVEY 8(f) rows)")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# --------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name).read().strip().splitlines() if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            if len(r) < 6:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for n, v in zip(names, r[2:6]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------------
def oracle_setup(wl):
    from oracle import nbv_oracle as orc
    s = wl.scene
    scn = orc.OracleScene(s.mean, s.logscale, s.quat, s.opacity, s.rgb, s.obj_logits, orc.default_config(wl.channel_mask))
    return orc, scn


def oracle_score_views(orc, scn, wl, H_T, cams):
    """S0' + (S1..S6 per view) + S7 with the oracle; returns seconds."""
    t0 = time.perf_counter()
    orc.score_candidates(scn, wl.train_cams[:0], cams, wl.target_obj, H_T=H_T)
    return time.perf_counter() - t0


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(wl, n_views: int):
    orc, scn = oracle_setup(wl)
    # H_T of ONE training view (untimed): scoring cost does not depend on how many views H_T sums
    H_T = np.zeros((scn.N, orc.NB))
    scn.view_hessian(wl.train_cams[0], out=H_T)
    dt = oracle_score_views(orc, scn, wl, H_T, wl.cand_cams[:n_views])
    return {"value": n_views / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "cpu": cpu_model(),
            "sample": "first %d candidate view(s) of the workload scored against H_T of its first training view "
                      "(%.1f s wall, OpenMP over pixels)" % (n_views, dt)}


def auto_sample_views(cfg_index: int) -> int:
    return 4          # at least 4 views (about 40 s of host time at config 2)


def run_reference(args, wl, rank: int):
    """--impl reference: the oracle, each step a bounded sample (n candidate views) of the workload."""
    if rank != 0:
        return
    # every step scores n candidate views; n = 1 at the large configs so that W + K steps end within a few minutes
    n = args.cpu_sample_views or {0: 4, 1: 2}.get(args.config, 1)
    orc, scn = oracle_setup(wl)
    H_T = np.zeros((scn.N, orc.NB))
    scn.view_hessian(wl.train_cams[0], out=H_T)
    C = len(wl.cand_cams)
    pick = lambda i: wl.cand_cams[[(i * n + j) % C for j in range(n)]]
    for i in range(args.warmup):
        oracle_score_views(orc, scn, wl, H_T, pick(i))
    total = 0.0
    for i in range(args.steps):
        total += oracle_score_views(orc, scn, wl, H_T, pick(args.warmup + i))
    v = n * args.steps / total
    sample = "each step = %d candidate view(s) of the workload scored by the oracle against H_T of one training view" % n
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(args, wl, "host", candidates_per_step=n, training_views=1),
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "cpu": cpu_model(), "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def workload_config(args, wl, where: str, candidates_per_step=None, training_views=None):
    """what this arm ran: the reference arm scores a bounded sample per step (candidates_per_step, training_views given)"""
    s = wl.scene
    return {"workload": "BASELINE.json configs[%d] (%s)" % (args.config, wl.name), "gaussians": s.N, "objects": s.K,
            "image": "%dx%d" % (int(wl.cand_cams[0]["width"]), int(wl.cand_cams[0]["height"])),
            "training_views": int(len(wl.train_cams) if training_views is None else training_views),
            "candidates_per_step": int(len(wl.cand_cams) if candidates_per_step is None else candidates_per_step),
            "workload_training_views": int(len(wl.train_cams)), "workload_candidates": int(len(wl.cand_cams)),
            "channels": "rgb+depth" if wl.channel_mask == 15 else "rgb", "target_obj": int(wl.target_obj), "P": 14,
            "seed": int(wl.seed), "parallelism": "replicas x%d" % args.gpus,
            "l2": "flushed between steps (512 MiB write); per-batch working set (keys, splats, H_T) exceeds the 126 MB L2"
                  if where == "device" else "n/a"}


# --------------------------------------------------------------------------------------------------
def bench_selection(nbv, wl, api, torch):
    """The rows SURVEY.md section 8(f) marks "next", timed on the same workload (extra keys, not the headline):
    greedy selection of 6 views and per-output normalised, fused scoring (Eq. 10-11)."""
    C, T = len(wl.cand_cams), len(wl.train_cams)
    rounds = min(6, C)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def fresh(n):
        n.reset_training()
        n.accumulate_training(wl.train_cams)

    res = {}
    nbv.select_greedy(wl.cand_cams, rounds, wl.target_obj, want_scores=False)          # warm-up: pool allocation
    fresh(nbv)
    a, b = ev(), ev()
    a.record()
    order, _ = nbv.select_greedy(wl.cand_cams, rounds, wl.target_obj, want_scores=False)
    b.record(); b.synchronize()
    ms = a.elapsed_time(b)
    scored = sum(C - r for r in range(rounds))
    res["greedy"] = {"rounds": rounds, "candidates": C, "ms": ms, "candidate_scorings_per_s": scored / (ms * 1e-3),
                     "order": [int(i) for i in order], "call": "nbv_select_greedy (every candidate rasterised once, rounds on cached blocks)"}
    fresh(nbv)
    n_rgb, n_d = api.NBV(channel_mask=api.CH_RGB), api.NBV(channel_mask=api.CH_DEPTH)
    for n in (n_rgb, n_d):
        n.load_scene(wl.scene)
        n.accumulate_training(wl.train_cams)
    api.score_candidates_fused(n_rgb, n_d, wl.train_cams, wl.cand_cams, wl.target_obj)  # warm-up
    a, b = ev(), ev()
    a.record()
    out = api.score_candidates_fused(n_rgb, n_d, wl.train_cams, wl.cand_cams, wl.target_obj)
    b.record(); b.synchronize()
    ms = a.elapsed_time(b)
    res["fused"] = {"candidates": C, "training_views_rescored": T, "ms": ms, "views_per_s": C / (ms * 1e-3),
                    "best": int(out["best"].item()), "denominators": [float(x) for x in out["denom"].cpu()],
                    "call": "nbv_score_candidates_fused (rgb and depth contexts; candidates and training views scored in both)"}
    # the object-mask output alone, and Eq. 11 with all three outputs
    n_o = api.NBV(channel_mask=api.CH_MASK)
    n_o.load_scene(wl.scene)
    n_o.accumulate_training(wl.train_cams)
    sc = torch.empty(C, dtype=torch.float32, device="cuda"); bb = torch.empty(1, dtype=torch.int32, device="cuda")
    n_o.score_candidates(wl.cand_cams, wl.target_obj, sc, bb)                           # warm-up
    n_o.set_stage_timing(True)
    a, b = ev(), ev()
    a.record()
    n_o.score_candidates(wl.cand_cams, wl.target_obj, sc, bb)
    b.record(); b.synchronize()
    ms = a.elapsed_time(b)
    st_ms, nv = n_o.stage_times()
    n_o.set_stage_timing(False)
    res["mask"] = {"candidates": C, "object_channels": int(wl.scene.K), "block_parameters": 11 + int(wl.scene.K), "ms": ms,
                   "views_per_s": C / (ms * 1e-3), "stage_ms_per_view": {k: v / max(nv, 1) for k, v in st_ms.items()},
                   "call": "nbv_score_candidates on a NBV_CH_MASK context (S4 once per group of 4 object channels)"}
    api.score_candidates_fused(n_rgb, n_d, wl.train_cams, wl.cand_cams, wl.target_obj, nbv_mask=n_o)      # warm-up
    a, b = ev(), ev()
    a.record()
    out = api.score_candidates_fused(n_rgb, n_d, wl.train_cams, wl.cand_cams, wl.target_obj, nbv_mask=n_o)
    b.record(); b.synchronize()
    ms = a.elapsed_time(b)
    res["fused3"] = {"candidates": C, "training_views_rescored": T, "ms": ms, "views_per_s": C / (ms * 1e-3),
                     "best": int(out["best"].item()), "denominators": [float(x) for x in out["denom"].cpu()],
                     "call": "nbv_score_candidates_fused with the mask context (Eq. 11, all three outputs)"}
    n_rgb.close(); n_d.close(); n_o.close()
    return res


def rank_candidates(cfg_index: int, wl, rank: int):
    """Candidate cameras rank `rank` scores: rank 0 keeps the workload's own set; every other replica draws its own set
    of the same size from a rank-seeded generator (same scene, same hemisphere recipe) -- independent units, no exchange."""
    if rank == 0:
        return wl.cand_cams
    from paper_2602_08266_b200 import synth
    c = synth.CONFIGS[cfg_index]
    f = synth._intrinsics(c)
    return synth.hemisphere_cameras(c["C"], c["radius"], c["W"], c["H"], f, f, np.random.default_rng(10_000 + rank))


def gather_over_ranks(per_step, dist, device):
    """(ranks, steps) array of every rank's per-step times; `dist` is torch.distributed or None (single process)."""
    import torch
    t = torch.tensor([list(per_step)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        parts = [torch.zeros_like(t) for _ in range(dist.get_world_size())]
        dist.all_gather(parts, t)
        t = torch.cat(parts)
    return t.cpu().numpy()


def aggregate(step_ms_per_rank, views_per_rank_step):
    """Whole-job throughput: units of all ranks / slowest rank's time.  step_ms_per_rank: (ranks, steps)."""
    t = np.asarray(step_ms_per_rank, dtype=np.float64)
    total_ms = t.sum(axis=1).max()
    steps = t.shape[1]
    return dict(value=t.shape[0] * views_per_rank_step * steps / (total_ms * 1e-3), ms_per_step=total_ms / steps)


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    from paper_2602_08266_b200 import synth
    wl = synth.make_workload(args.config)
    if args.impl == "reference":
        run_reference(args, wl, rank)
        return

    import torch
    from paper_2602_08266_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    wl.cand_cams = rank_candidates(args.config, wl, rank)   # replicas score their own candidate sets

    nbv = api.NBV(channel_mask=wl.channel_mask)
    if args.concurrency:
        nbv.set_concurrency(args.concurrency)
    t0 = time.perf_counter()
    nbv.load_scene(wl.scene)
    torch.cuda.synchronize()
    load_s = time.perf_counter() - t0
    ev = lambda: torch.cuda.Event(enable_timing=True)
    nbv.accumulate_training(wl.train_cams)              # untimed: creates the slots' work buffers
    nbv.reset_training()
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    nbv.accumulate_training(wl.train_cams)
    e1.record()
    torch.cuda.synchronize()
    train_ms = e0.elapsed_time(e1)

    C = len(wl.cand_cams)
    scores = torch.empty(C, dtype=torch.float32, device="cuda")
    best = torch.empty(1, dtype=torch.int32, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        nbv.score_candidates(wl.cand_cams, wl.target_obj, scores, best)
    # ---- timed region: K steps, device-timed per step, L2 flushed between steps (library instrumentation off) ----
    launches0 = nbv.kernel_launches()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    barrier()
    step_ms = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = ev(), ev()
        a.record()
        nbv.score_candidates(wl.cand_cams, wl.target_obj, scores, best)
        b.record()
        b.synchronize()
        step_ms.append(a.elapsed_time(b))
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = (nbv.kernel_launches() - launches0) // max(args.steps, 1)
    # ---- the same K steps again with the library's per-stage CUDA events on (they cost ~4%, hence a separate pass) ----
    nbv.set_stage_timing(True)
    for _ in range(args.steps):
        flush.fill_(1)
        nbv.score_candidates(wl.cand_cams, wl.target_obj, scores, best)
    stage_ms, n_timed_views = nbv.stage_times()
    # ---- and once more ONE BATCH PER CALL: in the full call the S3 launch of batch b+1 shares the SMs with the S4 launch of
    # batch b (two raster streams), so a launch's event-to-event duration there includes time the other kernel ran; with one
    # batch per call every raster launch has the GPU to itself and its duration is the kernel's own (`roofline` uses these) ----
    W_, H_ = int(wl.cand_cams[0]["width"]), int(wl.cand_cams[0]["height"])
    vpl = nbv.batch_views(W_, H_)                       # views per S3 / S4 / S5+S6 launch, as the library batches them
    vpl = min(vpl, C)
    nbv.set_stage_timing(True)                          # clears the accumulated times of the pass above
    for _ in range(args.steps):
        flush.fill_(1)
        for c0 in range(0, C, vpl):
            nbv.score_candidates(wl.cand_cams[c0:c0 + vpl], wl.target_obj, scores[c0:c0 + vpl], best)
    stage_ms_x, n_timed_views_x = nbv.stage_times()
    nbv.set_stage_timing(False)

    # ---- e2e: host cameras in, host scores out, through nbv_score_candidates_host ----
    for _ in range(min(args.warmup, 2)):
        nbv.score_candidates_host(wl.cand_cams, wl.target_obj)
    barrier()
    e2e_s = []
    for _ in range(args.steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h_scores, h_best = nbv.score_candidates_host(wl.cand_cams, wl.target_obj)
        e2e_s.append(time.perf_counter() - t0)
    barrier()

    # ---- counts of the same views (untimed pass) for the algorithmic work ----
    tot = dict(n_visible=0, n_keys=0, n_entries=0, n_pairs=0, n_touched=0, n_coarse=0)
    for cam in wl.cand_cams:
        nbv.gaussian_gains(cam, wl.target_obj)          # hot kernels: n_visible, n_keys, n_coarse, n_touched
        st = nbv.last_view_stats()
        nbv.render(cam)                                 # counting forward pass: n_entries, n_pairs
        st_r = nbv.last_view_stats()
        st["n_entries"], st["n_pairs"] = st_r["n_entries"], st_r["n_pairs"]
        for k in tot:
            tot[k] += st[k]

    # ---- gather over ranks ----
    t_all = gather_over_ranks(step_ms, dist, "cuda")
    e_all = gather_over_ranks(e2e_s, dist, "cuda")
    agg = aggregate(t_all, C)
    agg_e2e = aggregate(e_all * 1e3, C)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    ffma_tflops = api.measure_ffma_peak()               # measured fp32 CUDA-core peak (FFMA chains) on this box
    nch = 4 if wl.channel_mask & 8 else 3
    views = max(n_timed_views, 1)
    per_view_ms = {k: v / views for k, v in stage_ms.items()}
    per_view_ms_x = {k: v / max(n_timed_views_x, 1) for k, v in stage_ms_x.items()}       # one batch per call: exclusive
    avg = {k: v / C for k, v in tot.items()}            # per view
    evals = avg["n_entries"] * 256.0                    # (pixel, list entry) evaluations per view
    n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    alu_peak = n_sm * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12    # TFLOP/s
    work = {
        "backward": ("alu", evals * FLOP_PER_EVAL["backward"][nch] / 1e12, alu_peak, "TFLOP/s"),
        "forward": ("alu", evals * FLOP_PER_EVAL["forward"] / 1e12, alu_peak, "TFLOP/s"),
        "coarse_sort": ("hbm", avg["n_coarse"] * BYTES_PER_KEY / 1e9, peaks["hbm_gbs"], "GB/s"),
    }
    rl = {}
    for k, (bound, amount, peak, unit) in work.items():
        batched = k in ("backward", "forward")
        sec = (per_view_ms_x[k] if batched else per_view_ms[k]) * 1e-3
        ach = amount / sec if sec > 0 else 0.0
        rl[k] = {"bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                 "traffic": (NCU_TRAFFIC_BYTES_PER_VIEW[args.config][k] * vpl) if k in NCU_TRAFFIC_BYTES_PER_VIEW.get(args.config, {}) else None,
                 "traffic_source": TRAFFIC_SOURCE if k in NCU_TRAFFIC_BYTES_PER_VIEW.get(args.config, {}) else None,
                 "flops_source": ("executed fp32 flop per evaluation from " + FLOP_SOURCE) if batched else None,
                 "views_per_launch": vpl if batched else 1,
                 "ms_per_launch": (per_view_ms_x[k] * vpl) if batched else per_view_ms[k],
                 "ms_per_launch_in_full_call": per_view_ms[k] * (vpl if batched else 1),
                 "timing": ("CUDA events around the launch on its own stream, one batch per call (the launch has the GPU to itself); "
                            "in the full call launches of two batches overlap: ms_per_launch_in_full_call") if batched else
                           "CUDA events on the slot stream in the full call", "peak_source": peaks["source"] if bound == "hbm" else
                 "%d SM x 128 lanes x 2 x %.0f MHz (DESIGN.md section 8)" % (n_sm, peaks["sm_max_mhz"])}
    # dominant kernel = largest share of GPU time in the ncu launch list (profiles/): one of the two raster stages; the
    # S1-S2 stage times are taken on slot streams that wait behind the raster launches and are not exclusive
    dominant = max(("backward", "forward"), key=lambda k: per_view_ms_x[k])
    roofline = dict(rl[dominant], kernel=dominant)
    if roofline["bound"] == "alu":
        roofline["peak_measured_ffma"] = ffma_tflops
        roofline["frac_of_measured_ffma"] = roofline["achieved"] / ffma_tflops if ffma_tflops else None
    # whole-view bound: sum over stages of the stage's own lower bound
    t_min_ms = sum(1e3 * work[k][1] / work[k][2] for k in work)
    view_ms = agg["ms_per_step"] / C                    # wall time per view (stages of different views overlap)

    out = {
        "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": agg["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "dtype_note": "S1-S4 binary32 (S4's 40 moments per (tile, Gaussian)), their sum across tiles and S5-S6 binary64 (1-2% of a view)",
        "data": "synthetic", "config": workload_config(args, wl, "device"),
        "clocks": clocks,
        "e2e": {"value": agg_e2e["value"], "unit": UNIT, "h2d_bytes_per_step": int(72 * C), "d2h_bytes_per_step": int(4 * C + 4),
                "call": "nbv_score_candidates_host (host camera structs in, host scores + best out, stream synchronised)"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "stage_ms_per_view": per_view_ms,
        "stage_ms_per_view_exclusive": per_view_ms_x,
        "stage_rooflines": rl,
        "view_roofline": {"t_min_ms": t_min_ms, "t_measured_ms": view_ms, "frac": t_min_ms / view_ms if view_ms else None,
                          "note": "sum over stages of (executed fp32 work or algorithmic bytes / peak) against wall time per view"},
        "counts_per_view": avg,
        "setup": {"load_s": load_s, "training_views_per_s": len(wl.train_cams) / (train_ms * 1e-3) if train_ms else None},
        "best": int(h_best),
    }
    if world == 1 and not args.no_selection:
        out["selection"] = bench_selection(nbv, wl, api, torch)
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(wl, args.cpu_sample_views or auto_sample_views(args.config))
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
