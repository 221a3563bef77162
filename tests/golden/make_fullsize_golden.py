"""Writes tests/golden/fullsize_cfg{1,2,3,4}.json: the CPU oracle's scores for the FULL candidate set of BASELINE.json
configs 1-4 against the FULL training Hessian H_T, and the arg-max (Eq. 5).

Calls only `oracle/` and the seeded input generator (`paper_2602_08266_b200/synth.py`, which holds none of the method's
arithmetic); nothing here comes from the CUDA path.  The `-m gpu` tests in tests/test_gpu_golden.py compare
`nbv_score_candidates` over the whole candidate set with these values (1e-3 relative) and the index exactly.

    python tests/golden/make_fullsize_golden.py [--configs 1 2 3 4] [--work /tmp/nbv_golden] [--progress DIR] [--max-seconds S]

Cost: one oracle pass per view (about 3 s at config 1, 10-25 s at configs 2-4 on 8-16 host threads), 30 / 84 / 84 / 306
views.  Restartable: H_T (large, under --work) and the scores computed so far (a small JSON per config, under --progress,
default --work) are kept; --max-seconds stops cleanly between views so that a time-limited job can be continued by the
next one (H_T is recomputed when --work was lost, the finished candidates are not).

What is stored per config: `scores` (C binary64 numbers), `best`, the number of Gaussians with a non-zero block per
candidate, the training-view count, sha256 of oracle/nbv_oracle.cpp and of the Python oracle functions used, and a
checksum of the input arrays (so a test can tell stale values from a failing kernel).

A Gaussian whose candidate block is zero has gain exactly 0 (pinned: tests/test_oracle_gain.py, `H_c = 0 -> 0`), so the
oracle's `gaussian_gains` is called on the touched Gaussians only -- the same numbers, a fraction of the slogdets.
"""
from __future__ import annotations

import argparse
import dataclasses
import hashlib
import inspect
import json
import os
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from oracle import nbv_oracle as orc            # noqa: E402
from paper_2602_08266_b200 import synth         # noqa: E402

GOLDEN = Path(__file__).resolve().parent


def oracle_hashes() -> dict:
    cpp = hashlib.sha256((ROOT / "oracle" / "nbv_oracle.cpp").read_bytes()).hexdigest()
    fns = [orc.confidence, orc.gaussian_gains, orc.unpack_blocks, orc.softmax, orc.argmax_lowest, orc.select_greedy]
    py = hashlib.sha256("".join(inspect.getsource(f) for f in fns).encode()).hexdigest()
    return dict(oracle_cpp_sha256=cpp, oracle_py_functions_sha256=py)


def input_checksum(wl) -> str:
    h = hashlib.sha256()
    s = wl.scene
    for a in (s.mean, s.logscale, s.quat, s.opacity, s.rgb, s.obj_logits, wl.train_cams, wl.cand_cams):
        h.update(np.ascontiguousarray(a).tobytes())
    h.update(str((wl.channel_mask, wl.target_obj)).encode())
    return h.hexdigest()


# Config 4 (1,000,000 Gaussians, 50 + 256 cameras) costs the oracle 2-4 minutes per view: its stored values are a SAMPLE,
# H_T of the first SAMPLE_TRAIN[4] training views and the SAMPLE_CAND[4] candidates below (one in every batch region of the
# 256-candidate call: first / last batch, both raster streams); the test scores all 256 candidates in one call against the
# same H_T and compares the sampled ones.
SAMPLE_TRAIN = {4: 4}
SAMPLE_CAND = {4: [0, 37, 74, 111, 148, 185, 222, 255]}


def sampled_workload(cfg: int):
    """The workload of a config, its training views cut to the stored sample; the candidate indices the oracle scores."""
    wl = synth.make_workload(cfg)
    cand_idx = SAMPLE_CAND.get(cfg, list(range(len(wl.cand_cams))))
    if cfg in SAMPLE_TRAIN:
        wl = dataclasses.replace(wl, train_cams=wl.train_cams[: SAMPLE_TRAIN[cfg]])
    return wl, cand_idx


def run_config(cfg: int, work: Path, progress: Path, deadline: float) -> bool:
    wl, cand_idx = sampled_workload(cfg)
    s = wl.scene
    scn = orc.OracleScene(s.mean, s.logscale, s.quat, s.opacity, s.rgb, s.obj_logits, orc.default_config(wl.channel_mask))
    T, C = len(wl.train_cams), len(wl.cand_cams)
    tag = "cfg%d" % cfg
    ht_file, prog_file = work / (tag + "_HT.npy"), progress / (tag + "_progress.json")
    t0 = time.time()
    if ht_file.exists():
        H_T = np.load(ht_file)
    else:
        # H_T = sum over the training views (Eq. 6), in view order; checkpointed every few views (a time-limited job may stop)
        part_file, part_meta = work / (tag + "_HT_partial.npy"), work / (tag + "_HT_partial.json")
        done = 0
        H_T = np.zeros((s.N, orc.NB))
        if part_file.exists() and part_meta.exists():
            meta = json.loads(part_meta.read_text())
            if meta.get("input_sha256") == input_checksum(wl) and meta.get("hashes") == oracle_hashes():
                H_T, done = np.load(part_file), int(meta["views_done"])
        for i in range(done, T):
            if time.time() > deadline:
                print("%s: time budget used, %d/%d training views done" % (tag, i, T), flush=True)
                return False
            scn.view_hessian(wl.train_cams[i], out=H_T)
            print("%s training view %d/%d  %.0f s" % (tag, i + 1, T, time.time() - t0), flush=True)
            if (i + 1) % 4 == 0 and i + 1 < T:
                np.save(part_file, H_T)
                part_meta.write_text(json.dumps(dict(views_done=i + 1, input_sha256=input_checksum(wl), hashes=oracle_hashes())))
        np.save(ht_file, H_T)
    prog = json.loads(prog_file.read_text()) if prog_file.exists() else dict(scores={}, touched={})
    if prog.get("input_sha256", input_checksum(wl)) != input_checksum(wl) or prog.get("hashes", oracle_hashes()) != oracle_hashes():
        prog = dict(scores={}, touched={})              # progress of other inputs or another oracle: start over
    prog["input_sha256"], prog["hashes"] = input_checksum(wl), oracle_hashes()
    conf = orc.confidence(s.obj_logits, s.opacity, target=wl.target_obj)
    prior = np.ones(orc.P)
    for i in cand_idx:
        if str(i) in prog["scores"]:
            continue
        if time.time() > deadline:
            print("%s: time budget used, %d/%d candidates done" % (tag, len(prog["scores"]), len(cand_idx)), flush=True)
            return False
        H_c = scn.view_hessian(wl.cand_cams[i])
        touched = np.flatnonzero(np.abs(H_c).sum(axis=1) > 0)
        g = orc.gaussian_gains(H_T[touched], H_c[touched], conf[touched], prior)
        prog["scores"][str(i)] = float(g.sum())
        prog["touched"][str(i)] = int(touched.size)
        prog_file.write_text(json.dumps(prog))
        print("%s candidate %d (of %d stored)  score %.9g  touched %d  %.0f s" % (tag, i, len(cand_idx), g.sum(), touched.size, time.time() - t0),
              flush=True)
    scores = [prog["scores"][str(i)] for i in cand_idx]
    # `scores[j]` belongs to candidate `cand_idx[j]`; `best` is an index into the workload's candidate array
    out = dict(config=cfg, name=wl.name, N=s.N, K=s.K, n_train=T, n_cand=C, cand_idx=[int(i) for i in cand_idx],
               channel_mask=wl.channel_mask, target_obj=wl.target_obj, prior_precision=1.0, alpha_obj=0.3, alpha_opa=0.3,
               scores=scores, best=int(cand_idx[orc.argmax_lowest(np.array(scores))]),
               n_touched=[prog["touched"][str(i)] for i in cand_idx],
               ht_trace_sum=float(orc.unpack_blocks(H_T[:: max(1, s.N // 5000)]).trace(axis1=1, axis2=2).sum()),
               input_sha256=input_checksum(wl), cite="PAPER.md L185 Eq. 5, L199-205 Eq. 6, L229-244 Eq. 7-9, L695-706 Eq. 12",
               written_by="tests/golden/make_fullsize_golden.py", **oracle_hashes())
    if cfg == 1:
        # greedy multi-view selection (Eq. 5 repeated, "6 rounds") on the full config-1 candidate set
        g = orc.select_greedy(scn, wl.train_cams, wl.cand_cams, rounds=6, target=wl.target_obj)
        out["greedy_order"] = [int(v) for v in g["order"]]
        out["greedy_scores"] = [[None if np.isnan(v) else float(v) for v in row] for row in g["scores"]]
    (GOLDEN / ("fullsize_%s.json" % tag)).write_text(json.dumps(out, indent=1) + "\n")
    print("%s written: best %d, %.0f s" % (tag, out["best"], time.time() - t0), flush=True)
    return True


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[1, 2, 3, 4])
    ap.add_argument("--work", default="/tmp/nbv_golden")
    ap.add_argument("--progress", default=None)
    ap.add_argument("--max-seconds", type=float, default=1e9)
    a = ap.parse_args()
    os.makedirs(a.work, exist_ok=True)
    os.makedirs(a.progress or a.work, exist_ok=True)
    deadline = time.time() + a.max_seconds
    for c in a.configs:
        if not run_config(c, Path(a.work), Path(a.progress or a.work), deadline):
            break
