"""Writes tests/golden/mask_fullres.json: the CPU oracle's object-mask output (Eq. 1-2)
at the image size and channel count bench.py times it on -- 1280 x 720, K = 20 object channels, blocks of L = 31 parameters
-- on a 20,000-Gaussian scene (the recipe of BASELINE.json configs[2], fewer Gaussians: the oracle forms explicit 31-wide
rows per (pixel, Gaussian, channel) pair and needs minutes per view even so).

Calls only `oracle/` and the seeded input generator; nothing here comes from the CUDA path.

    python tests/golden/make_mask_golden.py

Stored: H_T of the first training view and the blocks of candidate 0 for a fixed sample of touched Gaussians (every
`BLOCK_STEP`-th touched one), the per-Gaussian gains of candidates 0 and 1 against that H_T for every touched Gaussian, both
scores, the arg-max, the sets of touched Gaussians, and the hashes / input checksum that tell stale values from a failing
kernel.
"""
from __future__ import annotations

import hashlib
import inspect
import json
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
N_GAUSSIANS, N_TRAIN, N_CAND, BLOCK_STEP, BG = 20_000, 1, 2, 192, 0


def workload():
    return synth.make_workload(2, n_gaussians=N_GAUSSIANS, n_train=N_TRAIN, n_cand=N_CAND)


def oracle_hashes() -> dict:
    src = b"".join((ROOT / "oracle" / f).read_bytes() for f in ("nbv_oracle.cpp", "nbv_oracle_ext.inc"))
    fns = [orc.confidence, orc.gaussian_gains_L, orc.unpack_blocks_L, orc.softmax, orc.argmax_lowest, orc.view_hessian_mask]
    py = hashlib.sha256("".join(inspect.getsource(f) for f in fns).encode()).hexdigest()
    return dict(oracle_cpp_sha256=hashlib.sha256(src).hexdigest(), oracle_py_functions_sha256=py)


def input_checksum(wl) -> str:
    h = hashlib.sha256()
    s = wl.scene
    for a in (s.mean, s.logscale, s.quat, s.opacity, s.rgb, s.obj_logits, wl.train_cams, wl.cand_cams):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def _short(a):
    """10 significant digits: the comparisons are at 1e-3"""
    return [[float("%.10g" % v) for v in row] for row in np.asarray(a)]


def main():
    wl = workload()
    s = wl.scene
    L = 11 + s.K
    scn = orc.OracleScene(s.mean, s.logscale, s.quat, s.opacity, s.rgb, s.obj_logits, orc.default_config(7))
    t0 = time.time()
    H_T = np.zeros((s.N, orc.mask_block_size(s.K)))
    for cam in wl.train_cams:
        orc.view_hessian_mask(scn, cam, BG, out=H_T)
        print("training view done  %.0f s" % (time.time() - t0), flush=True)
    conf = orc.confidence(s.obj_logits, s.opacity, target=-1)
    out = dict(N=s.N, K=s.K, L=L, image=[int(wl.cand_cams[0]["width"]), int(wl.cand_cams[0]["height"])], n_train=N_TRAIN, n_cand=N_CAND,
               bg_channel=BG, prior_precision=1.0, prior_precision_obj=1.0, alpha_obj=0.3, alpha_opa=0.3, block_step=BLOCK_STEP,
               cite="PAPER.md L122-139 Eq. 1-2, L248, L185 Eq. 5, L199-205 Eq. 6, L229-244 Eq. 7-9",
               written_by="tests/golden/make_mask_golden.py", input_sha256=input_checksum(wl), **oracle_hashes())
    tt = np.flatnonzero(np.abs(H_T).max(axis=1) > 0)
    out["train_touched"] = [int(v) for v in tt]
    out["train_blocks"] = _short(H_T[tt[::BLOCK_STEP]])
    scores, cands = [], []
    for i, cam in enumerate(wl.cand_cams):
        H_c = orc.view_hessian_mask(scn, cam, BG)
        t = np.flatnonzero(np.abs(H_c).max(axis=1) > 0)
        g = orc.gaussian_gains_L(H_T[t], H_c[t], conf[t], np.ones(L), L)
        scores.append(float(g.sum()))
        c = dict(touched=[int(v) for v in t], gains=[float("%.12g" % v) for v in g])
        if i == 0:
            c["blocks"] = _short(H_c[t[::BLOCK_STEP]])
        cands.append(c)
        print("candidate %d  score %.9g  touched %d  %.0f s" % (i, g.sum(), t.size, time.time() - t0), flush=True)
    out["scores"], out["best"], out["candidates"] = scores, orc.argmax_lowest(np.array(scores)), cands
    (GOLDEN / "mask_fullres.json").write_text(json.dumps(out) + "\n")
    print("written, %.0f s" % (time.time() - t0))


if __name__ == "__main__":
    main()
