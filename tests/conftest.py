import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: takes more than ~20 s on 8 host cores")


def make_oracle_scene(scene, channel_mask=7, **cfg_kw):
    from oracle import nbv_oracle as orc
    return orc.OracleScene(scene.mean, scene.logscale, scene.quat, scene.opacity, scene.rgb, scene.obj_logits,
                           orc.default_config(channel_mask, **cfg_kw))


def scene_from_arrays(mean, logscale, quat, opacity, rgb, K=2):
    """Scene for hand-built micro cases (uniform object logits)."""
    from paper_2602_08266_b200 import synth
    f = lambda a, s: np.ascontiguousarray(np.asarray(a, dtype=np.float32).reshape(s))
    n = np.asarray(mean).reshape(-1, 3).shape[0]
    return synth.Scene(f(mean, (n, 3)), f(logscale, (n, 3)), f(quat, (n, 4)), f(opacity, (n,)), f(rgb, (n, 3)),
                       np.zeros((n, K), dtype=np.float32), np.zeros(n, dtype=np.int32))


@pytest.fixture(scope="session")
def wl0():
    from paper_2602_08266_b200 import synth
    return synth.make_workload(0)
