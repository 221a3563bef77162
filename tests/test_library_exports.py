"""The C-ABI library loads on a CPU-only box and exports every symbol include/nbv.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nbv.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nbv_[a-z_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_the_header():
    from paper_2602_08266_b200 import api, build
    lib_path = build.build()
    lib = ctypes.CDLL(str(lib_path))
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(api.EXPORTS) == names


def test_default_config_values_without_a_gpu():
    from paper_2602_08266_b200 import api
    cfg = api.default_config()
    assert cfg.near_plane == pytest.approx(0.01) and cfg.blur == pytest.approx(0.3)
    assert cfg.alpha_min == pytest.approx(1 / 255) and cfg.alpha_max == pytest.approx(0.99)
    assert cfg.t_stop == pytest.approx(1e-4) and cfg.channel_mask == 7
    assert cfg.alpha_obj == pytest.approx(0.3) and cfg.alpha_opa == pytest.approx(0.3)
    assert list(cfg.prior_precision) == [1.0] * 14
    cfg = api.default_config(channel_mask=15, bg=(0.1, 0.2, 0.3), prior_precision=2.0)
    assert cfg.channel_mask == 15 and cfg.bg[1] == pytest.approx(0.2) and list(cfg.prior_precision) == [2.0] * 14


def test_product_path_fails_loudly_without_cuda():
    import torch
    from paper_2602_08266_b200 import api
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        api.NBV()


def test_camera_struct_layouts_agree():
    from paper_2602_08266_b200 import synth
    from oracle import nbv_oracle as orc
    assert synth.CAMERA_DTYPE.itemsize == 72 and orc.CAMERA_DTYPE == synth.CAMERA_DTYPE
