import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_sessionfinish(session, exitstatus):
    # worst parity errors seen by the GPU tests of this session (rel L2, max-abs ratio) -> a small
    # JSON in gpurun_out/ (scratch, git-ignored) used to calibrate / report the tolerances
    mod = sys.modules.get("test_gpu_parity")
    worst = getattr(mod, "WORST", None) if mod else None
    if not worst:
        return
    try:
        import json
        out = os.path.join(ROOT, "gpurun_out")
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_worst.json"), "w") as fh:
            json.dump({k: {"rel_l2": v[0], "max_ratio": v[1]} for k, v in sorted(worst.items())}, fh, indent=1)
    except Exception:
        pass
