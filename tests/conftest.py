import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    # GPU tests are skipped (not failed) when someone runs the whole suite on a CPU-only box.
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


def load_golden(name):
    """Parse a tests/golden/*.txt fixture: dims, nonzeros (idx SoA int32, vals fp32), factors A0.., outputs Y0.."""
    import numpy as np
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    lines = [ln.strip() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    dims = [int(x) for x in lines[0].split()]
    N = len(dims)
    mats, nz, cur = {}, [], None
    for ln in lines[1:]:
        if ln[0] in "AY" and ln[1:].isdigit():
            cur = ln
            mats[cur] = []
        elif cur is None:
            nz.append([float(x) for x in ln.split()])
        else:
            mats[cur].append([float(x) for x in ln.split()])
    nz = np.array(nz, dtype=np.float64)
    idx = np.ascontiguousarray(nz[:, :N].T.astype(np.int32))
    vals = nz[:, N].astype(np.float32)
    factors = [np.array(mats[f"A{m}"], dtype=np.float32) for m in range(N)]
    outs = [np.array(mats[f"Y{m}"], dtype=np.float64) for m in range(N)]
    return dims, idx, vals, factors, outs
