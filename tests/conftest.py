import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (builds oracle/liboracle.so with gcc on first use)."""
    import oracle
    oracle.build()
    return oracle


def rel_err(a, b):
    """max|a-b| / max|b| -- the parity metric of BASELINE.json:north_star."""
    import numpy as np
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    m = float(np.max(np.abs(b))) if b.size else 0.0
    if m == 0.0:
        return float(np.max(np.abs(a - b))) if b.size else 0.0
    return float(np.max(np.abs(a - b)) / m)


@pytest.fixture(scope="session")
def jt():
    """The CUDA path: builds libjt.so in-tree if stale and returns the binding (fails loudly, no fallback)."""
    from paper_2606_01547_b200 import build as _b
    _b.build()
    import paper_2606_01547_b200 as jt_mod
    jt_mod.lib()
    return jt_mod


def to_dev(a, dtype):
    """numpy float64 values -> CUDA tensor of the call's dtype ("f32"/"f64")."""
    import numpy as np
    import torch
    t = torch.float32 if dtype == "f32" else torch.float64
    return torch.as_tensor(np.ascontiguousarray(a), dtype=t, device="cuda").contiguous()


def gpu_simulate(jt, w, method="auto", conv=True):
    """Runs jt_simulate_image on a workloads.Workload; returns a float64 numpy image."""
    g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
    tn = to_dev(w.tnfw, w.dtype) if w.n_tnfw > 0 else None
    psf = to_dev(w.psf, w.dtype) if conv else None
    out = jt.simulate_image(g, w.sie, w.shear, tn, w.sources, psf, dtype=w.dtype, method=method)
    return out.double().cpu().numpy()
