"""jt_ray_shoot_noalloc -- ray-shooting for callers that cannot allocate device memory (include/jt.h).

Some users of libjt call it from a place where cudaMalloc is off limits: a custom-call / plug-in callback of a host
framework that hands over finished input and output buffers and forbids allocation, or a process whose memory pool has
already taken the whole GPU.  They cannot give jt_ray_shoot its workspace.  jt_ray_shoot_noalloc runs the same kernels on
a fixed 32 MiB scratch array built into the library.  This file checks that it returns what jt_ray_shoot returns, on
two calls in a row (the second smaller than the first, so anything the first call left in the shared array would show),
in both dtypes, with the subhalo list split over thread blocks (partial sums + arrival counters in the scratch) and
unsplit (records only), and that a problem too large for the array is refused without touching the outputs.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
"""
import ctypes

import numpy as np
import pytest
import torch

from conftest import to_dev


def _inputs(seed, n, M, dtype):
    rng = np.random.default_rng(seed)
    tx, ty = rng.uniform(-1.5, 1.5, n), rng.uniform(-1.5, 1.5, n)
    tn = np.empty((5, M))
    tn[0], tn[1] = rng.uniform(-2.0, 2.0, M), rng.uniform(-2.0, 2.0, M)
    tn[2] = 10.0 ** rng.uniform(np.log10(0.005), np.log10(0.05), M)          # Rs, BASELINE.json config 2 priors
    tn[3] = 10.0 ** rng.uniform(-4.0, -2.0, M)                               # alpha_Rs
    tn[4] = 5.0 * tn[2]                                                      # r_trunc
    if dtype == "f32":
        tx, ty, tn = (np.float32(a).astype(np.float64) for a in (tx, ty, tn))
    return tx, ty, tn


# (rays, subhalos): split list; a smaller split list right after it; records only (many rays, few subhalos); no subhalos
CASES = [(5000, 3000), (3001, 1500), (40000, 200), (777, 0)]
SIE, SHEAR = (1.1, 0.12, -0.07, 0.02, -0.01), (0.03, -0.02)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_noalloc_matches_ray_shoot_on_consecutive_calls(jt, orc, dtype):
    tol = 2e-12 if dtype == "f64" else 4e-7          # the tolerances of test_gpu_parity.test_ray_shoot_random
    cap = jt.ray_shoot_noalloc_capacity()
    assert cap == 32 << 20
    got, want, inputs = [], [], []
    # all no-alloc calls first, back to back on one stream, so call k+1 really runs on what call k left in the array
    for k, (n, M) in enumerate(CASES):
        tx, ty, tn = _inputs(900 + k, n, M, dtype)
        assert jt.ray_shoot_workspace_bytes(dtype, n, M) <= cap
        dx, dy = to_dev(tx, dtype), to_dev(ty, dtype)
        dtn = to_dev(tn, dtype) if M else None
        bx, by = torch.full_like(dx, float("nan")), torch.full_like(dy, float("nan"))      # outputs are the caller's
        jt.ray_shoot_noalloc(dx, dy, bx, by, SIE, SHEAR, dtn)
        got.append((bx, by))
        inputs.append((dx, dy, dtn, tx, ty, tn))
    for dx, dy, dtn, *_ in inputs:                    # the existing path, caller-allocated workspace
        want.append(jt.ray_shoot(dx, dy, SIE, SHEAR, dtn))
    torch.cuda.synchronize()
    for (bx, by), (wx, wy), (n, M) in zip(got, want, CASES):
        for a, w in ((bx, wx), (by, wy)):
            a, w = a.double().cpu().numpy(), w.double().cpu().numpy()
            assert np.isfinite(a).all(), (n, M)
            assert np.max(np.abs(a - w)) < tol, (n, M)
    # and, for the two split-list calls, against the oracle itself (the macro lens is double in both dtype modes)
    for k in (0, 1):
        _, _, _, tx, ty, tn = inputs[k]
        ox, oy = orc.ray_shoot(tx, ty, SIE, SHEAR, tn)
        assert np.max(np.abs(got[k][0].double().cpu().numpy() - ox)) < tol
        assert np.max(np.abs(got[k][1].double().cpu().numpy() - oy)) < tol


@pytest.mark.gpu
def test_noalloc_refuses_what_does_not_fit(jt):
    """160,000 rays through 50,000 subhalos in double need 49.8 MB of scratch: JT_ERR_WORKSPACE, outputs untouched."""
    n, M = 160000, 50000
    assert jt.ray_shoot_workspace_bytes("f64", n, M) > jt.ray_shoot_noalloc_capacity()
    tx, ty, tn = _inputs(5, n, M, "f64")
    dx, dy, dtn = to_dev(tx, "f64"), to_dev(ty, "f64"), to_dev(tn, "f64")
    bx, by = torch.full_like(dx, -7.0), torch.full_like(dy, -7.0)
    with pytest.raises(jt.JtError) as e:
        jt.ray_shoot_noalloc(dx, dy, bx, by, SIE, SHEAR, dtn)
    assert e.value.status == 3 and "built-in array" in str(e.value)
    # the C entry point itself says the same (the binding's check above is only there for the message)
    from paper_2606_01547_b200 import binding as b
    L = b._lens(b.JT_F64, SIE, SHEAR, dtn)
    rc = jt.lib().jt_ray_shoot_noalloc(b.JT_F64, n, ctypes.c_void_p(dx.data_ptr()), ctypes.c_void_p(dy.data_ptr()), ctypes.byref(L),
                                       ctypes.c_void_p(bx.data_ptr()), ctypes.c_void_p(by.data_ptr()), None)
    assert rc == 3
    torch.cuda.synchronize()
    assert bool((bx == -7.0).all()) and bool((by == -7.0).all())
