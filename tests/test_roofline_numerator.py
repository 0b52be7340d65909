"""bench.py's roofline numerator against the built library (no GPU needed).

`roofline.frac` = evaluations x TIER_COST (binding-pipe instructions per evaluation, per class of definition T) / time / peak.
TIER_COST is a table of literals in bench.py; this test recounts it from the SASS of the libjt.so the bench would load, so a
kernel edit that changes a class loop fails here instead of silently making `frac` stale (
profiles/r02_sass_loops.md shows the same loops by hand).

What is recounted: the three far-far series loops and the near (mid form) loop of k_trace<T, 8, GRID>, for both dtypes
-- five of the six classes (the cold class is charged like mid).  NOT recounted: the far form (f32 29.6, f64 50.6).  It is
inlined in the class loop beside the out-of-line near call and has no loop of its own; its figure is a count of the source
(profiles/r02_sass_loops.md, paragraph "far form") and carries 3-6 % of the evaluations of the configs.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


@pytest.fixture(scope="module")
def sass(jt):
    from paper_2606_01547_b200 import sass_loops
    return sass_loops


def _innermost(sass, kernel):
    return [(n, h) for n, inner, h in sass.loop_table(kernel) if inner == 0]


def test_tier_cost_f64_matches_sass(sass):
    import bench
    R = 8                                                   # rays per thread of k_trace<double, 8, GRID>
    loops = _innermost(sass, "k_trace<double, (int)8, (bool)1>")
    # far-far: one record x R rays per iteration, one MUFU (reciprocal seed) per ray, pure FP64 arithmetic
    farfar = sorted(sass.fp64_ops(h) for n, h in loops if h["MUFU"] == R and sass.fp64_ops(h) > 100 and sass.fp32_lane_ops(h) == 0)
    assert len(farfar) == 3, farfar
    long_, mid_, short_ = bench.TIER_COST["f64"][:3]
    assert [c / R for c in farfar] == [short_, mid_, long_], (farfar, bench.TIER_COST["f64"])
    # near: the mid form on two rays per iteration (5 MUFU per ray)
    near = [sass.fp64_ops(h) for n, h in loops if h["MUFU"] == 10 and sass.fp64_ops(h) > 100]
    assert len(near) == 1 and near[0] / 2 == bench.TIER_COST["f64"][4] == bench.TIER_COST["f64"][5], near


def test_tier_cost_f32_matches_sass(sass):
    import bench
    R = 8
    loops = _innermost(sass, "k_trace<float, (int)8, (bool)1>")
    # far-far: TWO records x R rays per iteration (packed FFMA2 on ray pairs): 2R MUFU; lane-ops count a packed op twice
    farfar = sorted(sass.fp32_lane_ops(h) for n, h in loops if h["MUFU"] == 2 * R and sass.fp64_ops(h) == 0)
    assert len(farfar) == 3, farfar
    long_, mid_, short_ = bench.TIER_COST["f32"][:3]
    assert [c / (2 * R) for c in farfar] == [short_, mid_, long_], (farfar, bench.TIER_COST["f32"])
    assert any(h["FFMA2"] > 0 for n, h in loops if h["MUFU"] == 2 * R)              # the packed path is what is counted
    near = [sass.fp32_lane_ops(h) for n, h in loops if h["MUFU"] == 10 and sass.fp64_ops(h) == 0 and h["LDS"] == 0]
    assert len(near) == 1 and near[0] / 2 == bench.TIER_COST["f32"][4] == bench.TIER_COST["f32"][5], near


def test_batch_kernel_runs_the_same_series_loops(sass):
    """k_batch (C3) is charged with the same per-evaluation costs: its far-far loops take one record x 8 rays."""
    import bench
    loops = _innermost(sass, "k_batch<float, (int)8, (int)2>")
    costs = sorted({sass.fp32_lane_ops(h) / 8 for n, h in loops if h["MUFU"] == 8 and sass.fp64_ops(h) == 0 and h["FFMA2"] > 0})
    assert costs == sorted(bench.TIER_COST["f32"][:3]), costs
