"""Host-side checks that need no GPU: libjt.so builds, loads, exports every symbol include/jt.h declares,
and rejects bad arguments before touching the device (error behaviour documented in include/jt.h)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
JT_VERSION_EXPECTED = 200


def _declared(header, macro):
    src = open(os.path.join(ROOT, "include", header)).read()
    return sorted(set(re.findall(macro + r"[^;(]*?\b(jt_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported(jt):
    """Every function include/*.h declares is exported by the library that header describes."""
    assert sorted(f for f in os.listdir(os.path.join(ROOT, "include")) if f.endswith(".h")) == ["jt.h", "jt_probe.h"]
    names = _declared("jt.h", "JT_API")
    assert {"jt_ray_shoot", "jt_source_brightness", "jt_psf_convolve", "jt_simulate_image", "jt_simulate_batch",
            "jt_psf_convolve_batch"} <= set(names), names
    L = ctypes.CDLL(jt.lib_path())
    for n in names:
        assert hasattr(L, n), n
    assert not hasattr(L, "jt_probe_alu")              # measurement probes live in their own library
    P = ctypes.CDLL(jt.probe_lib_path())
    assert _declared("jt_probe.h", "JT_PROBE_API") == ["jt_probe_alu"]
    assert hasattr(P, "jt_probe_alu")
    assert jt.version() == JT_VERSION_EXPECTED


def test_status_strings(jt):
    L = jt.lib()
    assert L.jt_status_string(0) == b"JT_OK" and L.jt_status_string(3) == b"JT_ERR_WORKSPACE"


def test_argument_validation_without_device(jt):
    from paper_2606_01547_b200 import binding as b
    L = jt.lib()
    g = b._Grid(10, 10, 0.05, 0.0, 0.0, 1)
    lens = b._Lens()
    S, keep = b._sources([[1, 0.2, 1.0, 0, 0, 0, 0]])
    dummy = ctypes.c_void_p(256)
    # unknown dtype / method
    assert L.jt_simulate_image(7, ctypes.byref(g), ctypes.byref(lens), ctypes.byref(S), 0, 0, None, 0, None, 0, dummy, None) == 2
    assert L.jt_psf_convolve(0, 8, 8, dummy, 3, 3, dummy, 9, None, 0, ctypes.c_void_p(512), None) == 2
    # even kernel, null pointers, aliasing, bad grid
    assert L.jt_psf_convolve(0, 8, 8, dummy, 4, 3, dummy, 1, None, 0, ctypes.c_void_p(512), None) == 1
    assert L.jt_psf_convolve(0, 8, 8, None, 3, 3, dummy, 1, None, 0, ctypes.c_void_p(512), None) == 1
    assert L.jt_psf_convolve(0, 8, 8, dummy, 3, 3, dummy, 1, None, 0, dummy, None) == 1
    bad = b._Grid(10, 10, -1.0, 0.0, 0.0, 1)
    assert L.jt_simulate_image(0, ctypes.byref(bad), ctypes.byref(lens), ctypes.byref(S), 0, 0, None, 0, None, 0, dummy, None) == 1
    bad = b._Grid(10, 10, 0.05, 0.0, 0.0, 17)
    assert L.jt_simulate_image(0, ctypes.byref(bad), ctypes.byref(lens), ctypes.byref(S), 0, 0, None, 0, None, 0, dummy, None) == 1
    lens.n_tnfw = 5          # subhalos announced but no arrays
    assert L.jt_ray_shoot(1, 10, dummy, dummy, ctypes.byref(lens), None, 0, ctypes.c_void_p(512), ctypes.c_void_p(768), None) == 1
    lens.n_tnfw = 0
    assert L.jt_ray_shoot(1, -1, dummy, dummy, ctypes.byref(lens), None, 0, ctypes.c_void_p(512), ctypes.c_void_p(768), None) == 1
    # workspace too small: the direct path needs its tap table (+ partial sums when the kernel columns are split over
    # CTAs), the FFT path its complex plane
    L.jt_psf_convolve_batch_workspace_bytes.restype = ctypes.c_size_t
    need = L.jt_psf_convolve_workspace_bytes(1, 64, 64, 21, 21, 1)
    assert need >= 21 * 21 * 8
    assert L.jt_psf_convolve(1, 64, 64, dummy, 21, 21, dummy, 1, dummy, need - 1, ctypes.c_void_p(512), None) == 3
    assert L.jt_psf_convolve_batch_workspace_bytes(1, ctypes.c_int64(1), 64, 64, 21, 21, 1) == need
    assert L.jt_psf_convolve_batch(1, ctypes.c_int64(0), 64, 64, None, 21, 21, None, 1, None, 0, None, None) == 0     # B = 0: no-op
    assert L.jt_psf_convolve_batch(1, ctypes.c_int64(-1), 64, 64, dummy, 21, 21, dummy, 1, None, 0, ctypes.c_void_p(512), None) == 1
    need = L.jt_psf_convolve_workspace_bytes(1, 64, 64, 21, 21, 2)
    assert need >= (64 + 64 + 21) * (84 // 2 + 1) * 16        # three half-spectrum planes of the 84 x 84 padded transform
    assert L.jt_psf_convolve(1, 64, 64, dummy, 21, 21, dummy, 2, dummy, need - 1, ctypes.c_void_p(512), None) == 3
    assert L.jt_psf_convolve(1, 64, 64, dummy, 21, 21, dummy, 2, None, 0, ctypes.c_void_p(512), None) == 3
    # a workspace that is only 8-byte aligned is refused by both methods (double2 / complex accesses would fault)
    for m in (1, 2):
        need = L.jt_psf_convolve_workspace_bytes(1, 64, 64, 21, 21, m)
        assert L.jt_psf_convolve(1, 64, 64, dummy, 21, 21, dummy, m, ctypes.c_void_p(4096 + 8), need, ctypes.c_void_p(512), None) == 1
        assert L.jt_psf_convolve_batch(1, ctypes.c_int64(1), 64, 64, dummy, 21, 21, dummy, m, ctypes.c_void_p(4096 + 8), need,
                                       ctypes.c_void_p(512), None) == 1
    # zero-sized problems are no-ops
    assert L.jt_ray_shoot(1, 0, None, None, ctypes.byref(lens), None, 0, None, None, None) == 0
    del keep


def test_workspace_queries_are_consistent(jt):
    g = jt.Grid(200, 200, 0.04, supersample=2)
    big = jt.simulate_image_workspace_bytes("f32", g, 10000, 21, 21, "direct")
    small = jt.simulate_image_workspace_bytes("f32", g, 0, 21, 21, "direct")
    assert big > small >= 200 * 200 * 4
    assert jt.ray_shoot_workspace_bytes("f64", 10 ** 7, 0) == 0          # no subhalos: no records, no split, no scratch
    rec = jt.ray_shoot_workspace_bytes("f64", 10 ** 7, 100)              # enough ray tiles: no split, only the derived records
    assert 100 * 8 * 16 <= rec <= 100 * 8 * 32 + 256
    assert jt.ray_shoot_workspace_bytes("f64", 1000, 10 ** 5) > 0


def test_no_cpu_fallback_without_device(jt):
    """On a box without a CUDA device a compute call must fail (JT_ERR_CUDA / UNSUPPORTED), never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2606_01547_b200 import binding as b
    L = jt.lib()
    lens = b._Lens()
    st = L.jt_ray_shoot(1, 4, ctypes.c_void_p(256), ctypes.c_void_p(512), ctypes.byref(lens), None, 0,
                        ctypes.c_void_p(768), ctypes.c_void_p(1024), None)
    assert st in (2, 4)


def test_noalloc_entry_point_limit_without_device(jt):
    """jt_ray_shoot_noalloc (for callers that cannot allocate device memory) refuses, before touching any device, a
    problem whose scratch does not fit its built-in 32 MiB array, and validates its arguments like jt_ray_shoot."""
    from paper_2606_01547_b200 import binding as b
    L = jt.lib()
    cap = L.jt_ray_shoot_noalloc_capacity()
    assert cap == 32 << 20
    dummy = [ctypes.c_void_p(256 * (k + 1)) for k in range(9)]
    lens = b._Lens()
    lens.n_tnfw = 50000
    lens.tnfw_cx, lens.tnfw_cy, lens.tnfw_Rs, lens.tnfw_alpha_Rs, lens.tnfw_r_trunc = [d.value for d in dummy[4:9]]
    assert L.jt_ray_shoot_workspace_bytes(1, 160000, 50000) > cap
    assert L.jt_ray_shoot_noalloc(1, 160000, dummy[0], dummy[1], ctypes.byref(lens), dummy[2], dummy[3], None) == 3
    assert L.jt_ray_shoot_noalloc(7, 10, dummy[0], dummy[1], ctypes.byref(lens), dummy[2], dummy[3], None) == 2
    assert L.jt_ray_shoot_noalloc(1, -1, dummy[0], dummy[1], ctypes.byref(lens), dummy[2], dummy[3], None) == 1
    assert L.jt_ray_shoot_noalloc(1, 10, dummy[0], dummy[1], ctypes.byref(lens), dummy[0], dummy[3], None) == 1   # aliasing
    assert L.jt_ray_shoot_noalloc(1, 0, None, None, ctypes.byref(lens), None, None, None) == 0                     # no-op
    lens.tnfw_Rs = None
    assert L.jt_ray_shoot_noalloc(1, 10, dummy[0], dummy[1], ctypes.byref(lens), dummy[2], dummy[3], None) == 1


def test_plan_queries_without_device(jt):
    """jt_psf_convolve_plan / jt_trace_plan_query are host-only: every launch shape the library has is reachable and named
    (the GPU parity tests assert these same plans on the cases they run)."""
    seen = set()
    for dtype in ("f64", "f32"):
        for shape in [(60, 60, 11, 11), (100, 100, 31, 31), (130, 75, 45, 45), (180, 180, 135, 135), (500, 500, 101, 101)]:
            p = jt.psf_convolve_plan(dtype, *shape, method="direct")
            seen.add((p["path"], p["tma"], p["z_split"] > 1, p["row_bands"] > 1))
            assert jt.psf_convolve_plan(dtype, *shape, method="fft")["path"] == "fft"
            assert jt.psf_convolve_plan(dtype, *shape, method="auto")["est_us"] <= p["est_us"] * (1 + 1e-12)
        p = jt.psf_convolve_plan(dtype, 16, 20, 5, 5, method="direct", B=130)
        seen.add((p["path"], p["tma"], p["z_split"] > 1, p["row_bands"] > 1))
    assert {("small", 0, False, False), ("tile", 1, True, False), ("tile", 0, True, False), ("tile", 1, True, True),
            ("tile", 1, False, False)} <= seen, seen
    g = jt.Grid(200, 200, 0.04, supersample=2)
    p = jt.trace_plan("f32", g, n_tnfw=10000)
    assert p["n_chunks"] > 1 and p["n_ctas"] % p["n_chunks"] == 0 and p["chunk_len"] * p["n_chunks"] >= 10000
    assert jt.trace_plan("f64", jt.Grid(500, 500, 0.02, supersample=5), n_tnfw=50000)["wide"] == 1
    assert jt.trace_plan("f64", jt.Grid(60, 60, 0.05), n_tnfw=0)["rays_per_thread"] == 1
    assert jt.trace_plan("f64", None, n_rays=1000, n_tnfw=0)["rays_per_thread"] == 8
    L = jt.lib()
    assert L.jt_psf_convolve_plan(0, 1, 8, 8, 4, 3, 0, None, None) == 1
    assert L.jt_trace_plan_query(0, None, 0, 0, None) == 1
