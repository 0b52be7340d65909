#!/usr/bin/env python
"""bench.py -- throughput of the lensed-image hot path on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2-f64] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A step is ONE pass of the whole hot path (grid -> ray-shoot through every deflector -> Sersic -> bin ->
PSF convolution) through jt_simulate_image (single systems) or
jt_simulate_batch (C3) on seeded synthetic inputs (workloads/).
`value` = ray x deflector evaluations per second, inputs resident in HBM (BASELINE.json:metric);
`e2e`   = the same with the step's inputs copied from pinned host memory and the image copied back,
          both inside the timed region;
`roofline` = the dominant kernel (the ray-tracing kernel) against the issue-limited ALU peak derived in
          DESIGN.md "Rooflines", its duration measured live with CUDA events recorded by the library on
          the launch stream (jt_profile_enable);
`cpu_baseline` = the oracle, as it stands, on this box's host cores on a bounded sample of the same workload.
With N > 1 every rank runs its own replica of the workload (replicas only, no
collective on the data path); the time is the max over ranks and the value the sum of the units.
`--impl reference` times the oracle instead (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ray_deflector_evals_per_s"
UNIT = "evals/s"
SM_COUNT = 148
# Algorithmic work per evaluation on the binding unit, counted in the SASS of each class loop
# (`python -m paper_2606_01547_b200.sass_loops`, output and the arithmetic in profiles/r02_sass_loops.md): loop body count
# of the pipe's opcodes / (records per iteration x rays per thread).  f32: FP32-pipe lane operations (a packed FFMA2 /
# FMUL2 / FADD2 counts as two: it holds the pipe for two cycles); f64: FP64-pipe instructions.  Order: far-far series at
# its three lengths (longest first), far form, near form on a warp tile outside / inside X^2 = 2 (both run the mid form
# on every ray; the per-ray generic fix-up inside is not counted).  The mix of classes is measured per run with
# jt_profile_tiers.  tests/test_roofline_numerator.py recounts the far-far and near entries from the built library's SASS
# on every CPU test run, so they cannot go stale; the far entry (29.6 / 50.6) is a count of the source (the form is inlined,
# it has no loop of its own) and weighs 3-7 % of the evaluations.
TIER_COST = {"f32": (13.25, 10.25, 9.25, 29.6, 36.0, 36.0), "f64": (23.25, 19.25, 17.25, 50.6, 77.0, 77.0)}
TIER_NAMES = ("far_far_long", "far_far_mid", "far_far_short", "far", "mid", "cold")
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the ncu --set full captures in
# profiles/r02_ncu_{c4f64,c2f64,c2f32,c3f32}.txt (the kernels are ALU-bound: compulsory traffic is the records in, the
# image out and, for C2, the partial sums of the split subhalo list)
NCU_TRAFFIC_BYTES = {"C4-f64": 11405568 + 4258048, "C2-f64": 2339072 + 784384, "C2-f32": 1172992 + 382208,
                     "C3-f32": 15794688 + 36633088}
ALU_LANES_PER_SM = {"f32": 128, "f64": 64}
WORKLOADS = ("C0-f64", "C1-f64", "C2-f32", "C2-f64", "C3-f32", "C4-f64")
PER_CONFIG = ("C2-f64", "C2-f32", "C3-f32")        # reported beside the headline workload in the same JSON line


# ------------------------------------------------------------------ distributed plumbing
def dist_init(n_gpus, backend=None):
    """Returns (rank, world, local_rank).  Single process when WORLD_SIZE is unset."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, 0
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if backend is None:
        import torch
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    if not dist.is_initialized():
        dist.init_process_group(backend=backend)
    return dist.get_rank(), dist.get_world_size(), int(os.environ.get("LOCAL_RANK", "0"))


def aggregate(units_local, ms_local, device=None):
    """Whole-job numbers: (sum of units over ranks, max of time over ranks).  No data-path collective exists;
    this is the only communication of the run."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(units_local), float(ms_local)
    dev = device if device is not None else ("cuda" if dist.get_backend() == "nccl" else "cpu")
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def shard_range(n, rank, world):
    """Contiguous, balanced [lo, hi) share of n independent units (systems of a batch) for `rank`."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


# ------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])), mx.append(float(f[1])), pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # samples under load = upper half of the clock samples (idle samples precede the first launch)
        return {"sm_mhz": float(np.median(sm)), "sm_mhz_max_seen": float(max(sm)), "sm_max_mhz": float(max(mx)),
                "power_w_max": float(max(pw)), "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------ workloads
def make_workload(name, rank=0):
    """BASELINE.json:configs[i] by name ("C2-f64", ...).  Rank r > 0 gets the same recipe with seed + r
    (an independent replica of the same shape)."""
    import workloads
    cfg, dtype = name.split("-")
    mk = {"C0": workloads.config_c0, "C1": workloads.config_c1, "C2": workloads.config_c2,
          "C3": workloads.config_c3, "C4": workloads.config_c4}[cfg]
    return mk(dtype=dtype, seed_offset=7919 * rank)


def describe(name, w, world):
    d = {"workload": name, "grid": "%dx%d" % (w.nx, w.ny), "pixel_scale": w.pixel_scale,
         "supersample": w.supersample, "n_tnfw": w.n_tnfw, "psf": "%dx%d" % w.psf.shape[-2:],
         "evals_per_step_per_gpu": int(w.evals), "l2": "256 MiB buffer rewritten between timed steps",
         "parallelism": "replicas x%d (no data-path collective)" % world}
    if hasattr(w, "B"):
        d["batch"] = w.B
    return d


class ImageRunner:
    """One lens system through jt_simulate_image; device buffers, workspace and output allocated once."""

    def __init__(self, jt, w, method="auto"):
        import torch
        self.jt, self.w, self.method = jt, w, method
        self.tdt = torch.float32 if w.dtype == "f32" else torch.float64
        self.grid = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
        # pinned host copies (e2e leg) and resident device copies (device-timed leg)
        self.h_tnfw = torch.as_tensor(np.ascontiguousarray(w.tnfw), dtype=self.tdt).pin_memory()
        self.h_psf = torch.as_tensor(np.ascontiguousarray(w.psf), dtype=self.tdt).pin_memory()
        self.d_tnfw = self.h_tnfw.to("cuda")
        self.d_psf = self.h_psf.to("cuda")
        self.out = torch.empty((w.ny, w.nx), dtype=self.tdt, device="cuda")
        self.h_out = torch.empty((w.ny, w.nx), dtype=self.tdt).pin_memory()
        nb = jt.simulate_image_workspace_bytes(w.dtype, self.grid, w.n_tnfw, w.psf.shape[0], w.psf.shape[1], method)
        self.ws = torch.empty(max(nb, 1), dtype=torch.uint8, device="cuda")
        self.h2d = self.h_tnfw.numel() * self.h_tnfw.element_size() + self.h_psf.numel() * self.h_psf.element_size()
        self.d2h = self.h_out.numel() * self.h_out.element_size()
        self.images = 1

    def step(self):
        tn = self.d_tnfw if self.w.n_tnfw > 0 else None
        self.jt.simulate_image(self.grid, self.w.sie, self.w.shear, tn, self.w.sources, self.d_psf,
                               dtype=self.w.dtype, method=self.method, workspace=self.ws, out=self.out)

    def step_e2e(self):
        self.d_tnfw.copy_(self.h_tnfw, non_blocking=True)
        self.d_psf.copy_(self.h_psf, non_blocking=True)
        self.step()
        self.h_out.copy_(self.out, non_blocking=True)


class BatchRunner:
    """B independent systems through jt_simulate_batch (C3)."""

    def __init__(self, jt, w):
        import torch
        self.jt, self.w = jt, w
        self.tdt = torch.float32 if w.dtype == "f32" else torch.float64
        self.grid = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
        pin = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=self.tdt).pin_memory()
        self.h = [pin(w.sie), pin(w.shear), pin(w.tnfw), pin(w.sources), pin(w.psf)]
        self.d = [t.to("cuda") for t in self.h]
        self.out = torch.empty((w.B, w.ny, w.nx), dtype=self.tdt, device="cuda")
        self.h_out = torch.empty((w.B, w.ny, w.nx), dtype=self.tdt).pin_memory()
        self.h2d = sum(t.numel() * t.element_size() for t in self.h)
        self.d2h = self.h_out.numel() * self.h_out.element_size()
        self.images = w.B

    def step(self):
        self.jt.simulate_batch(self.grid, *self.d, out=self.out)

    def step_e2e(self):
        """Pinned host -> device -> kernel -> pinned host, the batch cut into slices dealt to two streams so that the
        67 MB of images of slice i go back over PCIe while slice i + 1 is being simulated (systems are independent:
        a slice is just a smaller jt_simulate_batch call on views of the same buffers)."""
        import torch
        if not hasattr(self, "streams"):
            self.streams = [torch.cuda.Stream(), torch.cuda.Stream()]
            n = min(8, self.w.B)
            edges = [round(i * self.w.B / n) for i in range(n + 1)]
            self.slices = [(a, b) for a, b in zip(edges[:-1], edges[1:]) if b > a]
        cur = torch.cuda.current_stream()
        for st in self.streams:
            st.wait_stream(cur)
        for i, (a, b) in enumerate(self.slices):
            st = self.streams[i % 2]
            with torch.cuda.stream(st):
                for d, h in zip(self.d, self.h):
                    d[a:b].copy_(h[a:b], non_blocking=True)
                self.jt.simulate_batch(self.grid, *[d[a:b] for d in self.d], out=self.out[a:b], stream=st)
                self.h_out[a:b].copy_(self.out[a:b], non_blocking=True)
        for st in self.streams:
            cur.wait_stream(st)


# ------------------------------------------------------------------ the oracle on the host cores
def oracle_sample(w, target_evals=2.0e8):
    """A bounded sample of the workload for the CPU oracle: pixel rows spread evenly over the image (single
    systems) or the first systems of the batch, sized to about target_evals ray x deflector evaluations."""
    if hasattr(w, "B"):
        per = w.n_rays * (w.n_tnfw + 2)
        n = int(max(1, min(w.B, round(target_evals / per))))
        return {"kind": "systems", "systems": list(range(n)), "evals": n * per,
                "text": "first %d of %d systems, whole pipeline" % (n, w.B)}
    per_row = w.nx * w.supersample ** 2 * w.n_deflectors
    n = int(max(1, min(w.ny, round(target_evals / per_row))))
    rows = sorted(set(int(round(x)) for x in np.linspace(0, w.ny - 1, n)))
    return {"kind": "rows", "rows": rows, "evals": len(rows) * per_row,
            "text": "%d of %d pixel rows (all %d deflectors, all sub-rays) + one full-size %dx%d direct convolution"
                    % (len(rows), w.ny, w.n_deflectors, w.psf.shape[0], w.psf.shape[1])}


def oracle_step(orc, w, sample):
    """One pass of the oracle over the sample; returns seconds."""
    t0 = time.perf_counter()
    if sample["kind"] == "systems":
        orc.simulate_batch(w, systems=sample["systems"])
    else:
        img = np.zeros((w.ny, w.nx))
        for j in sample["rows"]:
            img[j] = orc.prepsf_rows(w, j, j + 1)[0]
        orc.convolve(img, w.psf)
    return time.perf_counter() - t0


def cpu_baseline(w, target_evals):
    import oracle as orc
    orc.build()
    cores = len(os.sched_getaffinity(0))
    orc.set_threads(cores)
    sample = oracle_sample(w, target_evals)
    sec = oracle_step(orc, w, sample)
    # the same oracle on ONE core, on a sample cores times smaller (both numbers are reported)
    orc.set_threads(1)
    s1 = oracle_sample(w, target_evals / max(cores, 1))
    sec1 = oracle_step(orc, w, s1)
    orc.set_threads(cores)
    return {"value": sample["evals"] / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": sample["text"], "seconds": sec,
            "single_core": {"value": s1["evals"] / sec1, "sample": s1["text"], "seconds": sec1}}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on this box's host cores (rank 0 only)."""
    if rank != 0:
        return
    w = make_workload(args.workload, 0)
    import oracle as orc
    orc.build()
    cores = len(os.sched_getaffinity(0))
    orc.set_threads(cores)
    sample = oracle_sample(w, args.ref_evals)
    for _ in range(args.warmup):
        oracle_step(orc, w, sample)
    secs = [oracle_step(orc, w, sample) for _ in range(args.steps)]
    total = sum(secs)
    value = sample["evals"] * args.steps / total
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": describe(args.workload, w, 1),
            # ms_per_step is the time of ONE SAMPLED step (evals_per_step_sampled evaluations), not of the whole workload
            # config.evals_per_step_per_gpu describes (config is kept identical to our arm's on purpose)
            "evals_per_step_sampled": int(sample["evals"]),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample["text"],
                             "evals_per_step_sampled": int(sample["evals"])},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ our arm
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def graph_time(torch, call, n_rep=20, repeats=3):
    """Device time per call in microseconds: n_rep back-to-back calls captured into a CUDA graph on a side stream, the
    replay timed with CUDA events (best of `repeats`) -- no Python / ctypes cost inside the number."""
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        for _ in range(3):
            call()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            for _ in range(n_rep):
                call()
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    best = None
    for _ in range(repeats):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        g.replay()
        b.record()
        b.synchronize()
        t = 1e3 * a.elapsed_time(b) / n_rep
        best = t if best is None else min(best, t)
    return best


def fft_conv_bytes(ny, nx, ky, kx, esz):
    """Algorithmic bytes of the FFT convolution: image in and out, kernel in, and the three
    half-spectrum planes of complex doubles, each written once and read once (SA [ny][Ph], SB [ky][Ph], SC [ny][Ph])."""
    def smooth(v, even):
        p = max(v, 2)
        while True:
            q = p
            for f in (2, 3, 5):
                while q % f == 0:
                    q //= f
            if q == 1 and not (even and p % 2):
                return p
            p += 1
    Px, Py = smooth(nx + kx - 1, True), smooth(ny + ky - 1, False)
    Ph = Px // 2 + 1
    return (2 * nx * ny + ky * kx) * esz + 2 * 16 * Ph * (2 * ny + ky), (Py, Px)


def conv_block(torch, jt, w, peaks, probes):
    """jt_psf_convolve alone on this workload's image and PSF shape, BOTH methods (CUDA-graph replay, device time per
    call), each against its own roofline: direct -> FMA peak of the dtype, FFT -> measured HBM bandwidth."""
    tdt = torch.float32 if w.dtype == "f32" else torch.float64
    esz = 4 if w.dtype == "f32" else 8
    lanes = ALU_LANES_PER_SM[w.dtype]
    ky, kx = w.psf.shape[-2:]
    psf = w.psf if w.psf.ndim == 2 else w.psf[0]
    rng = np.random.default_rng(154710)
    img = torch.as_tensor(rng.uniform(0.0, 1.0, (w.ny, w.nx)), dtype=tdt, device="cuda")
    ker = torch.as_tensor(np.ascontiguousarray(psf), dtype=tdt, device="cuda")
    out = torch.empty_like(img)
    fma = w.nx * w.ny * ky * kx
    fma_peak = SM_COUNT * lanes * peaks.get("sm_max_mhz", 1965.0) * 1e6
    nbytes, pad = fft_conv_bytes(w.ny, w.nx, ky, kx, esz)
    blk = {"shape": "%dx%d image, %dx%d kernel" % (w.ny, w.nx, ky, kx), "dtype": w.dtype,
           "auto_picks": jt.psf_convolve_plan(w.dtype, w.ny, w.nx, ky, kx, "auto")["method"],
           "direct_plan": {k: v for k, v in jt.psf_convolve_plan(w.dtype, w.ny, w.nx, ky, kx, "direct").items()
                           if k in ("path", "tma", "z_split", "row_bands", "oy", "warps")}}
    for method in ("direct", "fft"):
        try:
            ws = torch.empty(max(jt.psf_convolve_workspace_bytes(w.dtype, w.ny, w.nx, ky, kx, method), 1),
                             dtype=torch.uint8, device="cuda")
            us = graph_time(torch, lambda: jt.psf_convolve(img, ker, method=method, workspace=ws, out=out))
        except jt.JtError as e:
            blk[method] = {"error": str(e)}
            continue
        d = {"us": us, "gbs_algorithmic_io": (2 * w.nx * w.ny + ky * kx) * esz / (us * 1e-6) / 1e9}
        if method == "direct":
            meas = 2 * probes["ffma2"] if w.dtype == "f32" else probes["dfma"]
            d.update({"bound": "alu", "fma_per_s": fma / (us * 1e-6), "frac_of_derived_fma_peak": fma / (us * 1e-6) / fma_peak,
                      "frac_of_measured_fma_rate": fma / (us * 1e-6) / meas})
        else:
            d.update({"bound": "hbm", "bytes": nbytes, "pad": "%dx%d" % pad, "gbs": nbytes / (us * 1e-6) / 1e9,
                      "frac_of_measured_hbm": nbytes / (us * 1e-6) / 1e9 / peaks.get("hbm_gbs", 6650.0)})
        blk[method] = d
    return blk


def latency_block(torch, jt):
    """The launch-latency-bound configs C0 and C1 (parity configs, roofline fractions not
    meaningful): microseconds per image, device time from a CUDA-graph replay of 20 jt_simulate_image calls, and wall
    time per call through the Python binding (ctypes marshalling included)."""
    out = {}
    for name in ("C0-f64", "C1-f64"):
        r = ImageRunner(jt, make_workload(name, 0), "auto")
        us = graph_time(torch, r.step)
        for _ in range(20):
            r.step()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(200):
            r.step()
        torch.cuda.synchronize()
        wall = 1e6 * (time.perf_counter() - t0) / 200
        # the same call with the marshalling done once (binding.PreparedImage: one ctypes call per image)
        prep = jt.PreparedImage(r.grid, r.w.sie, r.w.shear, r.d_tnfw if r.w.n_tnfw else None, r.w.sources, r.d_psf,
                                dtype=r.w.dtype, method="auto", workspace=r.ws, out=r.out)
        for _ in range(20):
            prep()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(200):
            prep()
        torch.cuda.synchronize()
        out[name] = {"device_us_per_image_graph_replay": us, "python_call_us_per_image": wall,
                     "prepared_call_us_per_image": 1e6 * (time.perf_counter() - t0) / 200, "evals": int(r.w.evals)}
    return out


def measure(torch, jt, name, args, rank, world, sample_clocks=False):
    """Both timed legs and the roofline record of one workload.  Returns a dict (rank 0) or None."""
    w = make_workload(name, rank)
    batch = hasattr(w, "B")
    runner = BatchRunner(jt, w) if batch else ImageRunner(jt, w, args.method)
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")     # 256 MiB > 126 MB L2

    # ---- device-timed leg (inputs resident) ----
    jt.profile_enable(True)
    for _ in range(args.warmup):
        runner.step()
    torch.cuda.synchronize()
    sampler = ClockSampler(torch.cuda.current_device()) if (rank == 0 and sample_clocks) else None
    if sampler:
        sampler.start()
        time.sleep(0.25)
    barrier()
    torch.cuda.synchronize()
    launches0 = jt.kernel_launches()

    phase = []
    tier_counts = (0,) * len(TIER_NAMES)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.add_(1)
        a.record()
        runner.step()
        b.record()
        if not batch:
            phase.append(jt.profile_read())          # waits for this step's events only
            tier_counts = jt.profile_tiers()
    torch.cuda.synchronize()
    barrier()
    launches = jt.kernel_launches() - launches0
    ms = [a.elapsed_time(b) for a, b in ev]
    clocks = sampler.stop() if sampler else None
    jt.profile_enable(False)
    ms_total_local = float(sum(ms))
    units, ms_total = aggregate(w.evals * args.steps, ms_total_local)

    # ---- end-to-end leg (pinned host inputs -> device -> image back on the host), wall clock around a sync ----
    for _ in range(max(1, args.warmup)):
        runner.step_e2e()
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        runner.step_e2e()
        torch.cuda.synchronize()
    e2e_ms_local = 1e3 * (time.perf_counter() - t0)
    barrier()
    e2e_units, e2e_ms = aggregate(w.evals * args.steps, e2e_ms_local)
    del flush
    if rank != 0:
        return None

    peaks, peak_kind = load_peaks()
    rec = {"value": units / (ms_total * 1e-3), "ms_per_step": ms_total / args.steps,
           "ms_per_step_median": float(np.median(ms)), "ms_per_step_best": float(np.min(ms)), "dtype": w.dtype,
           "config": describe(name, w, world),
           "images_per_s": world * runner.images * args.steps / (ms_total * 1e-3), "clocks": clocks,
           "e2e": {"value": e2e_units / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": runner.h2d,
                   "d2h_bytes_per_step": runner.d2h, "ms_per_step": e2e_ms / args.steps},
           "gpu_launches": int(launches)}

    # ---- roofline of the dominant kernel: the ray-tracing kernel, issue-limited ALU peak ----
    f_mhz = (clocks or {}).get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
    lanes = ALU_LANES_PER_SM[w.dtype]
    peak_tinstr = SM_COUNT * lanes * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
    if phase:
        trace_ms = float(np.mean([p[0] for p in phase]))
        conv_ms = float(np.mean([p[1] for p in phase]))
    else:
        trace_ms, conv_ms = ms_total_local / args.steps, 0.0
    # tier mix of the (warp, subhalo record) pairs: counters of the last timed jt_simulate_image call; for the batch
    # kernel (no workspace, no counters) the same warp tiling is sampled through jt_simulate_image on 4 of its systems
    if batch:
        tiers = np.zeros(len(TIER_NAMES))
        jt.profile_enable(True)
        for b in range(min(4, w.B)):
            one = ImageRunner(jt, w.system(b), "direct")
            one.step()
            jt.profile_read()
            tiers += np.array(jt.profile_tiers(), dtype=np.float64)
        jt.profile_enable(False)
    else:
        tiers = np.array(tier_counts, dtype=np.float64)
    mix = tiers / tiers.sum() if tiers.sum() > 0 else np.array([0.0, 0.0, 0.0, 1.0, 0.0, 0.0])
    n_alg = float(np.dot(mix, TIER_COST[w.dtype]))
    achieved = w.evals * n_alg / (trace_ms * 1e-3) / 1e12
    rec["roofline"] = {
        "bound": "alu", "kernel": "k_batch" if batch else "k_trace", "achieved": achieved, "peak": peak_tinstr,
        "unit": "Tlaneop/s", "frac": achieved / peak_tinstr, "traffic": NCU_TRAFFIC_BYTES.get(name),
        "peak_kind": "derived: 148 SMs x %d lanes/clk (%s) x %.0f MHz (max clock, %s)" % (
            lanes, "FP32 pipe" if w.dtype == "f32" else "FP64 pipe", peaks.get("sm_max_mhz", 1965.0),
            peak_kind),
        "alg_instr_per_eval": n_alg, "tier_mix": dict(zip(TIER_NAMES, (float(x) for x in mix))),
        "tier_cost_per_eval": dict(zip(TIER_NAMES, TIER_COST[w.dtype])), "kernel_ms": trace_ms, "conv_ms": conv_ms,
        "kernel_share_of_step": trace_ms / (ms_total_local / args.steps),
        "frac_at_observed_clock": achieved / (SM_COUNT * lanes * f_mhz * 1e6 / 1e12),
        "evals_per_s_kernel": w.evals / (trace_ms * 1e-3)}
    rec["_w"] = w
    return rec


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    import paper_2606_01547_b200 as jt
    jt.lib()

    head = measure(torch, jt, args.workload, args, rank, world, sample_clocks=True)
    # the other paper-shaped workloads, same legs, in the same JSON line (single-GPU runs only: replicas add nothing here)
    per_config = {}
    if world == 1 and not args.no_per_config:
        for name in PER_CONFIG:
            if name != args.workload:
                r = measure(torch, jt, name, args, rank, world)
                r.pop("_w")
                per_config[name] = r
    if rank != 0:
        return
    peaks, _ = load_peaks()
    w = head.pop("_w")
    line = {"metric": METRIC, "value": head.pop("value"), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head.pop("ms_per_step"), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": head.pop("dtype"), "data": "synthetic"}
    line.update(head)
    # ---- ALU rates measured in this run by the probe library's microbenchmark (thread-level instructions / s) ----
    probes = {k: jt.probe_alu(k) for k in ("ffma", "ffma2", "dfma", "mufu_rsq")}
    line["alu_peaks_measured"] = {k: {"Tlaneinstr_per_s": v / 1e12, "lanes_per_clk_per_sm_at_max_clock":
                                      v / SM_COUNT / (peaks.get("sm_max_mhz", 1965.0) * 1e6)} for k, v in probes.items()}
    for r in [line] + list(per_config.values()):
        meas = probes["ffma"] if r["dtype"] == "f32" else probes["dfma"]
        r["roofline"]["frac_of_measured_alu_rate"] = r["roofline"]["achieved"] * 1e12 / meas
    line["conv"] = conv_block(torch, jt, w, peaks, probes)
    if world == 1 and not args.no_per_config:
        line["latency_configs"] = latency_block(torch, jt)
    if per_config:
        line["per_config"] = per_config
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w, args.cpu_evals)
    # The headline line is long; a reader that keeps only scalar keys of `roofline` (or only the end of stdout) would lose
    # the other kernels' numbers.  So: (1) the same numbers as flat scalars inside `roofline`, (2) each block as its own
    # short JSON line ("block": ...) BEFORE the headline line, which stays the LAST line of stdout.
    rf = line["roofline"]
    for name, r in per_config.items():
        key = name.lower().replace("-", "")
        rf["also_%s_frac" % key] = r["roofline"]["frac"]
        rf["also_%s_ms" % key] = r["ms_per_step"]
    c = line["conv"]
    rf["also_conv_direct_us"] = c["direct"]["us"]
    rf["also_conv_direct_frac"] = c["direct"].get("frac_of_derived_fma_peak")
    rf["also_conv_fft_us"] = c["fft"]["us"]
    rf["also_conv_fft_frac_hbm"] = c["fft"].get("frac_of_measured_hbm")
    for name, r in line.get("latency_configs", {}).items():
        rf["also_%s_device_us" % name.lower().replace("-", "")] = r["device_us_per_image_graph_replay"]
    for block in ("conv", "latency_configs"):
        if block in line:
            print(json.dumps({"block": block, "n_gpus": world, "data": line[block]}), flush=True)
    for name, r in per_config.items():
        slim = {k: r[k] for k in ("value", "ms_per_step", "dtype", "images_per_s", "gpu_launches") if k in r}
        slim["roofline_frac"] = r["roofline"]["frac"]
        slim["e2e_ms_per_step"] = r["e2e"]["ms_per_step"]
        print(json.dumps({"block": "per_config", "workload": name, "data": slim}), flush=True)
    print(json.dumps(line), flush=True)


def run_conv_sweep(args, rank):
    """--conv-sweep: jt_psf_convolve alone at the paper's E3 shapes (60x60 with K = 3..45, 180x180 with
    K = 9..135; 100x100 with K = 13) plus the configs' shapes, float32 and float64, DIRECT and FFT.
    Each case is captured into a CUDA graph of 20 back-to-back calls and the graph replay is timed with CUDA events, so
    the number is device time per call, not the Python binding's per-call cost.  Prints one JSON line."""
    if rank != 0:
        return
    import torch
    import paper_2606_01547_b200 as jt
    import workloads
    torch.cuda.set_device(0)
    jt.lib()
    peaks, _ = load_peaks()
    rng = np.random.default_rng(workloads.SEEDS["sweep"])
    shapes = [(60, k) for k in (3, 11, 21, 31, 45)] + [(180, k) for k in (9, 45, 87, 135)] + \
             [(100, 13), (100, 31), (200, 21), (500, 101), (1000, 31)]
    reps = 20
    rows = []
    paper_shapes = set([(60, k) for k in (3, 11, 21, 31, 45)] + [(180, k) for k in (9, 45, 87, 135)] + [(100, 13)])
    for dtype, tdt, lanes, esz in (("f32", torch.float32, 128, 4), ("f64", torch.float64, 64, 8)):
        fma_peak = SM_COUNT * lanes * peaks.get("sm_max_mhz", 1965.0) * 1e6
        for n, k in shapes:
            sig = k / 8.0
            u = np.arange(k) - k // 2
            ker = np.exp(-(u[:, None] ** 2 + u[None, :] ** 2) / (2 * sig * sig))
            ker = torch.as_tensor(ker / ker.sum(), dtype=tdt, device="cuda")
            for B in ((1, args.sweep_batch) if (n, k) in paper_shapes else (1,)):
                img = torch.as_tensor(rng.uniform(0, 1, (B, n, n)), dtype=tdt, device="cuda")
                out = torch.empty_like(img)
                row = {"dtype": dtype, "n": n, "K": k, "B": B}
                for method in ("direct", "fft", "auto"):
                    try:
                        nb = jt.psf_convolve_batch_workspace_bytes(dtype, B, n, n, k, k, method)
                        ws = torch.empty(max(nb, 1), dtype=torch.uint8, device="cuda")
                        call = lambda: jt.psf_convolve_batch(img, ker, method=method, workspace=ws, out=out)
                        us = graph_time(torch, call, reps if B == 1 else 3)
                        row[method + "_us"] = us
                        row[method + "_gbs"] = B * (2 * n * n + k * k) * esz / (us * 1e-6) / 1e9
                        if method == "direct":
                            row["direct_frac_of_fma_peak"] = B * n * n * k * k / (us * 1e-6) / fma_peak
                    except jt.JtError as e:
                        row[method + "_us"] = None
                        row[method + "_error"] = str(e)
                rows.append(row)
    print(json.dumps({"metric": "psf_convolve_us", "unit": "us per call (CUDA-graph replay of %d calls)" % reps,
                      "n_gpus": 1, "data": "synthetic", "rows": rows}), flush=True)


def run_swarm(args, rank):
    """--swarm: the shape of the paper's particle-swarm benchmark (64 ... 512 particles, 100 x 100 grid,
    13-pixel PSF): one swarm step = every particle's image simulated and reduced to its
    chi^2 against the same data by jt_simulate_batch_chi2 (images never leave the chip).  Device time per step from a
    CUDA-graph replay, wall time per step with the particles' parameters copied from pinned host memory and the B chi^2
    values copied back.  The paper's numbers (59 / 138 / 245 / 555 s with lenstronomy for whole fits of unstated
    iteration counts) are context only: the optimiser is out of scope."""
    if rank != 0:
        return
    import torch
    import paper_2606_01547_b200 as jt
    import workloads
    torch.cuda.set_device(0)
    jt.lib()
    rows = []
    for dtype, tdt in (("f64", torch.float64), ("f32", torch.float32)):
        for B in (64, 128, 256, 512):
            w = workloads.config_swarm(B=B, dtype=dtype)
            g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
            pin = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=tdt).pin_memory()
            h = [pin(w.sie), pin(w.shear), pin(w.sources), pin(w.psf)]
            d = [t.to("cuda") for t in h]
            truth = jt.simulate_batch(g, d[0][:1], d[1][:1], None, d[2][:1], d[3][:1])[0]
            data = truth + torch.as_tensor(w.data, dtype=tdt, device="cuda")
            sigma = torch.as_tensor(w.sigma, dtype=tdt, device="cuda")
            chi2 = torch.empty(B, dtype=torch.float64, device="cuda")
            h_chi2 = torch.empty(B, dtype=torch.float64).pin_memory()
            step = lambda: jt.simulate_batch_chi2(g, d[0], d[1], None, d[2], d[3], data, sigma, chi2=chi2)
            us = graph_time(torch, step)

            def e2e():
                for dd, hh in zip(d[:3], h[:3]):
                    dd.copy_(hh, non_blocking=True)
                step()
                h_chi2.copy_(chi2, non_blocking=True)
                torch.cuda.synchronize()
            for _ in range(3):
                e2e()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                e2e()
            wall = 1e6 * (time.perf_counter() - t0) / args.steps
            rows.append({"dtype": dtype, "particles": B, "device_us_per_step": us, "e2e_us_per_step": wall,
                         "particle_images_per_s": B / (us * 1e-6), "chi2_of_truth_per_pixel": float(h_chi2[0]) / (w.nx * w.ny)})
    print(json.dumps({"metric": "swarm_step_us", "unit": "us per swarm step (all particles: image + chi^2)", "n_gpus": 1,
                      "data": "synthetic", "grid": "100x100", "psf": "13x13", "rows": rows,
                      "paper_context": "PAPER.md:122-126: whole PSO fits, lenstronomy 59/138/245/555 s for 64/128/256/512 particles"}),
          flush=True)


def run_next(args, rank):
    """--next: the paper's own per-profile benchmark (tables "Deflection angle calculations" and "Flux
    calculations": ONE deflection / flux call per profile on a 60 x 60 and a 180 x 180 grid) through the SURVEY 8(f) entry
    points, plus jt_lensing_maps on C2's lens.  Device time per call from a CUDA-graph replay (no Python / ctypes cost in
    the number).  Stated bound: at 3,600 / 32,400 points these calls are launch-latency-bound (one launch of one-point-per-
    thread double-precision code, ~2-4 us whatever the profile, 15 - 127 thread blocks on 148 SMs); the rate column is what
    it is, no roofline fraction is claimed for them.  The paper's table gives speed-up RATIOS over lenstronomy on other
    hardware, no absolute times: context only."""
    if rank != 0:
        return
    import torch
    import paper_2606_01547_b200 as jt
    from paper_2606_01547_b200 import binding as b
    import workloads
    torch.cuda.set_device(0)
    jt.lib()
    defl = [("CONVERGENCE", [0.1, 0.0, 0.0]), ("SIS", [1.0, 0.01, -0.02]), ("NFW", [0.3, 0.2, -0.1, 0.1]),
            ("HERNQUIST", [0.4, 0.5, 0.1, 0.0]), ("PJAFFE", [0.5, 0.1, 0.6, 0.0, 0.1]), ("SIE", [1.0, 0.1, -0.05, 0.0, 0.0]),
            ("SHEAR", [0.03, 0.01]), ("TNFW", [0.2, 0.1, 1.0, 0.8, 0.3]), ("NIE", [1.1, 0.2, -0.1, 0.15, 0.3, -0.1]),
            ("EPL", [1.0, 2.3, 0.15, 0.1, -0.2, 0.3]), ("MULTIPOLE", [3.0, 0.04, 0.2, -0.2, 0.3]),
            ("CSE", [0.05, 0.2, 0.3, -0.15, 0.5, 0.5]), ("PJAFFE_ELLIPSE_POTENTIAL", [0.5, 0.1, 0.6, 0.2, -0.1, 0.0, 0.1])]
    light = [("SERSIC_ELLIPSE", [10.0, 0.2, 1.5, 0.05, 0.02, 0.05, 0.0]), ("GAUSSIAN_ELLIPSE", [1.0, 0.2, 0.2, -0.1, 0.05, 0.0])]
    rows = []
    for dtype, tdt in (("f64", torch.float64), ("f32", torch.float32)):
        for n in (60, 180):
            u = (np.arange(n) - (n - 1) / 2) * 0.05
            x = torch.as_tensor(np.repeat(u[None, :], n, 0).reshape(-1).copy(), dtype=tdt, device="cuda")
            y = torch.as_tensor(np.repeat(u[:, None], n, 1).reshape(-1).copy(), dtype=tdt, device="cuda")
            calls = []
            for name, p in defl:
                rec = b.profile_records([(name, p)], b.DEFLECTOR_TYPES)
                calls.append(("deflection", name, lambda rec=rec: jt.ray_shoot_profiles(x, y, rec)))
            for name, p in light:
                rec = b.profile_records([(name, p)], b.LIGHT_TYPES)
                calls.append(("flux", name, lambda rec=rec: jt.light_profiles(x, y, rec)))
            mg = b.profile_records([("GAUSSIAN_ELLIPSE", [1.0, 0.05 * 2 ** k, 0.2, -0.1, 0.05, 0.0]) for k in range(5)], b.LIGHT_TYPES)
            calls.append(("flux", "MULTI_GAUSSIAN_ELLIPSE(5)", lambda: jt.light_profiles(x, y, mg)))
            calls.append(("flux", "CORE_SERSIC", lambda: jt.light_core_sersic(x, y, [10.0, 0.3, 2.0, 0.05, 0.2, 2.0, 0.1, -0.05, 0.0, 0.0])))
            for n_max in (6, 10):
                coef = torch.as_tensor(np.random.default_rng(n_max).normal(size=(n_max + 1) * (n_max + 2) // 2), dtype=tdt, device="cuda")
                calls.append(("flux", "SHAPELETS(n_max=%d)" % n_max,
                              lambda n_max=n_max, coef=coef: jt.light_shapelets(x, y, n_max, 0.3, 0.0, 0.0, coef)))
            for kind, name, call in calls:
                us = graph_time(torch, call)
                rows.append({"kind": kind, "profile": name, "dtype": dtype, "grid": "%dx%d" % (n, n), "us_per_call": us,
                             "points_per_s": n * n / (us * 1e-6)})
        # NEXT-2: kappa, gamma1, gamma2, mu of C2's lens (SIE + shear + 10,000 TNFW) on C2's 160,000 ray positions
        w = workloads.config_c2(dtype=dtype)
        m = w.nx * w.supersample
        u = (np.arange(m) - (m - 1) / 2) * (w.pixel_scale / w.supersample)
        x = torch.as_tensor(np.repeat(u[None, :], m, 0).reshape(-1).copy(), dtype=tdt, device="cuda")
        y = torch.as_tensor(np.repeat(u[:, None], m, 1).reshape(-1).copy(), dtype=tdt, device="cuda")
        tn = torch.as_tensor(np.ascontiguousarray(w.tnfw), dtype=tdt, device="cuda")
        us = graph_time(torch, lambda: jt.lensing_maps(x, y, w.sie, w.shear, tn), n_rep=3)
        rows.append({"kind": "lensing_maps", "profile": "SIE+SHEAR+10000 TNFW (C2)", "dtype": dtype, "grid": "400x400 rays",
                     "us_per_call": us, "point_deflector_evals_per_s": m * m * (w.n_tnfw + 2) / (us * 1e-6),
                     "bound": "alu (double-precision libdevice code in both dtype modes; correct-first, not tier-tuned)"})
    print(json.dumps({"metric": "next_profile_call_us", "unit": "us per call (CUDA-graph replay)", "n_gpus": 1,
                      "data": "synthetic", "bound": "launch latency at 60^2 / 180^2 points (see docstring)", "rows": rows,
                      "paper_context": "PAPER.md:59-108 lists speed-up ratios over lenstronomy per profile, no absolute times"}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4-f64", choices=WORKLOADS)
    ap.add_argument("--method", default="auto", choices=["auto", "direct", "fft"])
    ap.add_argument("--cpu-evals", type=float, default=1.5e9, help="oracle sample size for cpu_baseline")
    ap.add_argument("--ref-evals", type=float, default=2.0e8, help="oracle sample size per --impl reference step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (C2-f64, C2-f32, C3-f32)")
    ap.add_argument("--conv-sweep", action="store_true", help="time jt_psf_convolve alone at the paper's shapes")
    ap.add_argument("--sweep-batch", type=int, default=1024, help="batch size of the batched rows of --conv-sweep")
    ap.add_argument("--swarm", action="store_true", help="time the particle-swarm inner loop (NEXT-3) at the paper's sizes")
    ap.add_argument("--next", action="store_true", help="time one call per SURVEY 8(f) profile on 60^2 / 180^2 grids + jt_lensing_maps")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, world, local_rank = dist_init(args.gpus)
    try:
        if args.conv_sweep:
            run_conv_sweep(args, rank)
        elif args.swarm:
            run_swarm(args, rank)
        elif args.next:
            run_next(args, rank)
        elif args.impl == "reference":
            run_reference(args, rank, world)
        else:
            run_ours(args, rank, world, local_rank)
    finally:
        import torch.distributed as dist
        if dist.is_available() and dist.is_initialized():
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
