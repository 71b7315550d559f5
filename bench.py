#!/usr/bin/env python
"""bench.py -- measurement of the hot path (SURVEY.md section 8d / DESIGN.md section 7).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload train] [--impl ours|reference]

A "step" is one pass of the whole hot path -- inpc_raster_forward + inpc_raster_backward (rows a1..a5)
-- over one seeded synthetic point cloud.  Default workload: BASELINE.json config 3 ("train":
2^23 points, 1297x840, D = 4, octree sampler), the one north_star quotes its target on.

One JSON line is printed by rank 0:
  value            emitted fragments per second over the whole fwd+bwd step, inputs resident in HBM
                   (all ranks' fragments / max-over-ranks device time of exactly K steps)
  e2e              the same metric through the C-ABI binding with HOST (pinned) buffers: per step the
                   inputs are copied host->device and every result device->host inside the timed region
  roofline         the dominant kernel: algorithmic bytes per launch / its mean launch duration (CUDA
                   events on the launching stream, recorded by the library around every stage)
  roofline_step    the whole fwd+bwd step against the same peak (north_star's 50 % target)
  cpu_baseline     the oracle, as it stands, on the host cores, on a bounded sample (rank 0, N = 1)
  clocks           nvidia-smi samples taken while the timed regions ran

Multi-GPU: the path does not shard in this build (north_star: one GPU, no collectives) -> REPLICAS ONLY:
every rank rasterises its own seeded cloud (seed + rank); the only communication is the barrier and
the max/sum of the timing scalars.  `--impl reference` times the oracle (oracle/, CPU) per step.
"""
from __future__ import annotations

import argparse
import datetime as _dt
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# flags of the two timed launch configurations (tests/harness.py runs its parity comparison with exactly these)
FLAGS_STEP = 1      # INPC_SAVE_FOR_BACKWARD: the forward of the fwd+bwd step
FLAGS_FWD = 0       # forward only (inference)

METRIC = "fragments/sec (fwd+bwd step, forward only for the inference config; ms/frame fwd and fwd+bwd beside it)"
UNIT = "fragments/s"
L2_BYTES = 126 * 1024 * 1024

# ------------------------------------------------------------------------------------------------
# algorithmic bytes: per fragment / pixel / point figures
def algorithmic_bytes(n_points: int, n_frag: int, n_pix: int, D: int) -> dict:
    F = 4 * D
    a12 = 24 * n_points + 8 * n_frag + 12 * n_pix                       # a1 + a2: project, count, scan, emit
    a34 = (8 + 4 + F) * n_frag + 4 * (D + 1) * n_pix                    # a3 + a4: sort + blend
    a5 = (8 + 4 + F + 8) * n_frag + (8 * (D + 1) + 8) * n_pix + (F + 12) * n_points   # a5: backward
    a5_walk = (8 + 4 + F + 8) * n_frag + (8 * (D + 1) + 8) * n_pix       # reverse traversal (k_back, k_big<bwd>)
    a5_out = (F + 12) * n_points                                         # per-point gradients (k_combine, k_split)
    return {"a1_a2": a12, "a3_a4": a34, "a5": a5, "a5_walk": a5_walk, "a5_out": a5_out,
            "fwd": a12 + a34, "bwd": a5, "fwd_bwd": a12 + a34 + a5}


# which path rows each library stage belongs to (for the per-kernel roofline)
STAGE_ROWS = {
    "k_blend": "a3_a4", "k_big_fwd": "a3_a4",
    "k_back": "a5_walk", "k_big_bwd": "a5_walk", "zero_bwd": "a5_walk",
    "zero_fwd": "a1_a2", "k_project_count": "a1_a2", "k_scan_u32": "a1_a2", "k_scatter": "a1_a2",
    "k_classify": "a1_a2", "k_build_items": "a1_a2",
    "k_cellsort": "a3_a4", "k_cellsort_big": "a3_a4",
    "k_combine": "a5_out", "k_split": "a5_out", "other": "a1_a2",
}


def measured_peak_gbs() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
# aggregation over ranks: time = max, units = sum (tested with gloo, world_size 2, on CPU)
def aggregate_over_ranks(local_ms: float, local_units: float, device="cpu") -> tuple[float, float]:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(units: float, ms: float) -> float:
    return units / (ms * 1e-3) if ms > 0 else 0.0


# ------------------------------------------------------------------------------------------------
# clocks: the profiling recipe's nvidia-smi line, sampled while the timed regions run
class ClockSampler:
    FIELDS = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int, period_ms: int = 50):
        self.path = os.path.join(tempfile.gettempdir(), f"inpc_clocks_{os.getpid()}.csv")
        self.windows = []
        self.proc = None
        try:
            self.out = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", str(period_ms)],
                                         stdout=self.out, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def window(self):
        sampler = self

        class _W:
            def __enter__(self_w):
                self_w.t0 = _dt.datetime.now()

            def __exit__(self_w, *exc):
                sampler.windows.append((self_w.t0, _dt.datetime.now()))
        return _W()

    def finish(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "note": "nvidia-smi unavailable"}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.out.close()
        rows = []
        with open(self.path) as f:
            for line in f:
                parts = [p.strip() for p in line.strip().split(",")]
                if len(parts) < 9:
                    continue
                try:
                    ts = _dt.datetime.strptime(parts[0], "%Y/%m/%d %H:%M:%S.%f")
                    rows.append((ts, float(parts[1]), float(parts[2]), float(parts[3]), parts[4:]))
                except ValueError:
                    continue
        try:
            os.remove(self.path)
        except OSError:
            pass
        inside = [r for r in rows if any(a <= r[0] <= b for a, b in self.windows)]
        note = "samples inside the timed regions"
        if not inside:
            inside, note = rows, "no sample fell inside a timed region; all samples of the run"
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "note": "no samples"}
        sm = sorted(r[1] for r in inside)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[4][1 + k].lower().startswith("active") for r in inside)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(r[2] for r in inside), "reasons": reasons,
                "power_w_max": max(r[3] for r in inside), "samples": len(inside), "note": note}


# ------------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline at N = 1, and --impl reference)
def oracle_step(wl, n_sample: int) -> tuple[float, int]:
    """One step (fwd+bwd; forward only for the inference config) of the oracle on the first n_sample points of the
    workload -> (seconds, fragments)."""
    import oracle
    t0 = time.perf_counter()
    ref = oracle.Raster.from_points(wl.pos[:n_sample], wl.opacity[:n_sample], wl.feat[:n_sample], wl.cam)
    ref.blend()
    if wl.backward:
        ref.backward(wl.g_img, wl.g_alpha)
    dt = time.perf_counter() - t0
    frags = ref.total
    del ref
    return dt, frags


def oracle_sample_size(wl, seconds_per_step: float) -> int:
    """Largest power-of-two prefix of the workload the oracle is expected to finish in the budget
    (calibrated on a 2^17-point prefix)."""
    n_cal = min(wl.N, 1 << 17)
    dt, _ = oracle_step(wl, n_cal)
    rate = n_cal / max(dt, 1e-6)
    n = int(min(wl.N, rate * seconds_per_step))
    p = 1 << 12
    while p * 2 <= n:
        p *= 2
    return min(p, wl.N)


def cpu_baseline(wl, budget_s: float = 12.0, openmp: bool = False) -> dict:
    """The oracle as it stands on the host cores: single-threaded (the build every test uses), or -- openmp=True --
    the SAME source built with -fopenmp on all cores (SURVEY.md 8d "Oracle timed beside it" (2))."""
    import oracle
    threads = oracle.use_openmp(True) if openmp else 1
    try:
        n = oracle_sample_size(wl, budget_s)
        dt, frags = oracle_step(wl, n)
    finally:
        if openmp:
            oracle.use_openmp(False)
    return {"value": frags / dt, "unit": UNIT, "cores": threads, "nproc": os.cpu_count(),
            "kind": "oracle (-fopenmp build, all cores)" if openmp else "oracle",
            "n_points_timed": int(n), "n_points": int(wl.N),
            "sample": f"first {n} of {wl.N} points of '{wl.name}' (same camera, full image), one fwd+bwd, "
                      f"{frags} fragments in {dt:.2f} s; oracle/oracle.cpp fp64, {threads} thread(s)"
                      + (" (bucket fill serial; sort, blend and backward parallel over pixels)" if openmp else ""),
            "seconds": dt}


def run_reference(args) -> int:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0                                     # under torchrun only rank 0 runs the oracle
    from paper_2403_16862_b200.workloads import make_workload
    wl = make_workload(args.workload)
    total = max(1, args.steps + args.warmup)
    n = oracle_sample_size(wl, min(15.0, 150.0 / total))
    for _ in range(args.warmup):
        oracle_step(wl, n)
    secs, frags = 0.0, 0
    for _ in range(args.steps):
        dt, fr = oracle_step(wl, n)
        secs += dt
        frags += fr
    value = frags / secs if secs > 0 else 0.0
    sample = (f"each step = oracle fwd+bwd on the first {n} of {wl.N} points of '{wl.name}' "
              f"(same camera, full image); single-threaded fp64 CPU")
    # The oracle is timed on a PREFIX of the cloud (a sparser cloud: fewer fragments per pixel, a different blended
    # fraction), so its throughput is that of a different configuration; the line says so where a reader of `config` looks.
    cfg = workload_config(wl, args)
    cfg["n_points_timed"] = int(n)
    cfg["same_config_as_gpu_arm"] = bool(n == wl.N)
    if n != wl.N:
        cfg["note"] = (f"timed on the first {n} of {wl.N} points (bounded CPU sample): throughput of a sparser cloud, "
                       "not of the full configuration")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(wl, args, n_sets: int = 1) -> dict:
    return {"workload": f"{wl.name}: BASELINE.json config '{args.workload}', N={wl.N} points, "
                        f"{wl.cam.width}x{wl.cam.height}, D={wl.D}, seed {wl.seed}",
            "n_points": wl.N, "width": wl.cam.width, "height": wl.cam.height, "D": wl.D,
            "pass": "forward + backward (grad_feat, grad_opacity, grad_uv)" if wl.backward else "forward only (feature image + alpha)",
            "point_order": "leaf-coherent (Morton order of the octree grid: secondary measurement)" if getattr(args, "order", "sampler") == "leaf"
                           else "unordered sampler output (random permutation)",
            "parallelism": "replicas only (one cloud per GPU, no data-path collective)",
            "l2_hygiene": "inputs + records larger than L2 (see l2 key)" if n_sets == 1 else
                          f"working set fits L2: {n_sets} independent buffer sets rotated (see l2 key)"}


def make_step_functions(raster, wl, dev, stream=None):
    """Device-resident buffers of one workload and the two calls a step is made of.
    -> fwd(flags), bwd(), dict of the tensors.  tests/test_gpu_parity.py launches these to check that what is
    timed here is what the parity tests compared with the oracle."""
    import numpy as np
    import torch
    W, H, D, N = wl.cam.width, wl.cam.height, wl.D, wl.N
    cam = raster.camera_struct(wl.cam)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    t = dict(pos=to_dev(wl.pos), op=to_dev(wl.opacity), feat=to_dev(wl.feat), g_img=to_dev(wl.g_img),
             g_alpha=to_dev(wl.g_alpha), cam=cam)
    t["ws"] = raster.alloc_workspace(N, D, W, H, FLAGS_STEP, dev)
    t["img"] = torch.empty((H, W, D), dtype=torch.float32, device=dev)
    t["alpha"] = torch.empty((H, W), dtype=torch.float32, device=dev)
    t["d_feat"] = torch.empty((N, D), dtype=torch.float32, device=dev)
    t["d_op"] = torch.empty((N,), dtype=torch.float32, device=dev)
    t["d_uv"] = torch.empty((N, 2), dtype=torch.float32, device=dev)
    if stream is None:
        stream = torch.cuda.current_stream()

    def fwd(f=FLAGS_STEP):
        raster.inpc_raster_forward(t["pos"], t["op"], t["feat"], cam, out_feat=t["img"], out_alpha=t["alpha"],
                                   workspace=t["ws"], flags=f, stream=stream)

    def bwd():
        raster.inpc_raster_backward(t["pos"], t["op"], t["feat"], cam, t["g_img"], t["g_alpha"], t["ws"],
                                    grad_feat=t["d_feat"], grad_opacity=t["d_op"], grad_uv=t["d_uv"], stream=stream)

    return fwd, bwd, t


# ------------------------------------------------------------------------------------------------
# DRAM traffic per launch: read from the committed ncu CSV, never typed in
def source_hash() -> str:
    """sha256 over the kernel sources (csrc/*, include/*.h): what a traffic capture is valid for."""
    import hashlib
    h = hashlib.sha256()
    for d in (os.path.join(ROOT, "paper_2403_16862_b200", "csrc"), os.path.join(ROOT, "include")):
        for fn in sorted(os.listdir(d)):
            if fn.endswith((".cu", ".cuh", ".h")):
                h.update(fn.encode())
                h.update(open(os.path.join(d, fn), "rb").read())
    return h.hexdigest()[:16]


TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r03_traffic.csv")      # raw `ncu --csv` output, see r03_traffic.md


def ncu_traffic(workload: str) -> dict:
    """{stage name: mean dram read+write bytes per launch} from profiles/r03_traffic.csv, or {} (with the reason)
    when the capture is for other kernel sources or another workload (profiles/r03_traffic.md records both)."""
    import csv
    import re
    md = TRAFFIC_CSV[:-4] + ".md"
    if not (os.path.exists(TRAFFIC_CSV) and os.path.exists(md)):
        return {"_note": "no committed capture (profiles/r03_traffic.csv)"}
    text = open(md).read()
    m_hash = re.search(r"source_hash:\s*`?([0-9a-f]{16})", text)
    m_wl = re.search(r"workload:\s*`?(\w+)", text)
    if not m_hash or m_hash.group(1) != source_hash():
        return {"_note": f"capture is for kernel sources {m_hash.group(1) if m_hash else '?'}, this build is {source_hash()}: traffic null"}
    if not m_wl or m_wl.group(1) != workload:
        return {"_note": f"capture is for workload {m_wl.group(1) if m_wl else '?'}: traffic null"}
    rows = [r for r in csv.reader(open(TRAFFIC_CSV)) if len(r) > 5]
    head = next(r for r in rows if "Kernel Name" in r)
    ik, im, iv, iu = head.index("Kernel Name"), head.index("Metric Name"), head.index("Metric Value"), head.index("Metric Unit")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc, cnt = {}, {}
    for r in rows:
        if r is head or not r[im].startswith("dram__bytes_"):
            continue
        name = r[ik].split("(")[0].replace("void ", "").replace("inpc::", "").strip()
        acc[name] = acc.get(name, 0.0) + float(r[iv].replace(",", "")) * scale.get(r[iu], 1.0)
        if r[im].startswith("dram__bytes_read"):
            cnt[name] = cnt.get(name, 0) + 1
    out = {k: acc[k] / max(cnt.get(k, 1), 1) for k in acc}
    out["_note"] = f"profiles/r03_traffic.csv (ncu dram__bytes_read.sum + dram__bytes_write.sum, mean per launch; sources {source_hash()})"
    return out


def traffic_of_stage(traffic: dict, stage: str, D: int = 4, save: bool = True):
    """Stage names carry no template arguments; the capture's kernel names do: k_blend<D, SAVE, DUMP>,
    k_big<D, MODE> (0 forward, 2 backward), k_cellsort_big<D, THREADS, CHUNK> (two launches per stage: summed)."""
    want = {"k_blend": f"k_blend<{D}, {1 if save else 0}, 0>", "k_big_fwd": f"k_big<{D}, 0>", "k_big_bwd": f"k_big<{D}, 2>",
            "k_scatter": "k_scatter<0>", "k_split": f"k_split<{D}, 0>"}          # <1> / <D, 1>: the fused-SH variants (next_rows)
    if stage in want:
        return traffic.get(want[stage])
    vals = [v for k, v in traffic.items() if not k.startswith("_") and k.split("<")[0] == stage
            and ("<" not in k or k.split("<")[1].split(",")[0].strip(" >") == str(D))]
    if not vals:
        return None
    return sum(vals) if stage == "k_cellsort_big" else sum(vals) / len(vals)


# ------------------------------------------------------------------------------------------------
def workload_statistics(raster, wl, T, dev) -> dict:
    """the workload characterised, not assumed -- per-pixel fragment counts, how much of them the
    cut-off lets through, depth ties, termination-ambiguous pixels.  One extra forward with INPC_SAVE_SORTED,
    outside every timed region; all reductions on the device."""
    import torch
    W, H, D, N = wl.cam.width, wl.cam.height, wl.D, wl.N
    flags = raster.SAVE_FOR_BACKWARD | raster.SAVE_SORTED
    try:
        ws = raster.alloc_workspace(N, D, W, H, flags, dev)
    except Exception as e:                                   # very large configs on a small device
        return {"note": f"skipped: {e}"}
    raster.inpc_raster_forward(T["pos"], T["op"], T["feat"], T["cam"], out_feat=T["img"], out_alpha=T["alpha"],
                               workspace=ws, flags=flags)
    cnt = raster.inpc_raster_get_counts(ws, W, H).reshape(-1).to(torch.int64)
    nb = raster.inpc_raster_get_blended_counts(ws, W, H).reshape(-1).to(torch.int64)
    off, _, dep, tr = raster.inpc_raster_get_sorted(ws, W, H, transmittance=True)
    total = int(cnt.sum())
    q = torch.quantile(cnt.to(torch.float32)[:: max(1, cnt.numel() // 4_000_000)], torch.tensor([0.5, 0.9, 0.99], device=dev))
    # depth ties: consecutive fragments of ONE pixel with equal depth bits
    ties = 0
    if total > 1:
        same = dep[1:] == dep[:-1]
        starts = torch.zeros(total + 1, dtype=torch.bool, device=dev)
        starts[off.to(torch.int64).clamp(max=total)] = True          # first fragment of every pixel
        ties = int((same & ~starts[1:total]).sum())
    # termination-ambiguous pixels as the KERNEL sees them: a transmittance it tested within 1e-4 (relative) of 1e-4
    near = ((tr - 1e-4).abs() < 1e-8) & (tr > 0)
    flagged = 0
    if total:
        pix_of = torch.searchsorted(off.to(torch.int64)[1:].contiguous(), torch.nonzero(near).reshape(-1), right=True)
        flagged = int(torch.unique(pix_of).numel())
    del ws
    return {"fragments": total, "pixels": int(cnt.numel()),
            "fragments_per_pixel": {"mean": total / max(1, cnt.numel()), "p50": float(q[0]), "p90": float(q[1]),
                                    "p99": float(q[2]), "max": int(cnt.max()) if cnt.numel() else 0},
            "blended_fragments": int(nb.sum()), "blended_fraction": float(nb.sum()) / max(1, total),
            "pixels_reaching_cutoff": int((nb < cnt).sum()),
            "depth_ties": ties, "termination_ambiguous_pixels": flagged,
            "note": "termination-ambiguous = a blended fragment's fp32 transmittance within 1e-4 (relative) of the 1e-4 cut-off"}


# ------------------------------------------------------------------------------------------------
def next_rows(raster, wl, T, dev, stream, reps: int = 10, n_frag: int = 0, peak_gbs: float = 0.0) -> dict:
    """Timings of the NEXT rows of the scope table on the same workload, outside the headline:
    f1 blending weights fused into the backward pass, f2 SH fused into the emission pass, f3 three resolution levels
    and four-cloud multisampling, f4 the view-specific sampler.  CUDA events, 3 warm-ups, mean of `reps`."""
    import numpy as np
    import torch
    from paper_2403_16862_b200.workloads import make_octree
    N, D, W, H = wl.N, wl.D, wl.cam.width, wl.cam.height
    cam = T["cam"]

    def ms(fn):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    out = {}
    alg = algorithmic_bytes(N, n_frag, W * H, D)

    def roof(nbytes, t_ms):                       # algorithmic bytes of the row / its time, against the measured HBM peak
        ach = nbytes / (t_ms * 1e-3) / 1e9
        return {"algorithmic_bytes": int(nbytes), "achieved_gbs": ach, "frac": (ach / peak_gbs) if peak_gbs else None}

    pos, op, feat, g_img, g_alpha, ws = T["pos"], T["op"], T["feat"], T["g_img"], T["g_alpha"], T["ws"]
    raster.inpc_raster_forward(pos, op, feat, cam, out_feat=T["img"], out_alpha=T["alpha"], workspace=ws, flags=FLAGS_STEP)
    bw = torch.empty((N,), dtype=torch.float32, device=dev)
    t_plain = ms(lambda: raster.inpc_raster_backward(pos, op, feat, cam, g_img, g_alpha, ws, grad_feat=T["d_feat"],
                                                     grad_opacity=T["d_op"], grad_uv=T["d_uv"]))
    t_w = ms(lambda: raster.inpc_raster_backward(pos, op, feat, cam, g_img, g_alpha, ws, grad_feat=T["d_feat"],
                                                 grad_opacity=T["d_op"], grad_uv=T["d_uv"], blend_weight=bw))
    out["f1_blend_weights"] = {"ms_backward": t_plain, "ms_backward_with_weights": t_w, "extra_bytes_per_point": 4}
    if D == 4:
        coeff = torch.randn((N, 36), dtype=torch.float32, device=dev) * 0.5
        o = raster.inpc_raster_forward_sh(pos, op, coeff, cam, flags=FLAGS_STEP)          # buffers allocated once, here
        gsh = (torch.empty((N, 36), dtype=torch.float32, device=dev), T["d_op"], T["d_uv"])
        t_f = ms(lambda: raster.inpc_raster_forward_sh(pos, op, coeff, cam, flags=FLAGS_STEP, out_feat=o[0], out_alpha=o[1],
                                                       workspace=o[2]))
        t_b = ms(lambda: raster.inpc_raster_backward_sh(pos, op, coeff, cam, g_img, g_alpha, o[2], grads=gsh))
        # the row's bytes: the plain pass's, with 144 B of coefficients per point read (forward) / written (backward)
        # in place of the 16 B of features
        out["f2_fused_sh"] = {"ms_forward": t_f, "ms_backward": t_b, "coefficient_bytes_per_point": 144,
                              "forward": roof(alg["fwd"] + (144 - 16) * N, t_f),
                              "backward": roof(alg["bwd"] + (144 - 16) * N, t_b),
                              "note": "outputs, gradients and workspace pre-allocated (no allocation in the timed loop)"}
        del coeff, o, gsh
    lv = raster.inpc_raster_forward_levels(pos, op, feat, cam, 3, flags=FLAGS_FWD)
    t_l = ms(lambda: raster.inpc_raster_forward_levels(pos, op, feat, cam, 3, flags=FLAGS_FWD, outs=lv[:3]))
    # three passes over the same cloud: the per-fragment / per-point bytes three times, the per-pixel bytes at 1 + 1/4 + 1/16
    out["f3_three_levels_forward"] = {"ms": t_l, **roof(3 * alg["fwd"] - (3 - 21 / 16) * (12 + 4 * (D + 1)) * W * H, t_l),
                                      "note": "levels 0, 1, 2 of one cloud, forward only; buffers pre-allocated"}
    del lv
    clouds = [(pos, op, feat)] * 4
    mo = raster.inpc_raster_forward_multisample(clouds, cam, n_levels=1, flags=raster.OUT_PLANAR)
    mws = raster.alloc_workspace(N, D, W, H, 0, dev)
    t_m = ms(lambda: raster.inpc_raster_forward_multisample(clouds, cam, n_levels=1, flags=raster.OUT_PLANAR, outs=mo, workspace=mws))
    out["f3_multisample_4_clouds"] = {"ms": t_m, "splats": 16 * N, **roof(4 * alg["fwd"], t_m),
                                      "note": "four clouds of N points averaged per pixel, [D,H,W] output (PAPER.md:172: 8M x 4 x 4 = 128 M splats)"}
    centre, level, prob, root = make_octree(1 << 20, seed=21)
    dc, dl, dp = (torch.from_numpy(a).to(dev) for a in (centre, level, prob))
    sws = {}

    def f_s():
        sws["o"] = raster.inpc_sample_view(dc, dl, dp, root, cam, seed=7, N=N, workspace=sws.get("w"))
        sws["w"] = sws["o"][2]

    t_s = ms(f_s)
    # per leaf: centre, level, probability in (20 B), p^ and the CDF written and read (32 B); per sample: 16 B out
    # (the CDF probes of a draw -- guide table, then ~4 of them -- hit L2 and are not counted)
    out["f4_sampler"] = {"ms": t_s, "leaves": 1 << 20, "samples": N, "samples_per_sec": N / (t_s * 1e-3),
                         "valid": raster.inpc_sample_get_stats(sws["w"])["n_valid"], **roof(52 * (1 << 20) + 16 * N, t_s)}
    t_s1 = ms(lambda: raster.inpc_sample_view(dc, dl, dp, root, cam, seed=7, N=N, workspace=sws["w"], flags=raster.SAMPLE_NO_RESAMPLE))
    out["f4_sampler_no_resample"] = {"ms": t_s1, "samples_per_sec": N / (t_s1 * 1e-3),
                                     "valid": raster.inpc_sample_get_stats(sws["w"])["n_valid"],
                                     "note": "INPC_SAMPLE_NO_RESAMPLE: one draw per sample (inference, PAPER.md:322)"}
    return out


# ------------------------------------------------------------------------------------------------
def run_ours(args) -> int:
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2403_16862_b200 import raster           # raises when the CUDA library is missing
    from paper_2403_16862_b200.workloads import CONFIGS, make_workload

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    raster.load()
    assert FLAGS_STEP == raster.SAVE_FOR_BACKWARD

    wl = make_workload(args.workload, seed=CONFIGS[args.workload]["seed"] + rank)
    if args.order == "leaf":                              # SURVEY 8d's secondary measurement; the headline order is the sampler's
        from paper_2403_16862_b200.workloads import leaf_coherent_order
        wl = leaf_coherent_order(wl)
    W, H, D, N = wl.cam.width, wl.cam.height, wl.D, wl.N
    stream = torch.cuda.current_stream()
    # L2 hygiene: a working set that fits the 126 MB L2 would be timed L2-warm, so small workloads rotate through
    # enough independent buffer sets (inputs, workspace, outputs) that a set is evicted before it comes round again
    in_bytes = sum(a.nbytes for a in (wl.pos, wl.opacity, wl.feat, wl.g_img, wl.g_alpha))
    set_bytes = in_bytes + raster.inpc_raster_workspace_bytes(N, D, W, H, FLAGS_STEP) + (W * H * (D + 1) + N * (D + 3)) * 4
    n_sets = 1 if in_bytes > L2_BYTES else max(4, int(-(-3 * L2_BYTES // set_bytes)))
    sets = [make_step_functions(raster, wl, dev, stream) for _ in range(n_sets)]
    fwd0, bwd0, T = sets[0]
    cam, ws = T["cam"], T["ws"]
    turn = [0]

    def fwd(f=FLAGS_STEP):
        sets[turn[0] % n_sets][0](f)

    def bwd():
        sets[turn[0] % n_sets][1]()

    do_bwd = bool(wl.backward)          # BASELINE.json: the inference config is forward only

    def step():
        if do_bwd:
            fwd()
            bwd()
        else:
            fwd(FLAGS_FWD)
        turn[0] += 1

    def fwd_only():
        fwd(FLAGS_FWD)
        turn[0] += 1

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        """-> (total ms of exactly `steps` calls, per-call ms list); CUDA events on the launch stream."""
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        barrier()
        ev[0].record(stream)
        for i in range(steps):
            fn()
            ev[i + 1].record(stream)
        barrier()
        per = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
        return ev[0].elapsed_time(ev[steps]), per

    def med_min(per):
        s = sorted(per)
        return s[len(s) // 2], s[0]

    clocks = ClockSampler(local_rank) if rank == 0 else None

    def windowed(fn, steps):
        if clocks:
            with clocks.window():
                return timed(fn, steps)
        return timed(fn, steps)

    for _ in range(max(args.warmup, 3) * (2 if n_sets > 1 else 1)):
        step()
    torch.cuda.synchronize()
    stats = raster.inpc_raster_get_stats(ws)
    n_frag = stats["n_fragments"]

    # ---- the headline: exactly K fwd+bwd steps, device-resident inputs -------------------------------
    l0 = raster.inpc_raster_launch_count()
    ms_total, per_step = windowed(step, args.steps)
    launches = raster.inpc_raster_launch_count() - l0
    ms_total, units = aggregate_over_ranks(ms_total, float(n_frag) * args.steps, dev)
    ms_step = ms_total / args.steps
    value = throughput(units, ms_total)
    ms_step_med, ms_step_min = med_min(per_step)

    # ---- forward only (inference flags) ---------------------------------------------------------------
    for _ in range(3):
        fwd_only()
    ms_fwd_total, per_fwd = windowed(fwd_only, args.steps)
    ms_fwd_total, _ = aggregate_over_ranks(ms_fwd_total, 0.0, dev)
    ms_fwd = ms_fwd_total / args.steps
    ms_fwd_med, ms_fwd_min = med_min(per_fwd)

    # ---- per-stage device times (library-side CUDA events on the launching stream; every kernel alone) -----
    raster.inpc_raster_set_kernel_timing(True)
    raster.inpc_raster_get_kernel_times(reset=True)
    ms_staged, _ = windowed(step, args.steps)
    stages = raster.inpc_raster_get_kernel_times(reset=True)
    raster.inpc_raster_set_kernel_timing(False)

    # ---- end to end: host buffers in, host buffers out, copies inside the timed region ----------------
    pos, op, feat, g_img, g_alpha = T["pos"], T["op"], T["feat"], T["g_img"], T["g_alpha"]
    img, alpha, d_feat, d_op, d_uv = T["img"], T["alpha"], T["d_feat"], T["d_op"], T["d_uv"]
    flags = FLAGS_STEP if do_bwd else FLAGS_FWD
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_in = [pin(wl.pos), pin(wl.opacity), pin(wl.feat), pin(wl.g_img), pin(wl.g_alpha)]
    d_in = [pos, op, feat, g_img, g_alpha]
    d_out = [img, alpha, d_feat, d_op, d_uv]
    if not do_bwd:                                        # forward only: no output gradients in, no gradients out
        h_in, d_in, d_out = h_in[:3], d_in[:3], d_out[:2]
    h_out = [torch.empty(t.shape, dtype=t.dtype).pin_memory() for t in d_out]
    h2d = sum(t.numel() * t.element_size() for t in h_in)
    d2h = sum(t.numel() * t.element_size() for t in h_out)

    # Three streams, two buffer sets: step i's host->device copy, step i-1's forward + backward and step i-2's
    # device->host copy overlap (PCIe is full duplex); every step still copies ITS inputs in and ITS results out
    # inside the timed region.
    s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    esets = []
    for b in range(2):
        di = d_in if b == 0 else [torch.empty_like(t) for t in d_in]
        do = d_out if b == 0 else [torch.empty_like(t) for t in d_out]
        wsb = ws if b == 0 else raster.alloc_workspace(N, D, W, H, flags, dev)
        ho = h_out if b == 0 else [torch.empty(t.shape, dtype=t.dtype).pin_memory() for t in d_out]
        esets.append({"d_in": di, "d_out": do, "ws": wsb, "h_out": ho,
                      "in_ready": torch.cuda.Event(), "done": torch.cuda.Event(), "out_free": torch.cuda.Event()})

    def e2e_pipeline(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        s_in.wait_stream(stream); s_out.wait_stream(stream)
        e0.record(s_in)
        for i in range(steps):
            S = esets[i % 2]
            if i >= 2:
                s_in.wait_event(S["done"])               # step i-2 has finished reading these inputs
            with torch.cuda.stream(s_in):
                for h, d in zip(h_in, S["d_in"]):
                    d.copy_(h, non_blocking=True)
                S["in_ready"].record(s_in)
            stream.wait_event(S["in_ready"])
            if i >= 2:
                stream.wait_event(S["out_free"])         # step i-2's results have left the device
            p_, o_, f_ = S["d_in"][:3]
            gi_, ga_ = S["d_in"][3:] if do_bwd else (None, None)
            im_, al_ = S["d_out"][:2]
            df_, dop_, du_ = S["d_out"][2:] if do_bwd else (None, None, None)
            raster.inpc_raster_forward(p_, o_, f_, cam, out_feat=im_, out_alpha=al_, workspace=S["ws"], flags=flags,
                                       stream=stream)
            if do_bwd:
                raster.inpc_raster_backward(p_, o_, f_, cam, gi_, ga_, S["ws"], grad_feat=df_, grad_opacity=dop_,
                                            grad_uv=du_, stream=stream)
            S["done"].record(stream)
            s_out.wait_event(S["done"])
            with torch.cuda.stream(s_out):
                for d, h in zip(S["d_out"], S["h_out"]):
                    h.copy_(d, non_blocking=True)
                S["out_free"].record(s_out)
        e1.record(s_out)
        stream.wait_stream(s_out)
        barrier()
        return e0.elapsed_time(e1)

    def e2e_step():                                       # the same, one stream, nothing overlapped
        for h, d in zip(h_in, d_in):
            d.copy_(h, non_blocking=True)
        fwd0(flags)
        if do_bwd:
            bwd0()
        for d, h in zip(d_out, h_out):
            h.copy_(d, non_blocking=True)

    e2e_steps = max(2, min(args.steps, 50))               # the same K steps as the device-resident figure (bounded: 6 ms each)
    e2e_step()
    ms_e2e_serial = timed(e2e_step, e2e_steps)[0] / e2e_steps
    e2e_pipeline(2)
    if clocks:
        with clocks.window():
            ms_e2e_total = e2e_pipeline(e2e_steps)
    else:
        ms_e2e_total = e2e_pipeline(e2e_steps)
    ms_e2e_total, units_e2e = aggregate_over_ranks(ms_e2e_total, float(n_frag) * e2e_steps, dev)
    clock_info = clocks.finish() if clocks else None

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    wstats = workload_statistics(raster, wl, T, dev) if not args.no_stats else {"note": "skipped (--no-stats)"}

    # ---- roofline --------------------------------------------------------------------------------------
    peak, peak_src = measured_peak_gbs()
    P = W * H
    alg = algorithmic_bytes(N, n_frag, P, D)
    per_stage = {k: (ms / n if n else 0.0) for k, (ms, n) in stages.items()}
    step_stage_ms = {k: ms / args.steps for k, (ms, n) in stages.items() if n}
    kernels = {k: v for k, v in step_stage_ms.items() if k.startswith("k_")}
    traffic = ncu_traffic(args.workload)
    groups = {}
    for g in ("a1_a2", "a3_a4", "a5_walk", "a5_out"):
        g_ms = sum(v for k, v in step_stage_ms.items() if STAGE_ROWS.get(k) == g)
        if g_ms <= 0:
            continue
        tr = [traffic_of_stage(traffic, k, D, do_bwd) for k in step_stage_ms if STAGE_ROWS.get(k) == g and k.startswith("k_")]
        tr = [t for t in tr if t is not None]
        ach = alg[g] / (g_ms * 1e-3) / 1e9
        groups[g] = {"algorithmic_bytes": alg[g], "ms": g_ms, "achieved": ach, "frac": ach / peak,
                     "kernels": sorted(k for k in step_stage_ms if STAGE_ROWS.get(k) == g),
                     "traffic": sum(tr) if tr else None}
        if ach > peak:
            groups[g]["note"] = ("above 1: the byte model (SURVEY 8d) counts every emitted fragment; this group only touches "
                                 "the fragments blended before the cut-off")
    dom = max(kernels, key=kernels.get)
    rows = STAGE_ROWS[dom]
    worst = min(groups, key=lambda g: groups[g]["frac"])
    roofline = {"bound": "hbm", "kernel": dom, "rows": rows, "achieved": groups[rows]["achieved"], "peak": peak,
                "unit": "GB/s", "frac": groups[rows]["frac"], "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg[rows], "ms_per_launch": per_stage[dom], "ms_rows": groups[rows]["ms"],
                "kernels_of_rows": groups[rows]["kernels"],
                "share_of_step": kernels[dom] / sum(step_stage_ms.values()),
                "traffic": traffic_of_stage(traffic, dom, D, do_bwd), "traffic_source": traffic.get("_note"),
                "furthest_below_roof": {"rows": worst, "frac": groups[worst]["frac"], "ms": groups[worst]["ms"],
                                        "kernels": groups[worst]["kernels"]},
                "note": "achieved = SURVEY 8d algorithmic bytes of the rows the dominant kernel implements / summed launch "
                        "time of the kernels implementing those rows (each timed alone); every group is in roofline_groups, "
                        "the whole step in roofline_step"}
    step_key = "fwd_bwd" if do_bwd else "fwd"
    ach_step = alg[step_key] / (ms_step * 1e-3) / 1e9
    ach_fwd = alg["fwd"] / (ms_fwd * 1e-3) / 1e9
    roofline_step = {"bound": "hbm", "pass": "forward + backward" if do_bwd else "forward only",
                     "algorithmic_bytes": alg[step_key], "achieved": ach_step,
                     "peak": peak, "unit": "GB/s", "frac": ach_step / peak, "frac_of_8TBps_nominal": ach_step / 8000.0,
                     "target_ms_for_50pct_of_8TBps": alg[step_key] / 4000.0 / 1e6,
                     "fwd_only": {"algorithmic_bytes": alg["fwd"], "achieved": ach_fwd, "frac": ach_fwd / peak}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "ms_per_step_median": ms_step_med, "ms_per_step_min": ms_step_min,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload_config(wl, args, n_sets),
        "ms_fwd": ms_fwd, "ms_fwd_median": ms_fwd_med, "ms_fwd_min": ms_fwd_min, "ms_fwd_bwd": ms_step,
        "fragments_per_sec_fwd": throughput(float(n_frag) * world, ms_fwd),
        "fragments_per_step_per_gpu": n_frag, "stats": stats, "workload_statistics": wstats,
        "e2e": {"value": throughput(units_e2e, ms_e2e_total), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e_total / e2e_steps, "steps": e2e_steps,
                "ms_per_step_one_stream": ms_e2e_serial,
                "how": "every step copies its pinned host inputs (pos, opacity, feat, grad_out) H2D, runs forward + "
                       "backward and copies img/alpha/grad_feat/grad_opacity/grad_uv D2H; three streams and two buffer "
                       "sets overlap step i's H2D, step i-1's kernels and step i-2's D2H (ms_per_step_one_stream: "
                       "the same without overlap)"},
        "gpu_launches": launches,
        "roofline": roofline, "roofline_groups": groups, "roofline_step": roofline_step,
        "stage_ms_per_step": step_stage_ms, "stage_timed_ms_per_step": ms_staged / args.steps,
        "l2": {"l2_bytes": L2_BYTES, "input_bytes": h2d, "record_bytes": stats["n_kept"] * (20 + 4 * D),
               "buffer_sets": n_sets,
               "policy": "inputs larger than L2" if n_sets == 1 else
                         f"inputs fit L2: {n_sets} independent buffer sets ({n_sets * set_bytes >> 20} MiB) rotated, one per step"},
        "clocks": clock_info,
    }
    if world == 1 and wl.backward and not args.no_next_rows:
        line["next_rows"] = next_rows(raster, wl, T, dev, stream, n_frag=n_frag, peak_gbs=peak)
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(wl)
        line["cpu_baseline_all_cores"] = cpu_baseline(wl, openmp=True)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="train", choices=["tiny", "1m", "train", "infer", "stress"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--order", default="sampler", choices=["sampler", "leaf"],
                    help="point storage order: the unordered sampler output (headline) or leaf-coherent (secondary, SURVEY 8d)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle leg (profiling runs)")
    ap.add_argument("--no-stats", action="store_true", help="skip the workload statistics (profiling runs)")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the timings of the NEXT rows f1-f4 (profiling runs)")
    ap.add_argument("--print-source-hash", action="store_true", help="print the kernel-source hash a traffic capture is recorded with")
    args = ap.parse_args(argv)
    if args.print_source_hash:
        print(source_hash())
        return 0
    if args.impl == "reference":
        return run_reference(args)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and world == 1:
        # convenience: relaunch under torchrun, one rank per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + \
              (argv if argv is not None else sys.argv[1:])
        return subprocess.call(cmd)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
