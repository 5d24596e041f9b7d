#!/usr/bin/env python
"""bench.py -- mesh-FT throughput of the B200-native deltaMic hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg C] [--impl ours|reference]

One "step" = one pass of the whole hot path over one synthetic workload: dm_mesh_ft_forward (rows A1-A5) then
dm_mesh_ft_backward (rows A1, A6, A7) with a spectrum cotangent resident in HBM.  The metric is (triangle x
frequency) pairs per second over forward+backward; the forward-only / backward-only rates and the "ms per render
at 128^3" (dm_render of the same workload, with its stage split) ride along in the same JSON line.

Default workload at N=1: config 4 of BASELINE.json (surface mode, 20 membranes, 102 400 triangles, 128^3 grid), the
configuration the north_star target is quoted on.  N>1 (torchrun): every rank processes its own mesh of the same
recipe (seed + rank) -- independent problems, no data-path collective, weak scaling; value = all ranks' pairs / max time.

--impl reference times the fp64 CPU oracle (oracle/, as it stands) on a bounded frequency sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "mesh-FT (triangle*frequency) pairs/s fwd+bwd"
UNIT = "pairs/s"
# SURVEY.md section 8(d) / DESIGN.md section 7: algorithmic FP32 lane-ops per (triangle, frequency) pair
FLOOR_OPS = {"fwd": {0: 26.0, 1: 23.0}, "bwd": {0: 60.0, 1: 60.0}}
FP32_LANES_PER_CLK_PER_SM = 128


def _cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    import platform
    return platform.processor() or platform.machine() or "unknown"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d.get("sm_max_mhz", 1965.0)), "MEASURED_PEAKS.json sm_max_mhz"
    return 1965.0, "fallback clocks.max.sm 1965 MHz (B200_PROFILING.md)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""

    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self._stop = threading.Event()
        self._thr = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [p.strip() for p in out.strip().split(",")]
                if len(parts) >= 7:
                    self.rows.append(parts)
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows), "power_w_max": max(float(r[2]) for r in self.rows)}


def oracle_sample(w, n_freq: int, seed: int = 0):
    """Times the oracle (forward + backward) on ``n_freq`` random stored frequencies of workload ``w``."""
    import oracle
    from workloads.configs import spectrum_cotangent

    rng = np.random.default_rng(seed)
    idx = np.sort(rng.choice(w.n_k, size=min(n_freq, w.n_k), replace=False))
    G = spectrum_cotangent(w).reshape(-1)[idx].astype(np.complex128)
    t0 = time.perf_counter()
    oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, flat_indices=idx)
    t1 = time.perf_counter()
    oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, G, flat_indices=idx)
    t2 = time.perf_counter()
    pairs = float(w.faces.shape[0]) * len(idx)
    return {"pairs": pairs, "fwd_s": t1 - t0, "bwd_s": t2 - t1, "n_freq": int(len(idx)), "cores": oracle.num_threads()}


def oracle_sample_single_thread(cfg: int, n_freq: int):
    """The same sample with the oracle's OpenMP loop on ONE thread ("once single-threaded"):
    a child process with OMP_NUM_THREADS=1, because the thread count is fixed when libgomp starts."""
    code = ("import json, sys; sys.path.insert(0, %r); import bench; from workloads import build_workload; "
            "o = bench.oracle_sample(build_workload(%d), %d); print('ORACLE1 ' + json.dumps(o))" % (ROOT, cfg, n_freq))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600, env=env).stdout
        for line in out.splitlines():
            if line.startswith("ORACLE1 "):
                return json.loads(line[8:])
    except Exception:
        pass
    return None


def ncu_summary():
    """Numbers taken from the committed ncu capture of the dominant kernel (profiles/r02_ncu_summary.json: DRAM bytes per
    full-grid launch, issued instructions per pair, pipe utilisation), with the command that produced them.  Static
    evidence, labelled as such; absent file = absent keys."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_summary.json")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        return json.load(f)


def time_config(dm, cfg: int, warmup: int, steps: int):
    """Forward / backward times of another BASELINE.json config (device-resident inputs, L2 flushed), for the extra
    roofline entries of the JSON line."""
    import torch
    from workloads import build_workload
    from workloads.configs import spectrum_cotangent

    w = build_workload(cfg)
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    vd = torch.as_tensor(w.vertices, device="cuda")
    Gd = torch.as_tensor(spectrum_cotangent(w), device="cuda")
    F = torch.empty(w.spectrum_shape, dtype=torch.complex64, device="cuda")
    dv = torch.empty((w.vertices.shape[0], 3), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    fw, bw, bk = [], [], []
    for it in range(warmup + steps):
        flush.fill_(1)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        plan.mesh_ft_forward(vd, out=F)
        ev[1].record()
        plan.mesh_ft_backward(vd, Gd, out=dv)
        ev[2].record()
        k = plan.stage_ms()["mesh_ft"]
        if it >= warmup:
            fw.append(ev[0].elapsed_time(ev[1]))
            bw.append(ev[1].elapsed_time(ev[2]))
            bk.append(k)
    plan.close()
    return w, float(np.median(fw)), float(np.median(bw)), float(np.median(bk))


def run_reference(args):
    """The reference arm of this tier = the oracle, timed on host cores on a bounded sample of the workload."""
    from workloads import build_workload

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = build_workload(args.cfg)
    n_freq = max(8, int(args.ref_freqs))
    for _ in range(max(0, args.warmup)):
        oracle_sample(w, max(4, n_freq // 8))
    res = [oracle_sample(w, n_freq, seed=s) for s in range(max(1, args.steps))]
    t = sum(r["fwd_s"] + r["bwd_s"] for r in res) / len(res)
    value = res[0]["pairs"] / t
    sample = f"{res[0]['n_freq']} random stored frequencies x all {w.faces.shape[0]} triangles per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "cfg": args.cfg, "mode": "surface" if w.mode else "volume",
                   "n_triangles": int(w.faces.shape[0]), "grid": list(w.n), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": res[0]["cores"], "cpu_model": _cpu_model(), "kind": "oracle", "sample": sample,
                         "fwd_pairs_s": res[0]["pairs"] / np.mean([r["fwd_s"] for r in res]),
                         "bwd_pairs_s": res[0]["pairs"] / np.mean([r["bwd_s"] for r in res])},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_sharded(args):
    """--shard slab: ONE problem (config --cfg) whose stored spectrum is sharded over the ranks by x-slab (SURVEY.md
    section 8(e)): forward = every rank's rows + one all-gather of F, backward = every rank's rows +
    one all-reduce of dL/dv (NCCL).  Strong scaling: value = the problem's pairs / max-over-ranks time."""
    import torch
    import torch.distributed as dist

    import paper_2303_10440_b200 as dm
    from paper_2303_10440_b200.sharding import sharded_mesh_ft_backward, sharded_mesh_ft_forward
    from workloads import build_workload
    from workloads.configs import spectrum_cotangent

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dm.load_library()
    if world > 1:
        # which algorithm / transport (NVLS, P2P) the collectives took; left on stderr so that whoever launched the ranks
        # sees the communicator lines of every rank
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w = build_workload(args.cfg)                      # the same mesh on every rank
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    vd = torch.as_tensor(w.vertices, device="cuda")
    Gd = torch.as_tensor(spectrum_cotangent(w), device="cuda")
    F = torch.zeros(w.spectrum_shape, dtype=torch.complex64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    hv = torch.as_tensor(w.vertices).pin_memory()
    hg = torch.as_tensor(np.random.default_rng(10 + w.seed).standard_normal(w.n).astype(np.float32)).pin_memory()
    himg = torch.empty(w.n, dtype=torch.float32).pin_memory()
    hdv = torch.empty((w.vertices.shape[0], 3), dtype=torch.float32).pin_memory()
    gimg = torch.empty(w.n, dtype=torch.float32, device="cuda")
    ggrad = torch.empty(w.n, dtype=torch.float32, device="cuda")
    Gimg = torch.empty(w.spectrum_shape, dtype=torch.complex64, device="cuda")

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step(ev):
        flush.fill_(1)
        ev[0].record(stream)
        sharded_mesh_ft_forward(plan, vd, out=F)
        ev[1].record(stream)
        dv = sharded_mesh_ft_backward(plan, vd, Gd)
        ev[2].record(stream)
        return dv

    def e2e_step():
        vd.copy_(hv, non_blocking=True)
        ggrad.copy_(hg, non_blocking=True)
        sharded_mesh_ft_forward(plan, vd, out=F)
        plan.spectrum_to_image(F, w.psf_cov, out=gimg)
        himg.copy_(gimg, non_blocking=True)
        plan.image_to_spectrum_cotangent(ggrad, w.psf_cov, out=Gimg)
        hdv.copy_(sharded_mesh_ft_backward(plan, vd, Gimg), non_blocking=True)

    def new_ev():
        return [torch.cuda.Event(enable_timing=True) for _ in range(3)]

    for _ in range(max(args.warmup, 0)):
        step(new_ev())
    launches0 = plan.launch_count()
    barrier()
    evs = [new_ev() for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        for ev in evs:
            step(ev)
        barrier()
    launches = plan.launch_count() - launches0
    fwd_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    bwd_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    e2e_step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_n = max(1, min(args.steps, 3))
    e0.record(stream)
    for _ in range(e2e_n):
        e2e_step()
    e1.record(stream)
    barrier()
    # the other way to use N GPUs, for comparison: every rank the WHOLE problem on its own (no collective), weak scaling
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    plan.mesh_ft_forward(vd, out=F)
    plan.mesh_ft_backward(vd, Gd)
    barrier()
    r0.record(stream)
    for _ in range(e2e_n):
        flush.fill_(1)
        plan.mesh_ft_forward(vd, out=F)
        plan.mesh_ft_backward(vd, Gd)
    r1.record(stream)
    barrier()
    t = torch.tensor([fwd_ms + bwd_ms, fwd_ms, bwd_ms, e0.elapsed_time(e1) / e2e_n, r0.elapsed_time(r1) / e2e_n],
                     dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    step_ms, fwd_ms, bwd_ms, e2e_ms, rep_ms = (float(x) for x in t.tolist())
    if rank == 0:
        sm_max_mhz, peak_src = _peaks()
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        peak = FP32_LANES_PER_CLK_PER_SM * n_sm * sm_max_mhz * 1e6 / 1e12 * world
        pairs = float(w.pairs)
        achieved = FLOOR_OPS["bwd"][w.mode] * pairs / (bwd_ms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": pairs / (step_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "cfg": w.cfg, "mode": "surface" if w.mode else "volume",
                       "n_triangles": int(w.faces.shape[0]), "grid": list(w.n), "pairs_per_pass": pairs,
                       "l2": "flushed between timed iterations (256 MB write)",
                       "parallelism": f"x-slab of the stored spectrum over {world} rank(s); all-gather of F, all-reduce of dL/dv"},
            "fwd_ms": fwd_ms, "bwd_ms": bwd_ms,
            "e2e": {"value": pairs / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": hv.numel() * 4 + hg.numel() * 4, "d2h_bytes_per_step": himg.numel() * 4 + hdv.numel() * 4,
                    "what": "sharded forward + all-gather + image stage, cotangent stage + sharded backward + all-reduce, "
                            "pinned host buffers in and out on every rank"},
            "gpu_launches": int(launches), "clocks": clk.summary(),
            "replicas": {"value": world * pairs / (rep_ms * 1e-3), "unit": UNIT, "ms_per_step": rep_ms, "scaling": "weak",
                         "steps": e2e_n, "what": "every rank the whole problem on its own, no collective (includes the L2 flush)"},
            "roofline": {"bound": "alu", "kernel": "dm_k_backward_fast + all-reduce (whole sharded backward)",
                         "achieved": achieved, "peak": peak, "unit": "T lane-op/s over all ranks", "frac": achieved / peak,
                         "traffic": None, "peak_source": f"{world} x 128 x {n_sm} SMs x {sm_max_mhz:.0f} MHz ({peak_src})"},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2303_10440_b200 as dm
    from workloads import build_workload
    from workloads.configs import image_cotangent, spectrum_cotangent

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dm.load_library()  # fails loudly when the CUDA extension is missing
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # every rank owns one mesh of the same recipe (independent problems; seed offset = rank)
    w = build_workload(args.cfg, seed_offset=rank)
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    slab = None
    if args.x_slab:  # profiling aid: restrict the mesh-FT calls to rows [a, b) of the stored spectrum (not a bench number)
        slab = tuple(int(x) for x in args.x_slab.split(":"))
        plan.set_slab(*slab)
    vd = torch.as_tensor(w.vertices, device="cuda")
    Gd = torch.as_tensor(spectrum_cotangent(w), device="cuda")
    F = torch.empty(w.spectrum_shape, dtype=torch.complex64, device="cuda")
    dv = torch.empty((w.vertices.shape[0], 3), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step(ev):
        flush.fill_(1)  # L2 flush between timed iterations (outside the events)
        ev[0].record(stream)
        plan.mesh_ft_forward(vd, out=F)
        ev[1].record(stream)
        plan.mesh_ft_backward(vd, Gd, out=dv)
        ev[2].record(stream)

    def new_ev():
        return [torch.cuda.Event(enable_timing=True) for _ in range(3)]

    for _ in range(max(args.warmup, 0)):
        step(new_ev())
    launches0 = plan.launch_count()
    barrier()
    evs = [new_ev() for _ in range(args.steps)]
    bwd_kernel_ms = []
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for ev in evs:
            step(ev)
            bwd_kernel_ms.append(plan.stage_ms()["mesh_ft"])  # syncs; = A1 + A6 kernel time of this step's backward
        barrier()
        t_wall = time.perf_counter() - t_wall0
    launches = plan.launch_count() - launches0
    fwd_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    bwd_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    step_ms = fwd_ms + bwd_ms
    t = torch.tensor([step_ms, fwd_ms, bwd_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    step_ms, fwd_ms, bwd_ms = (float(x) for x in t.tolist())
    pairs = float(w.pairs) if slab is None else float(w.faces.shape[0]) * (slab[1] - slab[0]) * w.n[1] * (w.n[2] // 2 + 1)
    if slab is not None:
        if rank == 0:
            print(json.dumps({"profiling_only": True, "x_slab": list(slab), "pairs": pairs, "fwd_ms": fwd_ms, "bwd_ms": bwd_ms,
                              "bwd_kernel_ms": float(np.mean(bwd_kernel_ms))}), flush=True)
        return

    # ---- end to end through the public API with HOST buffers (render + render_backward) ---------------------------
    hv = torch.as_tensor(w.vertices).pin_memory()
    hg = torch.as_tensor(image_cotangent(w) if w.cfg in (1, 3, 5) else
                         np.random.default_rng(10 + w.seed).standard_normal(w.n).astype(np.float32)).pin_memory()
    himg = torch.empty(w.n, dtype=torch.float32).pin_memory()
    hdv = torch.empty((w.vertices.shape[0], 3), dtype=torch.float32).pin_memory()
    gimg = torch.empty(w.n, dtype=torch.float32, device="cuda")
    ggrad = torch.empty(w.n, dtype=torch.float32, device="cuda")
    render_ms, stage = [], {}

    def e2e_step():
        vd.copy_(hv, non_blocking=True)
        ggrad.copy_(hg, non_blocking=True)
        plan.render(vd, w.psf_cov, out=gimg)
        himg.copy_(gimg, non_blocking=True)
        plan.render_backward(vd, w.psf_cov, ggrad, out=dv)
        hdv.copy_(dv, non_blocking=True)

    e2e_step()
    barrier()
    e2e_n = max(1, min(args.steps, 3))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_n):
        e2e_step()
    e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1) / e2e_n
    t = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_ms = float(t.item())
    # ms per render (forward only) with its stage split
    for _ in range(3):
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record(stream)
        plan.render(vd, w.psf_cov, out=gimg)
        r1.record(stream)
        stage = plan.stage_ms()
        render_ms.append(r0.elapsed_time(r1))
    # narrow band (frequencies with h_hat > 1 % only), reported beside the full-grid numbers
    plan.set_narrow_band(w.psf_cov, 0.01)
    nb = {"cutoff": 0.01, "fwd_ms": [], "bwd_ms": []}
    for _ in range(3):
        ev = new_ev()
        step(ev)
        torch.cuda.synchronize()
        nb["fwd_ms"].append(ev[0].elapsed_time(ev[1]))
        nb["bwd_ms"].append(ev[1].elapsed_time(ev[2]))
    nb["in_band_fraction"] = float((torch.view_as_real(F).abs().sum(-1) > 0).float().mean())
    nb["fwd_ms"], nb["bwd_ms"] = float(np.median(nb["fwd_ms"])), float(np.median(nb["bwd_ms"]))
    plan.set_narrow_band(None)
    h2d = hv.numel() * 4 + hg.numel() * 4
    d2h = himg.numel() * 4 + hdv.numel() * 4

    if rank == 0:
        sm_max_mhz, peak_src = _peaks()
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        clocks = clk.summary()
        peak = FP32_LANES_PER_CLK_PER_SM * n_sm * sm_max_mhz * 1e6 / 1e12  # T lane-op/s
        bk_ms = float(np.mean(bwd_kernel_ms))
        achieved = FLOOR_OPS["bwd"][w.mode] * pairs / (bk_ms * 1e-3) / 1e12
        sm_mhz = clocks.get("sm_mhz") or sm_max_mhz
        ncu = ncu_summary()
        roofline = {
            "bound": "alu", "kernel": "dm_k_backward_fast (A6, dominant)", "achieved": achieved, "peak": peak,
            "unit": "T lane-op/s (FP32 issue: 128 lanes/clk/SM)", "frac": achieved / peak,
            "traffic": (ncu or {}).get("dram_bytes_per_full_grid_launch"),
            "peak_source": f"128 x {n_sm} SMs x {sm_max_mhz:.0f} MHz ({peak_src}); DESIGN.md section 7",
            "frac_at_measured_clock": achieved / (peak * sm_mhz / sm_max_mhz),
            "algorithmic_ops_per_pair": FLOOR_OPS["bwd"][w.mode], "kernel_ms": bk_ms,
        }
        # forward: the strip walk issues fewer instructions per pair than the itemised per-pair floor (it shares vertex work
        # along the strip), so the fraction is taken against min(floor, issued): it can never exceed the issue utilisation
        fwd_issued = ((ncu or {}).get("forward") or {}).get("issued_instr_per_pair_full_grid") if w.cfg == 4 else None
        fwd_ops = min(FLOOR_OPS["fwd"][w.mode], fwd_issued) if fwd_issued else FLOOR_OPS["fwd"][w.mode]
        roofline["forward"] = {"achieved": fwd_ops * pairs / (fwd_ms * 1e-3) / 1e12,
                               "frac": fwd_ops * pairs / (fwd_ms * 1e-3) / 1e12 / peak,
                               "algorithmic_ops_per_pair": fwd_ops, "itemised_floor_ops_per_pair": FLOOR_OPS["fwd"][w.mode],
                               "issued_instr_per_pair": fwd_issued,
                               "note": "ops per pair = min(itemised floor, issued instructions per pair measured by ncu at cfg 4)"}
        if ncu:
            roofline["ncu"] = ncu
        # the other full-size configs (volume mode carries 5 more operations per pair against the same floor)
        extra = {}
        for c in [int(x) for x in args.extra_cfgs.split(",") if x.strip()]:
            if c == w.cfg or world > 1:
                continue
            wc, f_ms, b_ms, k_ms = time_config(dm, c, 3 if c <= 2 else 1, 10 if c <= 2 else (2 if c < 5 else 1))
            pc = float(wc.pairs)
            extra[f"cfg{c}"] = {
                "mode": "surface" if wc.mode else "volume", "pairs_per_pass": pc, "fwd_ms": f_ms, "bwd_ms": b_ms,
                "bwd_kernel_ms": k_ms, "fwd_bwd_pairs_s": pc / ((f_ms + b_ms) * 1e-3),
                "frac_backward": FLOOR_OPS["bwd"][wc.mode] * pc / (k_ms * 1e-3) / 1e12 / peak,
                "frac_forward": FLOOR_OPS["fwd"][wc.mode] * pc / (f_ms * 1e-3) / 1e12 / peak}
        roofline["other_configs"] = extra
        o = oracle_sample(w, args.ref_freqs)
        o1 = oracle_sample_single_thread(w.cfg, max(8, args.ref_freqs // 8))
        sample = f"{o['n_freq']} random stored frequencies x all {w.faces.shape[0]} triangles, forward+backward"
        # the CPU image stage (PSF multiply + numpy irfftn, fp64) on this grid, for the "ms per render" stage split
        import oracle as _oracle
        t0 = time.perf_counter()
        _oracle.spectrum_to_image(F.cpu().numpy(), w.n, w.spacing, w.origin, w.psf_cov.astype(np.float64))
        cpu_image_stage_ms = (time.perf_counter() - t0) * 1e3
        line = {
            "metric": METRIC, "value": world * pairs / (step_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "cfg": w.cfg, "mode": "surface" if w.mode else "volume",
                       "n_triangles": int(w.faces.shape[0]), "n_vertices": int(w.vertices.shape[0]), "grid": list(w.n),
                       "pairs_per_pass": pairs, "l2": "flushed between timed iterations (256 MB write)",
                       "parallelism": f"replicas x{world}"},
            "fwd_pairs_s": world * pairs / (fwd_ms * 1e-3), "bwd_pairs_s": world * pairs / (bwd_ms * 1e-3),
            "fwd_ms": fwd_ms, "bwd_ms": bwd_ms,
            "fwd_ms_median": float(np.median([e[0].elapsed_time(e[1]) for e in evs])),
            "bwd_ms_median": float(np.median([e[1].elapsed_time(e[2]) for e in evs])),
            "render_ms": float(np.median(render_ms)), "render_stage_ms": stage,
            "e2e": {"value": world * pairs / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms,
                    "what": "dm_render + dm_render_backward with pinned host vertices/dL_dimage in, image/dL_dv out"},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
            "cpu_baseline": {"value": o["pairs"] / (o["fwd_s"] + o["bwd_s"]), "unit": UNIT, "cores": o["cores"],
                             "cpu_model": _cpu_model(), "kind": "oracle", "sample": sample, "fwd_pairs_s": o["pairs"] / o["fwd_s"],
                             "bwd_pairs_s": o["pairs"] / o["bwd_s"],
                             "single_thread": None if o1 is None else {
                                 "value": o1["pairs"] / (o1["fwd_s"] + o1["bwd_s"]), "cores": o1["cores"],
                                 "sample": f"{o1['n_freq']} random stored frequencies x all triangles",
                                 "fwd_pairs_s": o1["pairs"] / o1["fwd_s"], "bwd_pairs_s": o1["pairs"] / o1["bwd_s"]},
                             "image_stage_ms": cpu_image_stage_ms,
                             "image_stage": "PSF multiply + numpy irfftn (fp64) of one spectrum of this grid"},
            "narrow_band": nb, "wall_s_timed_region": t_wall,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=4, help="BASELINE.json config 1..5 (default 4, the target config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-freqs", type=int, default=192, help="stored frequencies per oracle sample")
    ap.add_argument("--shard", default="auto", choices=["auto", "replicas", "slab"],
                    help="slab: ONE problem sharded by x-slab of the stored spectrum (all-gather of F, all-reduce of dL/dv over "
                         "NCCL), strong scaling, with the replica figure under the key 'replicas'; replicas: every rank its own "
                         "problem, weak scaling, no data-path collective; auto (default): replicas at --gpus 1, slab above")
    ap.add_argument("--extra-cfgs", default="1,2,3,5", help="other BASELINE.json configs timed (N=1 only) for the extra roofline "
                    "entries; '' switches them off")
    ap.add_argument("--x-slab", default="", help="a:b -- profiling aid (ncu counters overflow on the 0.4 s full-grid launch): run "
                    "forward/backward on rows [a,b) of the spectrum only and print a short line that is NOT a bench result")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.shard == "auto":
        args.shard = "slab" if max(args.gpus, world) > 1 else "replicas"
    if args.impl == "ours" and args.gpus != world:
        raise SystemExit(f"bench.py --gpus {args.gpus} must be launched with one process per GPU (python -m torch.distributed.run "
                         f"--nproc-per-node {args.gpus} ... bench.py --gpus {args.gpus}); this process sees WORLD_SIZE={world}")
    if args.impl == "reference":
        run_reference(args)
    elif args.shard == "slab":
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
