#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (S1-S8: project/cull, tile ranges, key emission,
per-tile radix sort, forward composite, loss stage, backward composite, per-surfel chain)
over one synthetic workload of BASELINE.json (default and headline: configs[1], 64x1024, 300k surfels).

    python bench.py --gpus N --steps K --warmup W            (ours; torchrun for N > 1)
    python bench.py --impl reference --steps K --warmup W    (the CPU oracle, as it stands)
    python bench.py --config {tiny,nc,kitti,large,batch}     (the other BASELINE.json configs; nc = headline)

Prints ONE JSON line (rank 0).  metric = Gaussian-pixel intersections/s for forward+backward
(intersection = contributing (pixel, surfel) pair, counted on the device and equal to the
oracle's count); ms_per_step = fwd+loss+bwd ms per step (ms_per_frame = per rendered frame).  Timing: CUDA events
around each graph-replayed step on the launching stream, a 256 MiB L2 scrub before every timed step,
max over ranks; mean, median, p10 and p90 of the per-step times.  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import csv
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

UNIT = "intersections/s"

# Algorithmic work per contributing pair, counted once from the oracle's expression tree
# (oracle/lgs_oracle.cpp composite_pixel / lgs_oracle_backward) and frozen -- DESIGN.md "Roofline".
FWD_FP32_PER_PAIR, FWD_SFU_PER_PAIR = 31, 2
BWD_FP32_PER_PAIR, BWD_SFU_PER_PAIR = 89, 3
FP32_LANES, SFU_LANES = 128, 16          # per SM (B200_PROFILING.md); the SM count is read from the device

# The workloads (BASELINE.json configs).  `k16`: algorithmic key count of SURVEY.md 8(d) -- (surfel, 16x16 tile) pairs of
# the oracle's list reference, summed over the frames of a step (oracle.tile_lists(..., tile=16); seeds fixed) -- NOT the
# implementation's own key count, which is larger because it lists per 8x4 tile.  Re-counted by the cpu_baseline leg.
# `nfp`: N_fp of SURVEY.md 8(d) -- (frame, surfel) pairs with a non-empty FOOTPRINT (some beam meets the surfel inside its
# 3 sigma ellipse; oracle.footprint_surfels, summed over the frames), which is what the record / partial-sum terms of
# B_alg count; the implementation's own n_visible (non-empty pixel RECT, a superset) is reported beside it.
# tests/test_bench_constants.py recounts both with the oracle.
CONFIGS = {
    "tiny": dict(maker="make_tiny", shape="64x256, 2000 surfels", name="tiny", k16=2_532, nfp=875),
    "nc": dict(maker="make_newer_college", shape="64x1024, 300k surfels", name="newer_college_shaped", k16=367_601, nfp=196_079),
    "kitti": dict(maker="make_kitti", shape="64x2048, 1M surfels, 10 poses", name="kitti_shaped", k16=3_915_181, nfp=2_829_696),
    "large": dict(maker="make_large_map", shape="128x2048, 4M surfels", name="large_map", k16=670_771, nfp=407_669),
    "batch": dict(maker="make_mapping_batch", shape="8 x 64x1024, 2M surfels", name="mapping_batch", k16=19_957_842, nfp=11_118_274),
}
L2_NOTE = "GPU arm: 256 MiB scrub before every timed step; reference arm: CPU program, no device cache involved"


def config_dict(cfg: str, w) -> dict:
    """The `config` object of the JSON line: identical in both arms (ours / reference), so that the driver's
    same-config check compares like with like; what only one arm knows about its run goes into `run`."""
    return {"workload": workload_string(cfg, w), "frames_per_step": len(w.sensors), "l2": L2_NOTE}
DRAM_CSV = os.path.join(ROOT, "profiles", "r2_kernel_dram_bytes.csv")   # written from an ncu --set full capture


def metric_name(cfg: str) -> str:
    return "fwd+bwd Gaussian-pixel intersections/s (%s)" % CONFIGS[cfg]["shape"]


def workload_string(cfg: str, w) -> str:
    """The same string in both arms (ours / reference)."""
    S = w.sensors[0]
    return "%s %dx%d, %d surfels, %d frame%s per step (fwd+loss+bwd)" % (
        CONFIGS[cfg]["name"], S.H, S.W, w.N, len(w.sensors), "" if len(w.sensors) == 1 else "s")


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            j = json.load(f)
        return float(j["hbm_gbs"]), float(j.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def _ncu_dram_bytes() -> dict:
    """dram__bytes_read.sum + dram__bytes_write.sum per launch and kernel group, from the committed summary of one
    ncu --set full capture (profiles/r2_kernel_dram_bytes.md names the command)."""
    out = {}
    if os.path.exists(DRAM_CSV):
        with open(DRAM_CSV) as f:
            for row in csv.DictReader(f):
                out[row["group"]] = out.get(row["group"], 0.0) + float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.lines, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def wait_first(self, timeout=10.0):
        """nvidia-smi takes ~0.1-1 s to emit its first line: block until it is sampling."""
        t0 = time.perf_counter()
        while self.proc is not None and not self.lines and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)

    def stop(self, t_from=0.0, t_to=float("inf")) -> dict:
        """Statistics over the samples taken in [t_from, t_to] (time.perf_counter() values)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, ln in self.lines:
            if ts < t_from or ts > t_to:
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _workload(cfg: str):
    """The workload of a config and, per frame, the synthetic scan it is compared with (range + normal images)."""
    import workloads
    w = getattr(workloads, CONFIGS[cfg]["maker"])()
    scans = []
    for f, S in enumerate(w.sensors):
        if w.scene is not None:
            scans.append(workloads.simulate_scan(w.scene, S, w.scan_seed + (f if cfg == "batch" else 0)))
        else:
            scans.append(None)       # tiny: the target is the oracle's render of the perturbed surfels (cpu leg / reference arm)
    return w, scans


def _tiny_target(w):
    import oracle
    S = w.sensors[0]
    return oracle.render_forward(w.perturbed_mean, w.quat, w.scale, w.opacity, S).range.astype(np.float32), None


def _oracle_frame(w, S, tgt, tn, keep):
    """One frame through the oracle as it stands: forward + loss + backward. Returns I_c."""
    import oracle
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED)
    lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, keep, **w.lambdas)
    oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, lr.gD, lr.gA, lr.gN, oracle.BOUNDED)
    return fo.stats["I_c"]


def run_reference(args):
    """--impl reference: the fp64 CPU oracle on the box's host cores, same config / metric; a step is a bounded sample
    of the workload (one frame of it: frame k of step k, cycling)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = args.config
    w, scans = _workload(cfg)
    if cfg == "tiny":
        scans = [_tiny_target(w)]
    nf = len(w.sensors)

    def frame(k):
        f = k % nf
        keep = None if w.keep_masks is None else w.keep_masks[f]
        return _oracle_frame(w, w.sensors[f], scans[f][0], scans[f][1], keep)

    for k in range(1 if args.warmup > 0 else 0):
        frame(k)
    t0 = time.perf_counter()
    ic = 0
    for k in range(args.steps):
        ic += frame(k)
    dt = time.perf_counter() - t0
    val = ic / dt
    cores = oracle.num_threads()
    sample = "%d whole frame%s of the workload (forward+loss+backward, bounded mode, OpenMP)" % (args.steps, "" if args.steps == 1 else "s")
    print(json.dumps({
        "impl": "reference", "metric": metric_name(cfg), "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "ms_per_frame": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, w), "run": {"sample": "one frame of the workload per step"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def aggregate_over_ranks(times_ms, units, world: int, device):
    """Whole-job numbers of a replicas-only run: every time is the MAX over ranks, the units
    processed are the SUM over ranks.  Works on any torch.distributed backend (NCCL on the GPUs; the CPU test uses gloo)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], float(u.item())


def _stats(ms_list):
    a = np.asarray(ms_list, dtype=np.float64)
    return {"mean": float(a.mean()), "median": float(np.median(a)), "p10": float(np.percentile(a, 10)),
            "p90": float(np.percentile(a, 90)), "min": float(a.min()), "n": int(a.size)}


class _Problem:
    """Device-side state of one config: parameters, targets, the rasteriser object(s) and the step function."""

    def __init__(self, cfg, w, scans, dev, lgs, torch):
        self.cfg, self.w, self.dev, self.lgs, self.torch = cfg, w, dev, lgs, torch
        self.F = len(w.sensors)
        self.S = w.sensors[0]
        self.host = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in (w.mean, w.quat, w.scale, w.opacity)]
        self.p = [h.to(dev) for h in self.host]
        self.lam = w.lambdas
        self.batched = cfg == "batch"
        # targets per frame (pinned host copies for the end-to-end legs)
        if cfg == "tiny":
            # BASELINE.json configs[0]: the target is a render of the perturbed surfels -- made here with the product itself
            Rt = lgs.Rasterizer(w.N, self.S, 8 * w.N, device=dev)
            Rt.forward(torch.from_numpy(w.perturbed_mean).to(dev), *self.p[1:])
            torch.cuda.synchronize(dev)
            tg = [Rt.range.cpu().numpy().copy()]
            tnn = [None]
            del Rt
        else:
            tg = [s[0] for s in scans]
            tnn = [s[1] for s in scans]
        self.tgt_pin = torch.from_numpy(np.stack(tg)).pin_memory()
        self.tn_pin = None if tnn[0] is None else torch.from_numpy(np.stack(tnn)).pin_memory()
        self.tgt = self.tgt_pin.to(dev)
        self.tn = None if self.tn_pin is None else self.tn_pin.to(dev)
        self.keep = None
        if w.keep_masks is not None:
            self.keep = torch.from_numpy(np.stack(w.keep_masks).astype(np.uint8)).to(dev)
        self.R = None
        self.max_keys = None
        self.world = 1                    # > 1: frame-sharded batch (bench.py --config batch --gpus N)

    def size_keys(self):
        """The key count is data-dependent: overflow -> lgs_query reports the capacity needed -> retry (one host sync,
        before the timed region).  Returns (n_visible, n_keys, n_contrib) per step."""
        lgs, w, torch = self.lgs, self.w, self.torch
        if self.batched:
            probe = lgs.BatchRasterizer(w.N, w.sensors, 1 << 20, device=self.dev)
            probe.forward(*self.p)
            nv, nk, nc, ovf = probe.query()
            del probe
            torch.cuda.empty_cache()
            self.max_keys = int(1.05 * nk) + 4096
            self.R = lgs.BatchRasterizer(w.N, w.sensors, self.max_keys, device=self.dev)
            self.R.forward(*self.p)
            nv, nk, nc, ovf = self.R.query()
            assert not ovf
            return nv, nk, nc
        probe = lgs.Rasterizer(w.N, self.S, 1 << 20, device=self.dev)
        need = 0
        for S in w.sensors:
            probe.set_pose(S.T_ws)
            probe.forward(*self.p)
            need = max(need, probe.query()[1])
        del probe
        torch.cuda.empty_cache()
        self.max_keys = int(1.25 * need) + 1024
        self.R = self.new_rasterizer()
        nv = nk = nc = 0
        for S in w.sensors:
            self.R.set_pose(S.T_ws)
            self.R.forward(*self.p)
            a, b, c, ovf = self.R.query()
            assert not ovf
            nv, nk, nc = nv + a, nk + b, nc + c
        return nv, nk, nc

    def new_rasterizer(self):
        return self.lgs.Rasterizer(self.w.N, self.S, self.max_keys, device=self.dev)

    def step(self, stream, R=None, p=None, tgt=None, tn=None):
        """forward + loss + backward of every frame of the workload (gradients of the frames of a batch summed)."""
        R = self.R if R is None else R
        p = self.p if p is None else p
        tgt = self.tgt if tgt is None else tgt
        tn = self.tn if tn is None else tn
        lam = self.lam
        if self.batched:
            R.forward(*p, stream=stream)
            R.loss_stage(tgt, tn, self.keep, lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False, stream=stream)
            R.backward(*p, stream=stream)
            if self.world > 1:             # frame-sharded batch: the only exchange step of the path
                with self.torch.cuda.stream(stream):
                    self.lgs.all_reduce_gradients((R.g_mean, R.g_quat, R.g_scale, R.g_opacity), self.world)
            return
        for f, S in enumerate(self.w.sensors):
            if self.F > 1:
                R.set_pose(S.T_ws)
            R.forward(*p, stream=stream)
            R.loss_stage(tgt[f], None if tn is None else tn[f], None if self.keep is None else self.keep[f],
                         lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False, stream=stream)
            R.backward(*p, stream=stream)

    def serial_batch_step(self, stream, R1):
        """The batch config as F single-frame calls with accumulate = 1 (what lgs_render_*_batch replaces)."""
        lam = self.lam
        for f, S in enumerate(self.w.sensors):
            R1.set_pose(S.T_ws)
            R1.forward(*self.p, stream=stream)
            R1.loss_stage(self.tgt[f], self.tn[f], self.keep[f], lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"],
                          False, stream=stream)
            R1.backward(*self.p, accumulate=(f > 0), stream=stream)

    def kernels_per_step(self):
        # project, ranges, placement, tile sort x2 (length classes), composite | loss x2 | clear, backward composite, chain
        return (6 + 2 * self.F + 3) if self.batched else 11 * self.F

    def result_signature(self, R=None):
        """(loss scalars, checksums of the gradient buffers) of the last step -- compared between the eager step and the
        replayed graph after the timed loop."""
        R = self.R if R is None else R
        loss = (R.loss5[:, 0] if self.batched else R.loss[:1]).double().cpu()
        sums = [float(t.double().abs().sum()) for t in (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)]
        return loss, sums


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_04127_b200 as lgs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    local_rank %= max(torch.cuda.device_count(), 1)          # (more ranks than GPUs: testing only, ranks share a device)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        # NCCL over NVLink; LGS_BENCH_BACKEND=gloo exercises the multi-rank code path on a box with fewer GPUs than ranks
        backend = os.environ.get("LGS_BENCH_BACKEND", "nccl")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(backend)
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: replicas only: every rank renders the same synthetic workload
    cfg = args.config
    w, scans = _workload(cfg)
    sharded = cfg == "batch" and world > 1
    if sharded:
        # The one place the path shards: the keyframes of a mapping batch are independent given a
        # replicated map.  Every rank renders its contiguous share in one batched call, then ONE all-reduce (NCCL) of the
        # gradient buffers -- inside the timed step.  Total work is fixed: strong scaling.
        mine = lgs.frames_of_rank(len(w.sensors), rank, world)
        if len(mine) == 0:
            raise RuntimeError("more ranks than keyframes (%d > %d)" % (world, len(w.sensors)))
        w.sensors = [w.sensors[f] for f in mine]
        w.keep_masks = [w.keep_masks[f] for f in mine]
        scans = [scans[f] for f in mine]
        args.no_graph = True               # (the collective is enqueued eagerly)
    P = _Problem(cfg, w, scans, dev, lgs, torch)
    P.world = world if sharded else 1
    nv, nk, nc = P.size_keys()             # the only host syncs before the timed region
    R = P.R
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # L2 scrub (> 126 MB L2)

    with torch.cuda.stream(stream):
        P.step(stream)
    stream.synchronize()
    eager_sig = P.result_signature()
    graph = None
    if not args.no_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            P.step(stream)

    def run_step():
        if graph is not None:
            graph.replay()
        else:
            P.step(stream)

    def timed(n, scrub=True, pre=None, post=None, fn=None):
        """Per-step device times (ms); the scrub runs outside the event pair."""
        evs = []
        with torch.cuda.stream(stream):
            for _ in range(n):
                if scrub:
                    flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if pre:
                    pre()
                (fn or run_step)()
                if post:
                    post()
                e1.record(stream)
                evs.append((e0, e1))
        stream.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            flush.zero_()
            run_step()
    clocks = ClockSampler(local_rank)
    clocks.start()
    clocks.wait_first()
    barrier()
    t_wall0 = time.perf_counter()
    step_ms = timed(args.steps, scrub=True)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    total_ms = float(sum(step_ms))
    # The timed region of a short run is shorter than nvidia-smi's sampling period: the same loop is continued,
    # untimed, until the load has lasted >= 0.75 s, and the clocks are the samples of that window.
    if sharded:
        for _ in range(4):           # (a fixed count: the step holds a collective, every rank must run the same number)
            timed(args.steps, scrub=True)
    while not sharded and time.perf_counter() - t_wall0 < 0.75:
        timed(min(args.steps, 100), scrub=True)
    clk = clocks.stop(t_wall0, time.perf_counter())
    clk["window"] = "timed region + identical untimed continuation, %.2f s" % (time.perf_counter() - t_wall0)
    # ---- the replayed graph computed what the eager step computed (loss scalars, gradient checksums)
    graph_sig = P.result_signature()
    check = {"loss_equal": bool(torch.allclose(graph_sig[0], eager_sig[0], rtol=1e-5, atol=0.0)),
             "grad_checksum_rel_diff": max(abs(a - b) / max(abs(b), 1e-30) for a, b in zip(graph_sig[1], eager_sig[1]))}
    assert check["loss_equal"] and check["grad_checksum_rel_diff"] < 1e-4, check     # (float atomics: order noise only)
    warm_ms = float(sum(timed(args.steps, scrub=False)))

    # ---- end to end through the public API with HOST buffers: H2D of the map + scan, step, D2H of grads + loss
    g_bufs = (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)
    g_host = [torch.empty_like(t, device="cpu").pin_memory() for t in g_bufs]
    loss_src = R.loss5 if P.batched else R.loss
    loss_host = torch.empty_like(loss_src, device="cpu").pin_memory()

    def h2d():
        for d, h in zip(P.p, P.host):
            d.copy_(h, non_blocking=True)
        P.tgt.copy_(P.tgt_pin, non_blocking=True)
        if P.tn is not None:
            P.tn.copy_(P.tn_pin, non_blocking=True)

    def d2h():
        for h, d in zip(g_host, g_bufs):
            h.copy_(d, non_blocking=True)
        loss_host.copy_(loss_src, non_blocking=True)

    timed(2, True, h2d, d2h)
    e2e_serial_ms = float(sum(timed(args.steps, True, h2d, d2h)))
    scan_bytes = P.tgt_pin.numel() * 4 + (0 if P.tn_pin is None else P.tn_pin.numel() * 4)
    h2d_bytes = sum(h.numel() * 4 for h in P.host) + scan_bytes
    d2h_bytes = sum(h.numel() * 4 for h in g_host) + loss_host.numel() * 4
    e2e_ms, e2e_note = e2e_serial_ms, "copies and kernels serialised on one stream"
    if not P.batched and P.F == 1 and not args.no_graph:
        e2e_ms = _e2e_pipelined(P, args.steps, torch, dev)
        e2e_note = ("pipelined: three parameter / target / workspace / gradient sets, H2D of the next steps and D2H of the "
                    "previous ones on their own streams under step k's kernels; timed from the first H2D to the last D2H")

    # the same, as a mapping loop runs it: the map and its gradients stay on the device (the optimiser step reads them
    # there, lgs_adam_step); per step only the scan's images come from the host and the loss goes back
    def h2d_scan():
        P.tgt.copy_(P.tgt_pin, non_blocking=True)
        if P.tn is not None:
            P.tn.copy_(P.tn_pin, non_blocking=True)

    def d2h_loss():
        loss_host.copy_(loss_src, non_blocking=True)

    timed(2, True, h2d_scan, d2h_loss)
    e2e_res_ms = float(sum(timed(args.steps, True, h2d_scan, d2h_loss)))

    # ---- per-kernel times, live, with CUDA events on the launching stream (not graph-replayed)
    lgs.lgs_profile_enable(True)
    acc = {}
    nprof = max(3, min(args.steps, 20))
    with torch.cuda.stream(stream):
        for _ in range(nprof):
            # three scrubs (~200 us of GPU work): the whole step is enqueued before the GPU reaches it, so
            # the event pairs bracket kernels running back to back, not the host's launch latency
            flush.zero_(); flush.zero_(); flush.zero_()
            if P.batched or P.F == 1:
                P.step(stream)
            else:                      # (the slots hold one call each: profile the last frame of a multi-pose step)
                R.forward(*P.p, stream=stream)
                R.loss_stage(P.tgt[-1], None if P.tn is None else P.tn[-1], None, stream=stream, **P.lam)
                R.backward(*P.p, stream=stream)
            for k, v in lgs.lgs_profile_read(stream).items():
                acc[k] = acc.get(k, 0.0) + v / nprof
    lgs.lgs_profile_enable(False)

    # ---- measured issue peaks: FFMA and MUFU.EX2 micro-benchmarks of the library, on this device
    scratch = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
    ffma_rate, _ = lgs.lgs_microbench(lgs.LGS_MB_FFMA, scratch, stream=stream)
    mufu_rate, _ = lgs.lgs_microbench(lgs.LGS_MB_MUFU_EX2, scratch, stream=stream)

    extras = {}
    if rank == 0 and cfg == "nc" and not args.no_extras:
        extras = _next_sections(P, R, stream, flush, lgs, torch, args)
    if rank == 0 and cfg == "batch":
        R1 = P.new_rasterizer()
        ser = timed(max(3, args.steps // 4), True, fn=lambda: P.serial_batch_step(stream, R1))
        extras["serial_calls"] = {"ms_per_step": float(np.median(ser)), "ms_per_frame": float(np.median(ser)) / P.F,
                                  "note": "the same %d frames as %d x (lgs_render_forward, loss, lgs_render_backward with "
                                          "accumulate = 1), eager launches, median" % (P.F, P.F)}

    # ---- max over ranks, whole-job throughput
    (total_ms, warm_ms, e2e_ms, e2e_res_ms), units = aggregate_over_ranks([total_ms, warm_ms, e2e_ms, e2e_res_ms],
                                                                          float(nc) * args.steps, world, dev)
    if rank == 0:
        out = _report(args, cfg, P, world, n_sm, nv, nk, nc, total_ms, step_ms, warm_ms, e2e_ms, e2e_note, e2e_serial_ms,
                      e2e_res_ms, h2d_bytes, d2h_bytes, scan_bytes, loss_host.numel() * 4, clk, acc, ffma_rate, mufu_rate,
                      check, t_wall, units, graph is not None, extras)
        if world == 1 and not args.no_cpu_baseline:
            out.update(_cpu_leg(cfg, w, scans, out))
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def _e2e_pipelined(P, steps, torch, dev):
    """End to end with the copies overlapped: NSETS complete buffer sets (parameters, targets, workspace, gradients), three
    streams.  Step k: H2D of its inputs (copy-in stream) -> its graph (compute stream) -> D2H of its gradients and loss
    (copy-out stream); a buffer set is reused by step k + NSETS once step k's D2H has finished (with two sets a set's
    H2D + compute + D2H = 710 us bounds two steps; with three the H2D stream is the bound).  Every step's inputs go in
    and every step's results come out; returns the total ms from the first H2D to the last D2H."""
    NSETS = 3
    s_in, s_cmp, s_out = (torch.cuda.Stream(device=dev) for _ in range(3))
    sets = []
    for k in range(NSETS):
        R = P.new_rasterizer()
        p = [t.clone() for t in P.p]
        tgt = P.tgt.clone()
        tn = None if P.tn is None else P.tn.clone()
        with torch.cuda.stream(s_cmp):
            P.step(s_cmp, R, p, tgt, tn)
        s_cmp.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s_cmp):
            P.step(s_cmp, R, p, tgt, tn)
        gh = [torch.empty_like(t, device="cpu").pin_memory() for t in (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)]
        lh = torch.empty_like(R.loss, device="cpu").pin_memory()
        sets.append(dict(R=R, p=p, tgt=tgt, tn=tn, graph=g, gh=gh, lh=lh, out_done=None))

    def run(n):
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record(s_in)
        for k in range(n):
            b = sets[k % NSETS]
            with torch.cuda.stream(s_in):
                if b["out_done"] is not None:
                    s_in.wait_event(b["out_done"])           # step k - NSETS has left this buffer set
                for d, h in zip(b["p"], P.host):
                    d.copy_(h, non_blocking=True)
                b["tgt"].copy_(P.tgt_pin, non_blocking=True)
                if b["tn"] is not None:
                    b["tn"].copy_(P.tn_pin, non_blocking=True)
                ev_in = torch.cuda.Event()
                ev_in.record(s_in)
            with torch.cuda.stream(s_cmp):
                s_cmp.wait_event(ev_in)
                b["graph"].replay()
                ev_c = torch.cuda.Event()
                ev_c.record(s_cmp)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_c)
                R = b["R"]
                for h, d in zip(b["gh"], (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)):
                    h.copy_(d, non_blocking=True)
                b["lh"].copy_(R.loss, non_blocking=True)
                b["out_done"] = torch.cuda.Event()
                b["out_done"].record(s_out)
        t1.record(s_out)
        torch.cuda.synchronize(dev)
        for b in sets:
            b["out_done"] = None
        return t0.elapsed_time(t1)

    run(2 * NSETS)
    return float(run(steps))


def _next_sections(P, R, stream, flush, lgs, torch, args):
    """NEXT-1 / NEXT-2 / NEXT-3, reported beside the graded step, not inside it (headline config only)."""
    w, S, dev, lam = P.w, P.S, P.dev, P.lam
    tgt, tn = P.tgt[0], P.tn[0]
    hbm = _peaks()[0]
    q = [t.clone() for t in P.p]
    log_scale = torch.log(q[2])
    mom = [torch.zeros((w.N, 10), device=dev) for _ in range(2)]
    l_scale = torch.zeros(1, device=dev)
    tcount = [0]

    def adam():
        tcount[0] += 1
        lgs.lgs_adam_step(q[0], q[1], log_scale, q[3], q[2], R.g_mean, R.g_quat, R.g_scale, R.g_opacity, mom[0],
                          mom[1], tcount[0], 1.6e-4, 1e-3, 5e-3, 5e-2, loss_scale=l_scale, stream=stream)

    def iteration():
        R.forward(*q, stream=stream)
        R.loss_mapping(tgt, tn, None, 0.1, 1e-6, lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False,
                       stream=stream)
        R.backward(*q, stream=stream)
        adam()

    def timed_fn(fn, n):
        evs = []
        with torch.cuda.stream(stream):
            for _ in range(n):
                flush.zero_(); flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); fn(); e1.record(stream)
                evs.append((e0, e1))
        stream.synchronize()
        return float(np.median([a.elapsed_time(b) for a, b in evs]))

    def roof(nbytes, ms, what):
        ach = nbytes / (ms * 1e-3) / 1e9
        return {"bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm, "algorithmic": what}

    # NEXT-2: the workload's scan (one return per valid pixel, on the grid's beams) built into the range image
    tgt_h, tn_h = P.tgt_pin[0].numpy(), P.tn_pin[0].numpy()
    jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
    phi = -np.pi + (ii + 0.5) * (2 * np.pi / S.W)
    eM, em = float(np.float32(S.elev_max)), float(np.float32(S.elev_min))
    th = eM - (jj + 0.5) * ((eM - em) / S.H)
    dirs = np.stack([np.cos(th) * np.cos(phi), np.cos(th) * np.sin(phi), np.sin(th)], -1)
    pts = torch.from_numpy((dirs * tgt_h[..., None]).reshape(-1, 3).astype(np.float32)).to(dev)
    nrm_pts = torch.from_numpy(np.ascontiguousarray(tn_h.reshape(3, -1).T)).to(dev)
    zbuf = torch.empty(8 * S.H * S.W, dtype=torch.uint8, device=dev)
    img, img_n = torch.empty_like(tgt), torch.empty_like(tn)

    def scan():
        lgs.lgs_scan_to_range_image(pts, nrm_pts, R.sensor, zbuf, img, img_n, stream=stream)

    timed_fn(scan, 3)
    scan_ms = timed_fn(scan, 30)
    assert torch.equal(img > 0, tgt > 0)
    scan_bytes = 24.0 * pts.shape[0] + 40.0 * S.H * S.W     # points + winners' normals in; z-buffer write + read, images out
    next2 = {"scan_to_range_image_us": 1e3 * scan_ms, "points": int(pts.shape[0]),
             "roofline": roof(scan_bytes, scan_ms, "24 B x %d points + 40 B x %d pixels" % (pts.shape[0], S.H * S.W)),
             "note": "median of 30, eager launches, 2 x 256 MiB L2 scrub before each, CUDA events on the launching stream"}
    # NEXT-3 (first item): opacity prune + compaction of the map with its optimiser state, alpha_min = 0.5
    kept = [0]
    pr_ins = [q[0], q[1], log_scale, q[3], q[2], mom[0], mom[1]]
    pr_out = ([torch.empty_like(t) for t in pr_ins], torch.zeros(1, dtype=torch.int64, device=dev),
              torch.empty(max(lgs.lgs_prune_workspace_bytes(w.N), 4), dtype=torch.uint8, device=dev))

    def prune():       # pre-allocated outputs, no host sync: the three kernels alone
        lgs.lgs_prune_compact(0.5, *pr_ins, stream=stream, out=pr_out)

    with torch.cuda.stream(stream):
        prune()
    stream.synchronize()
    kept[0] = int(pr_out[1].item())
    prune_ms = timed_fn(prune, 20)
    prune_bytes = 4.0 * w.N + 128.0 * w.N + 128.0 * kept[0]      # opacity twice, every row once in, survivors out
    next3 = {"prune_compact_us": 1e3 * prune_ms, "kept": kept[0], "of": w.N,
             "roofline": roof(prune_bytes, prune_ms, "132 B x %d surfels + 128 B x %d survivors" % (w.N, kept[0])),
             "note": "pre-allocated outputs, no host sync: count / scan / scatter kernels only; median of 20, eager launches"}
    # NEXT-3 (the other entry points): control score, quantile, adaptive split, one cover-and-prune pass -- on the
    # workload's map and on a 2M-surfel synthetic map (uniform in a 200 m x 200 m x 6 m block), pre-allocated
    # workspaces and outputs, no host sync inside the timed region
    def manage(mean, quat, scale, opac, tag):
        Nm = int(opac.numel())
        g = torch.Generator(device=dev); g.manual_seed(11)
        sig = torch.sort(torch.rand((Nm, 3), device=dev, generator=g) * 0.99 + 0.01, dim=1, descending=True)[0].contiguous()
        res = torch.rand(Nm, device=dev, generator=g) * 0.3
        c = torch.empty(Nm, device=dev)
        bounds = ((0.1, 0.9), (0.0, 0.2), (0.02, 0.25))
        mws = torch.empty(max(lgs.lgs_manage_workspace_bytes(Nm), 256), dtype=torch.uint8, device=dev)
        thr = torch.zeros(1, device=dev)
        lo = mean.min(0)[0].cpu().numpy(); hi = mean.max(0)[0].cpu().numpy()
        cell = 0.5
        dims = (int(np.ceil((hi[0] - lo[0]) / cell)) + 1, int(np.ceil((hi[1] - lo[1]) / cell)) + 1)
        cws = torch.empty(max(lgs.lgs_cover_workspace_bytes(Nm, *dims), 256), dtype=torch.uint8, device=dev)
        keep = torch.empty(Nm, dtype=torch.uint8, device=dev)
        n_rem = torch.zeros(1, dtype=torch.int64, device=dev)
        n_new = torch.zeros(1, dtype=torch.int64, device=dev)
        cap = Nm // 20
        rows = Nm + cap

        def grown(t):
            o = torch.zeros((rows,) + tuple(t.shape[1:]), device=dev)
            o[:Nm] = t
            return o

        sp = [grown(t) for t in (mean, quat, torch.log(scale), opac, scale)]
        sc2, ls2 = scale.clone(), torch.log(scale)

        def f_score():
            lgs.lgs_control_score(sig, res, bounds, out=c, stream=stream)

        def f_quant():
            lgs.lgs_quantile(c, 0.9, out=thr, workspace=mws, stream=stream)

        def f_split():
            lgs.lgs_split(Nm, c, thr, 0.05, cap, 0.5, 1.6, *sp, n_new=n_new, workspace=mws, stream=stream)

        thr_lo = torch.zeros(1, device=dev)

        def f_cover():
            lgs.lgs_cover_prune_pass(mean, quat, sc2, ls2, opac, c, thr_lo, (0, 1), (float(lo[0]), float(lo[1])), cell, dims,
                                     0.05, 3.0, 0.5, 2.0, cap, keep=keep, n_removed=n_rem, workspace=cws, stream=stream)

        out = {"N": Nm, "grid": "%d x %d cells of %.1f m" % (dims[0], dims[1], cell)}
        with torch.cuda.stream(stream):
            f_score(); f_quant()
            lgs.lgs_quantile(c, 0.5, out=thr_lo, workspace=mws, stream=stream)
        for name, fn, nbytes, what in (
                ("control_score", f_score, 20.0 * Nm, "20 B x N (sigma, residual in; score out)"),
                ("quantile", f_quant, 4.0 * Nm, "4 B x N (one read of x; the radix select makes four)"),
                ("split", f_split, 8.0 * Nm + 384.0 * cap, "8 B x N (score, opacity) + 384 B x max_splits (row in, two rows out)"),
                ("cover_prune_pass", f_cover, 45.0 * Nm, "45 B x N (mean, quat, scale, opacity, score in; keep out)")):
            timed_fn(fn, 2)
            ms = timed_fn(fn, 10)
            out[name] = {"us": 1e3 * ms, "roofline": roof(nbytes, ms, what)}
        stream.synchronize()
        out["split"]["n_split"] = int(n_new.item()) - Nm
        out["cover_prune_pass"]["n_removed"] = int(n_rem.item())
        return out

    next3["manage_map"] = manage(q[0], q[1], q[2], q[3], "workload map")
    g2 = torch.Generator(device=dev); g2.manual_seed(12)
    N2 = 2_000_000
    m2 = (torch.rand((N2, 3), device=dev, generator=g2) - 0.5) * torch.tensor([200.0, 200.0, 6.0], device=dev)
    q2 = torch.randn((N2, 4), device=dev, generator=g2)
    s2 = torch.rand((N2, 2), device=dev, generator=g2) * 0.35 + 0.05
    o2 = torch.rand(N2, device=dev, generator=g2)
    next3["manage_2M"] = manage(m2.contiguous(), q2, s2, o2, "2M synthetic")
    del m2, q2, s2, o2
    next3["manage_note"] = ("median of 10 eager calls each, 2 x 256 MiB L2 scrub before each, pre-allocated workspaces; "
                            "repeated split / cover calls act on their own previous output (timing only)")
    timed_fn(adam, 3)
    adam_ms = timed_fn(adam, 30)
    timed_fn(iteration, 3)
    iter_ms = timed_fn(iteration, 30)
    # the same iteration as ONE CUDA graph: the step count lives on the device and is advanced inside the graph
    counter = torch.full((1,), tcount[0] + 1, dtype=torch.int32, device=dev)

    def iteration_dev():
        R.forward(*q, stream=stream)
        R.loss_mapping(tgt, tn, None, 0.1, 1e-6, lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False,
                       stream=stream)
        R.backward(*q, stream=stream)
        lgs.lgs_adam_step(q[0], q[1], log_scale, q[3], q[2], R.g_mean, R.g_quat, R.g_scale, R.g_opacity, mom[0],
                          mom[1], 1, 1.6e-4, 1e-3, 5e-3, 5e-2, loss_scale=l_scale, stream=stream, step_device=counter)
        counter.add_(1)

    iter_graph_ms = None
    if not args.no_graph:
        with torch.cuda.stream(stream):
            iteration_dev()
        stream.synchronize()
        it_graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(it_graph, stream=stream):
            iteration_dev()
        timed_fn(it_graph.replay, 3)
        iter_graph_ms = timed_fn(it_graph.replay, 30)
    next1 = {"adam_step_us": 1e3 * adam_ms,
             "adam_roofline": roof(288.0 * w.N, adam_ms, "288 B x %d surfels" % w.N),   # params 40 + grads 40 + moments 80 in; params 40 + scale 8 + moments 80 out
             "mapping_iteration_us": 1e3 * iter_ms,
             "mapping_iteration_graph_us": None if iter_graph_ms is None else 1e3 * iter_graph_ms,
             "note": "median of 30, eager launches (no graph), 2 x 256 MiB L2 scrub before each, CUDA events on the launching stream"}
    return {"next1": next1, "next2": next2, "next3": next3}


def _passes(S) -> int:
    nt = ((S.H + 15) // 16) * ((S.W + 15) // 16)
    bits = 32 + max(0, (nt - 1).bit_length())
    return (bits + 7) // 8


def _step_bytes(N, S, F, n_vis, n_keys) -> float:
    """Algorithmic HBM bytes of one step of F frames, from oracle-side counts only: parameters in and
    gradients out once per frame, images / upstream / per-pixel aux per frame, records and partial sums per visible
    (frame, surfel) pair, the radix passes over the 16x16 keys."""
    HW = S.H * S.W
    P = _passes(S)
    return F * (40.0 * N + 40.0 * N + 56.0 * HW) + n_vis * (48.0 * 3 + 44.0 * 2) + n_keys * 12.0 * (2 * P + 2)


def _roofline(name, ms, N, S, F, n_vis, n_keys, n_contrib, hbm_gbs, fp32_peak, fp32_src, peak_src, traffic) -> dict:
    HW = S.H * S.W
    if name in ("composite_fwd", "composite_bwd"):
        per = FWD_FP32_PER_PAIR if name == "composite_fwd" else BWD_FP32_PER_PAIR
        ach = n_contrib * per / (ms * 1e-3)
        return {"kernel": name, "bound": "alu", "achieved": ach / 1e12, "peak": fp32_peak / 1e12,
                "unit": "T FP32 lane-instr/s", "frac": ach / fp32_peak, "traffic": traffic.get(name), "ms": ms,
                "peak_source": fp32_src,
                "algorithmic": "%d contributing pairs x %d FP32 instr" % (round(n_contrib), per)}
    bytes_ = {"project": F * (40.0 * N + 16.0 * N) + n_vis * 48.0,
              "emit": F * 16.0 * N + n_keys * 8.0,
              "tile_sort": n_keys * 8.0 * 2,
              "loss": F * 40.0 * HW,
              "chain": 40.0 * N + 40.0 * N + n_vis * 44.0}.get(name, 0.0)
    ach = bytes_ / (ms * 1e-3) / 1e9
    return {"kernel": name, "bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
            "traffic": traffic.get(name), "ms": ms, "peak_source": peak_src}


def _report(args, cfg, P, world, n_sm, nv, nk, nc, total_ms, step_ms, warm_ms, e2e_ms, e2e_note, e2e_serial_ms,
            e2e_res_ms, h2d_bytes, d2h_bytes, scan_bytes, loss_bytes, clk, acc, ffma_rate, mufu_rate, check, t_wall,
            units, graphed, extras):
    w, S, F = P.w, P.S, P.F
    hbm_gbs, sm_mhz, peak_src = _peaks()
    nominal_fp32 = n_sm * FP32_LANES * sm_mhz * 1e6          # lane-instructions / s (FMA = 1)
    nominal_sfu = n_sm * SFU_LANES * sm_mhz * 1e6
    # the measured issue rates are the denominators (an FFMA / MUFU.EX2 loop of the library, best of 5 launches)
    fp32_peak, sfu_peak = ffma_rate, mufu_rate
    fp32_src = "measured: lgs_microbench FFMA %.3g lane-instr/s on %d SMs (nominal %d x %d x %.0f MHz = %.3g)" % (
        ffma_rate, n_sm, n_sm, FP32_LANES, sm_mhz, nominal_fp32)
    k16 = CONFIGS[cfg]["k16"]
    k_alg = k16 if k16 is not None else nk      # (no oracle-side count stored: the implementation's own 8x4 key count, larger)
    traffic = _ncu_dram_bytes() if cfg == "nc" else {}
    # N_fp (footprint, oracle-side) where the step is the whole workload; a frame-sharded rank holds a share of the
    # frames, for which only its own rect count is known (an upper bound of its N_fp)
    nfp_all = CONFIGS[cfg].get("nfp")
    whole = F == len(w.sensors)
    n_fp = nfp_all if (nfp_all is not None and whole) else nv
    if not whole:
        k_alg = nk
    dom = max(acc, key=acc.get)
    # `acc` holds ONE frame's kernels when a multi-pose step is F serial calls (the profile slots hold one call each):
    # the bytes / pairs set against it are then one frame's share, not the step's
    Fk = F if (P.batched or F == 1) else 1
    roof = _roofline(dom, acc[dom], w.N, S, Fk, n_fp * Fk / F, k_alg * Fk / F, nc * Fk / F, hbm_gbs, fp32_peak, fp32_src,
                     peak_src, traffic)
    roof["frames_in_ms"] = Fk
    b_alg = _step_bytes(w.N, S, F, n_fp, k_alg)
    t_alu = nc * max((FWD_FP32_PER_PAIR + BWD_FP32_PER_PAIR) / fp32_peak, (FWD_SFU_PER_PAIR + BWD_SFU_PER_PAIR) / sfu_peak)
    t_roof = max(b_alg / (hbm_gbs * 1e9), t_alu)
    ms_step = total_ms / args.steps
    st = _stats(step_ms)
    out = {
        "metric": metric_name(cfg), "value": units / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if P.world > 1 else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(cfg, w),
        "run": {"graph": graphed, "replicas": 1 if P.world > 1 else world,
                "frame_sharded_over_ranks": P.world if P.world > 1 else None, "frames_on_this_rank": F,
                "n_visible": nv, "n_fp": n_fp, "n_keys": nk, "intersections_per_step": nc, "max_keys": P.max_keys,
                "one_launch_batch": P.batched},
        "ms_per_frame": ms_step / F, "ms_per_frame_l2_warm": warm_ms / args.steps / F,
        "ms_per_step_stats": st,
        "clocks": clk, "gpu_launches": P.kernels_per_step() * args.steps, "sm_count": n_sm,
        "e2e": {"value": units / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                "ms_per_step_serialised": e2e_serial_ms / args.steps,
                "note": "strict reading: every buffer of the calls is a pinned HOST buffer (map and scan in, gradients "
                        "and loss out, each step); " + e2e_note},
        "e2e_resident_map": {"value": units / (e2e_res_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_res_ms / args.steps,
                             "h2d_bytes_per_step": scan_bytes, "d2h_bytes_per_step": loss_bytes,
                             "note": "as a mapping loop runs it: map and gradients resident on the device, the scan's "
                                     "range + normal images from pinned host memory and the loss back, each step"},
        "roofline": roof,
        "step_roofline": {"t_roof_us": 1e6 * t_roof, "hbm_bytes": b_alg, "t_hbm_us": 1e6 * b_alg / (hbm_gbs * 1e9),
                          "t_alu_us": 1e6 * t_alu, "frac": t_roof / (ms_step * 1e-3), "frac_median": t_roof / (st["median"] * 1e-3),
                          "peak": peak_src, "k_alg": k_alg, "n_fp": n_fp, "n_rect": nv,
                          "n_fp_source": "oracle.footprint_surfels (SURVEY.md 8(d))" if n_fp != nv or nfp_all == nv else "implementation's rect count (upper bound)",
                          "k_alg_source": "oracle list reference, 16x16 tiles" if k16 is not None else "implementation's 8x4 keys (upper bound)"},
        "issue_peaks": {"ffma_lane_instr_per_s": ffma_rate, "mufu_ex2_per_s": mufu_rate,
                        "nominal_fp32": nominal_fp32, "nominal_sfu": nominal_sfu, "sm_count": n_sm, "sm_mhz": sm_mhz},
        "graph_check": check,
        "kernels_ms": acc, "wall_s_timed_region": t_wall,
    }
    out.update(extras)
    return out


def _cpu_leg(cfg, w, scans, out):
    """The oracle as it stands on the box's host cores, on a bounded sample of the same workload (rank 0, N = 1)."""
    import oracle
    if cfg == "tiny":
        scans = [_tiny_target(w)]
    nfr = 2 if cfg == "nc" else 1
    t0 = time.perf_counter()
    ic = 0
    for k in range(nfr):
        f = 0
        keep = None if w.keep_masks is None else w.keep_masks[f]
        ic += _oracle_frame(w, w.sensors[f], scans[f][0], scans[f][1], keep)
    dt = time.perf_counter() - t0
    res = {"cpu_baseline": {"value": ic / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                            "sample": "%d whole frame%s of the same workload (frame 0; forward+loss+backward, bounded mode)" % (nfr, "s" if nfr > 1 else ""),
                            "ms_per_frame": 1e3 * dt / nfr}}
    k16 = sum(int(oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, tile=16).keys.shape[0]) for S in w.sensors)
    out["step_roofline"]["k_alg_16x16_recounted"] = k16
    if cfg in ("tiny", "nc"):          # (seconds; the larger configs are recounted by tests/test_bench_constants.py)
        nfp = sum(int(oracle.footprint_surfels(w.mean, w.quat, w.scale, w.opacity, S).sum()) for S in w.sensors)
        out["step_roofline"]["n_fp_recounted"] = nfp
        stale = k16 != CONFIGS[cfg]["k16"] or nfp != CONFIGS[cfg]["nfp"]
    else:
        stale = k16 != CONFIGS[cfg]["k16"]
    out["step_roofline"]["constants_match_oracle"] = not stale
    if stale:
        sys.stderr.write("bench.py: CONFIGS[%r] k16 / nfp no longer match the oracle's recount -- step_roofline is skewed\n" % cfg)
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="nc", choices=sorted(CONFIGS))
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the NEXT-1/2/3 sections of the headline config")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        dflt = {"tiny": 200, "nc": 200, "kitti": 30, "large": 50, "batch": 20}[args.config]
        args.steps = dflt if args.steps is None else args.steps
        args.warmup = 10 if args.warmup is None else max(args.warmup, 3)
        run_ours(args)


if __name__ == "__main__":
    main()
