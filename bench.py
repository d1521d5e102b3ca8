#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (S1-S8: project/cull, tile ranges, key emission,
per-tile radix sort, forward composite, loss stage, backward composite, per-surfel chain)
over one synthetic frame of BASELINE.json configs[1] (64x1024, 300k surfels).

    python bench.py --gpus N --steps K --warmup W            (ours; torchrun for N > 1)
    python bench.py --impl reference --steps K --warmup W    (the CPU oracle, as it stands)

Prints ONE JSON line (rank 0).  metric = Gaussian-pixel intersections/s for forward+backward
(intersection = contributing (pixel, surfel) pair, counted on the device and equal to the
oracle's count); ms_per_step = fwd+loss+bwd ms/frame.  Timing: CUDA events around each
graph-replayed step on the launching stream, a 256 MiB L2 scrub before every timed step,
max over ranks.  See DESIGN.md "Measurement".
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

METRIC = "fwd+bwd Gaussian-pixel intersections/s (64x1024, 300k surfels)"
UNIT = "intersections/s"

# Algorithmic work per contributing pair, counted once from the oracle's expression tree
# (oracle/lgs_oracle.cpp composite_pixel / lgs_oracle_backward) and frozen -- DESIGN.md "Roofline".
FWD_FP32_PER_PAIR, FWD_SFU_PER_PAIR = 31, 2
BWD_FP32_PER_PAIR, BWD_SFU_PER_PAIR = 89, 3
N_SM, FP32_LANES, SFU_LANES = 148, 128, 16
# Algorithmic key count of SURVEY.md 8(d): (surfel, 16x16 tile) pairs of the oracle's list reference on this
# workload (oracle.tile_lists(..., tile=16), seed fixed) -- NOT the implementation's own
# key count, which is larger because it lists per 8x4 tile.  Re-counted by the cpu_baseline leg when it runs.
K_ALG_16X16 = 367_601
# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the ncu --set full capture summarised in
# profiles/r1e_launches.md (one launch of every kernel of a step, L2 flushed by ncu before each).
NCU_DRAM_BYTES = {"project": 12.8e6 + 3.5e6, "emit": 0.3e6 + 10.2e6, "tile_sort": 2.1e6 + 3.1e6, "composite_fwd": 28.8e6 + 125e3,
                  "loss": 1.0e6 + 2.3e6, "composite_bwd": 44.8e6 + 119e3, "chain": 30.3e6 + 6e3}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            j = json.load(f)
        return float(j["hbm_gbs"]), float(j.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


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


def _workload():
    from workloads import make_newer_college, simulate_scan
    w = make_newer_college()
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    return w, S, tgt, tn


def _oracle_step(w, S, tgt, tn):
    """One frame through the oracle as it stands: forward + loss + backward. Returns I_c."""
    import oracle
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED)
    lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, None, **w.lambdas)
    oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, lr.gD, lr.gA, lr.gN, oracle.BOUNDED)
    return fo.stats["I_c"]


def run_reference(args):
    """--impl reference: the fp64 CPU oracle on the box's host cores, same config / metric."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w, S, tgt, tn = _workload()
    for _ in range(max(args.warmup, 0) and 1):
        _oracle_step(w, S, tgt, tn)
    t0 = time.perf_counter()
    ic = 0
    for _ in range(args.steps):
        ic += _oracle_step(w, S, tgt, tn)
    dt = time.perf_counter() - t0
    val = ic / dt
    cores = oracle.num_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "newer_college_shaped 64x1024, 300000 surfels, 1 frame per step"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d whole frames (forward+loss+backward, bounded mode, OpenMP)" % args.steps},
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


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_04127_b200 as lgs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: replicas only: every rank renders the same synthetic frame
    w, S, tgt_h, tn_h = _workload()
    host = [torch.from_numpy(x).pin_memory() for x in (w.mean, w.quat, w.scale, w.opacity)]
    tgt_pin, tn_pin = torch.from_numpy(tgt_h).pin_memory(), torch.from_numpy(tn_h).pin_memory()
    p = [h.to(dev) for h in host]
    tgt, tn = tgt_pin.to(dev), tn_pin.to(dev)
    lam = w.lambdas

    # ---- size the key buffer once from a probe frame (the only host sync before the timed region)
    probe = lgs.Rasterizer(w.N, S, 8 * w.N, device=dev)
    probe.forward(*p)
    nv, nk, nc, ovf = probe.query()
    assert not ovf
    del probe
    R = lgs.Rasterizer(w.N, S, int(1.25 * nk) + 1024, device=dev)
    stream = torch.cuda.Stream(device=dev)

    def step():
        R.forward(*p, stream=stream)
        R.loss_stage(tgt, tn, None, lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False, stream=stream)
        R.backward(*p, stream=stream)

    kernels_per_step = 6 + 2 + 3   # project, ranges, placement, tile sort x2 (length classes), composite | loss x2 | clear, backward composite, chain
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # L2 scrub (> 126 MB L2)

    with torch.cuda.stream(stream):
        step()
    stream.synchronize()
    graph = None
    if not args.no_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            step()

    def run_step():
        if graph is not None:
            graph.replay()
        else:
            step()

    def timed(n, scrub=True, pre=None, post=None):
        """Sum of per-step device times (ms); the scrub runs outside the event pair."""
        evs = []
        with torch.cuda.stream(stream):
            for _ in range(n):
                if scrub:
                    flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if pre:
                    pre()
                run_step()
                if post:
                    post()
                e1.record(stream)
                evs.append((e0, e1))
        stream.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            flush.zero_()
            run_step()
    clocks = ClockSampler(local_rank)
    clocks.start()
    clocks.wait_first()
    barrier()
    t_wall0 = time.perf_counter()
    total_ms = timed(args.steps, scrub=True)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    # The timed region of a short run (100 steps = 30 ms) is shorter than nvidia-smi's sampling period: the same
    # loop is continued, untimed, until the load has lasted >= 0.75 s, and the clocks are the samples of that window.
    while time.perf_counter() - t_wall0 < 0.75:
        timed(min(args.steps, 100), scrub=True)
    clk = clocks.stop(t_wall0, time.perf_counter())
    clk["window"] = "timed region + identical untimed continuation, %.2f s" % (time.perf_counter() - t_wall0)
    warm_ms = timed(args.steps, scrub=False)

    # ---- end to end through the public API with HOST buffers: H2D of the map + scan, step, D2H of grads + loss
    g_host = [torch.empty_like(t, device="cpu").pin_memory() for t in (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)]
    loss_host = torch.empty(4, dtype=torch.float32).pin_memory()

    def h2d():
        for d, h in zip(p, host):
            d.copy_(h, non_blocking=True)
        tgt.copy_(tgt_pin, non_blocking=True)
        tn.copy_(tn_pin, non_blocking=True)

    def d2h():
        for h, d in zip(g_host, (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)):
            h.copy_(d, non_blocking=True)
        loss_host.copy_(R.loss, non_blocking=True)

    timed(2, True, h2d, d2h)
    e2e_ms = timed(args.steps, True, h2d, d2h)

    # the same, as a mapping loop runs it: the map and its gradients stay on the device (the optimiser step reads them
    # there, lgs_adam_step); per step only the scan's images come from the host and the loss goes back
    def h2d_scan():
        tgt.copy_(tgt_pin, non_blocking=True)
        tn.copy_(tn_pin, non_blocking=True)

    def d2h_loss():
        loss_host.copy_(R.loss, non_blocking=True)

    timed(2, True, h2d_scan, d2h_loss)
    e2e_res_ms = timed(args.steps, True, h2d_scan, d2h_loss)
    h2d_bytes = sum(h.numel() * 4 for h in host) + tgt_pin.numel() * 4 + tn_pin.numel() * 4
    d2h_bytes = sum(h.numel() * 4 for h in g_host) + 16

    # ---- per-kernel times, live, with CUDA events on the launching stream (not graph-replayed)
    lgs.lgs_profile_enable(True)
    acc = {}
    nprof = max(3, min(args.steps, 20))
    with torch.cuda.stream(stream):
        for _ in range(nprof):
            # three scrubs (~200 us of GPU work): the whole step is enqueued before the GPU reaches it, so
            # the event pairs bracket kernels running back to back, not the host's launch latency
            flush.zero_(); flush.zero_(); flush.zero_()
            step()
            for k, v in lgs.lgs_profile_read(stream).items():
                acc[k] = acc.get(k, 0.0) + v / nprof
    lgs.lgs_profile_enable(False)
    nv, nk, nc, ovf = R.query(stream)

    # ---- NEXT-1, reported beside the graded step, not inside it: the optimiser step alone and one
    # whole mapping iteration forward -> lgs_loss_mapping (Eq. 13 image side) -> backward -> lgs_adam_step
    next1 = next2 = next3 = None
    if rank == 0:
        q = [t.clone() for t in p]
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

        # NEXT-2: the workload's scan (one return per valid pixel, on the grid's beams) built into the range image
        jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
        phi = -np.pi + (ii + 0.5) * (2 * np.pi / S.W)
        th = float(np.float32(S.elev_max)) - (jj + 0.5) * ((float(np.float32(S.elev_max)) - float(np.float32(S.elev_min))) / S.H)
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
                 "roofline": {"bound": "hbm", "achieved": scan_bytes / (scan_ms * 1e-3) / 1e9, "peak": _peaks()[0], "unit": "GB/s",
                              "frac": scan_bytes / (scan_ms * 1e-3) / 1e9 / _peaks()[0],
                              "algorithmic": "24 B x %d points + 40 B x %d pixels" % (pts.shape[0], S.H * S.W)},
                 "note": "three launch-latency-bound kernels on 4 MB of data; same timing protocol as next1"}
        # NEXT-3 (first item): opacity prune + compaction of the map with its optimiser state, alpha_min = 0.5
        kept = [0]

        def prune():
            kept[0] = lgs.lgs_prune_compact(0.5, q[0], q[1], log_scale, q[3], q[2], mom[0], mom[1], stream=stream)[0]

        with torch.cuda.stream(stream):
            prune()
        stream.synchronize()
        prune_ms = timed_fn(prune, 20)
        prune_bytes = 4.0 * w.N + 128.0 * w.N + 128.0 * kept[0]      # opacity twice, every row once in, survivors out
        next3 = {"prune_compact_us": 1e3 * prune_ms, "kept": kept[0], "of": w.N,
                 "roofline": {"bound": "hbm", "achieved": prune_bytes / (prune_ms * 1e-3) / 1e9, "peak": _peaks()[0], "unit": "GB/s",
                              "frac": prune_bytes / (prune_ms * 1e-3) / 1e9 / _peaks()[0],
                              "algorithmic": "132 B x %d surfels + 128 B x %d survivors" % (w.N, kept[0])},
                 "note": "binding call: allocates its outputs and reads n_out back (one host sync) inside the timed region"}
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
        adam_bytes = 288.0 * w.N      # params 40 + grads 40 + moments 80 in; params 40 + scale 8 + moments 80 out
        hbm_gbs0 = _peaks()[0]
        next1 = {"adam_step_us": 1e3 * adam_ms, "adam_roofline": {"bound": "hbm", "achieved": adam_bytes / (adam_ms * 1e-3) / 1e9,
                                                                "peak": hbm_gbs0, "unit": "GB/s",
                                                                "frac": adam_bytes / (adam_ms * 1e-3) / 1e9 / hbm_gbs0,
                                                                "algorithmic": "288 B x %d surfels" % w.N},
                 "mapping_iteration_us": 1e3 * iter_ms,
                 "mapping_iteration_graph_us": None if iter_graph_ms is None else 1e3 * iter_graph_ms,
                 "note": "median of 30, eager launches (no graph), 2 x 256 MiB L2 scrub before each, CUDA events on the launching stream"}

    # ---- max over ranks, whole-job throughput
    (total_ms, warm_ms, e2e_ms, e2e_res_ms), units = aggregate_over_ranks([total_ms, warm_ms, e2e_ms, e2e_res_ms],
                                                                          float(nc) * args.steps, world, dev)

    if rank == 0:
        hbm_gbs, sm_mhz, peak_src = _peaks()
        fp32_peak = N_SM * FP32_LANES * sm_mhz * 1e6      # lane-instructions / s (FMA = 1)
        sfu_peak = N_SM * SFU_LANES * sm_mhz * 1e6
        dom = max(acc, key=acc.get)
        dom_ms = acc[dom]
        roof = _roofline(dom, dom_ms, w.N, S, nv, K_ALG_16X16, nc, hbm_gbs, fp32_peak, peak_src)
        b_alg = _step_bytes(w.N, S, nv, K_ALG_16X16)
        t_alu = nc * max((FWD_FP32_PER_PAIR + BWD_FP32_PER_PAIR) / fp32_peak, (FWD_SFU_PER_PAIR + BWD_SFU_PER_PAIR) / sfu_peak)
        t_roof = max(b_alg / (hbm_gbs * 1e9), t_alu)
        ms_step = total_ms / args.steps
        out = {
            "metric": METRIC, "value": units / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "newer_college_shaped 64x1024, 300000 surfels, 1 frame per step (fwd+loss+bwd)",
                       "l2": "256 MiB scrub before every timed step", "graph": graph is not None,
                       "replicas": world, "n_visible": nv, "n_keys": nk, "intersections_per_frame": nc,
                       "max_keys": R.max_keys},
            "ms_per_frame": ms_step, "ms_per_frame_l2_warm": warm_ms / args.steps,
            "clocks": clk, "gpu_launches": kernels_per_step * args.steps,
            "e2e": {"value": units / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                    "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                    "note": "strict reading: every buffer of the calls is a pinned HOST buffer (map and scan in, gradients "
                            "and loss out, each step)"},
            "e2e_resident_map": {"value": units / (e2e_res_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_res_ms / args.steps,
                                 "h2d_bytes_per_step": tgt_pin.numel() * 4 + tn_pin.numel() * 4, "d2h_bytes_per_step": 16,
                                 "note": "as a mapping loop runs it: map and gradients resident on the device, the scan's "
                                         "range + normal images from pinned host memory and the loss back, each step"},
            "roofline": roof,
            "step_roofline": {"t_roof_us": 1e6 * t_roof, "hbm_bytes": b_alg, "t_hbm_us": 1e6 * b_alg / (hbm_gbs * 1e9),
                              "t_alu_us": 1e6 * t_alu, "frac": t_roof / (ms_step * 1e-3), "peak": peak_src},
            "kernels_ms": acc, "wall_s_timed_region": t_wall, "next1": next1, "next2": next2, "next3": next3,
        }
        if world == 1 and not args.no_cpu_baseline:
            import oracle
            t0 = time.perf_counter()
            ic = _oracle_step(w, S, tgt_h, tn_h)
            ic += _oracle_step(w, S, tgt_h, tn_h)
            dt = time.perf_counter() - t0
            k16 = int(oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, tile=16).keys.shape[0])
            out["step_roofline"]["k_alg_16x16_recounted"] = k16
            out["cpu_baseline"] = {"value": ic / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                                   "sample": "2 whole frames of the same workload (forward+loss+backward, bounded mode)",
                                   "ms_per_frame": 1e3 * dt / 2}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def _passes(S) -> int:
    nt = ((S.H + 15) // 16) * ((S.W + 15) // 16)
    bits = 32 + max(0, (nt - 1).bit_length())
    return (bits + 7) // 8


def _step_bytes(N, S, n_vis, n_keys) -> float:
    """Algorithmic HBM bytes of one step, from oracle-side counts only."""
    HW = S.H * S.W
    P = _passes(S)
    return 40.0 * N + 40.0 * N + 20.0 * HW + 20.0 * HW + 16.0 * HW + n_vis * 48.0 * 3 + n_vis * 44.0 * 2 + n_keys * 12.0 * (2 * P + 2)


def _roofline(name, ms, N, S, n_vis, n_keys, n_contrib, hbm_gbs, fp32_peak, peak_src) -> dict:
    HW = S.H * S.W
    if name in ("composite_fwd", "composite_bwd"):
        per = FWD_FP32_PER_PAIR if name == "composite_fwd" else BWD_FP32_PER_PAIR
        ach = n_contrib * per / (ms * 1e-3)
        return {"kernel": name, "bound": "alu", "achieved": ach / 1e12, "peak": fp32_peak / 1e12,
                "unit": "T FP32 lane-instr/s", "frac": ach / fp32_peak, "traffic": NCU_DRAM_BYTES.get(name), "ms": ms,
                "peak_source": "148 SMs x 128 FP32 lanes x sm_max_mhz (DESIGN.md)",
                "algorithmic": "%d contributing pairs x %d FP32 instr" % (n_contrib, per)}
    P = _passes(S)
    bytes_ = {"project": 40.0 * N + 16.0 * N + n_vis * 48.0,
              "emit": 16.0 * N + n_keys * 8.0,
              "tile_sort": n_keys * 8.0 * 2,
              "loss": 40.0 * HW,
              "chain": 40.0 * N + 40.0 * N + n_vis * 44.0}.get(name, 0.0)
    ach = bytes_ / (ms * 1e-3) / 1e9
    return {"kernel": name, "bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
            "traffic": NCU_DRAM_BYTES.get(name), "ms": ms, "peak_source": peak_src}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 100 if args.steps is None else args.steps
        args.warmup = 10 if args.warmup is None else max(args.warmup, 3)
        run_ours(args)


if __name__ == "__main__":
    main()
