#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: rays/s (and fps) of the 2048x1024
equirect render of config 3 (multi-room floor, ~1k subfields); MLP samples/s and roofline fraction.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]
                  [--precision auto|fp32|bf16]

A step = one whole pass of the hot path (ray generation, occupancy walk, binning, grouped tiny
MLP, compositing) over one frame of synthetic input (scenegen, seeded).
N > 1 (torchrun): every rank renders a whole frame of its own pose of the replicated scene -- rays
are independent, no data-path collective; value = total rays of all ranks / max-over-ranks time.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the workload.
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

FLOP_PER_SAMPLE = {(32, 2): 12160, (32, 3): 14208, (64, 3): 44800}   # algorithmic, unpadded, no biases
# FP32 ALU peak (bound "alu"): 148 SMs x 128 FMA lanes x 2 FLOP x 1.965 GHz (B200_PROFILING.md clocks)
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def flop_per_sample(width, n_hidden, pe_p=63, pe_d=27):
    macs = pe_p * width + (n_hidden - 1) * width * width + width + width * width + (width + pe_d) * width + 3 * width
    return 2 * macs


def executed_flop_per_sample(width, n_hidden, pe_p=63, pe_d=27):
    """Unpadded contraction the tensor kernel actually runs: the feature layer (no activation) is folded
    into the colour layer on the host, so its width x width product is not evaluated per sample."""
    return flop_per_sample(width, n_hidden, pe_p, pe_d) - 2 * width * width


def ncu_traffic(kernel):
    """DRAM bytes (read + write) of one launch of `kernel` on this workload, from the committed ncu --set full
    capture (profiles/traffic.json, written by hand from the capture named there); None if not recorded."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(kernel)
    except (OSError, ValueError):
        return None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.idx)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(sc, row_stride):
    """Time the oracle, as it stands, on every row_stride-th row of pose 0.  Returns rays/s etc."""
    from oracle import load_oracle
    o = load_oracle()
    s = o.scene_from(sc)
    rows = list(range(0, sc.H, row_stride))
    t0 = time.perf_counter()
    n_samples = 0
    for r in rows:
        out = s.render_rows(sc.poses[0], sc.W, sc.H, r, r + 1, full=False)
        n_samples += int(out["n_emitted"].sum())
    dt = time.perf_counter() - t0
    rays = len(rows) * sc.W
    return dict(rays=rays, seconds=dt, rays_per_s=rays / dt, samples=n_samples, cores=o.num_threads(),
                sample=f"pose 0, every {row_stride}th image row ({len(rows)} rows x {sc.W} px = {rays} rays, "
                       f"{n_samples} MLP samples), wall clock")


def run_reference(args):
    """--impl reference: the oracle on this box's host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from scenegen import make_scene
    sc = make_scene(args.config)
    # each step is a bounded sample (every stride-th row); the stride grows with the number of steps so that the
    # whole --steps K --warmup W run stays within a few minutes on 8 host cores (8 steps of every 8th row ~ 100 s)
    stride = args.ref_row_stride * max(1, -(-(args.warmup + args.steps) // 8))
    vals = []
    for it in range(args.warmup + args.steps):
        r = oracle_sample(sc, stride)
        if it >= args.warmup:
            vals.append(r)
    rays_s = sum(v["rays"] for v in vals) / sum(v["seconds"] for v in vals)
    ms = 1e3 * sum(v["seconds"] for v in vals) / len(vals)
    line = {"impl": "reference", "metric": "rays_per_second_equirect_render", "value": rays_s, "unit": "rays/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(sc, args, "oracle (geometry f32, field+compositing f64)"),
            "cpu_baseline": {"value": rays_s, "unit": "rays/s", "cores": vals[0]["cores"], "kind": "oracle",
                             "sample": vals[0]["sample"]},
            "e2e": {"value": rays_s, "unit": "rays/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(sc, args, precision):
    return {"workload": f"BASELINE.json configs[{args.config - 1}] '{sc.name}': {sc.W}x{sc.H} equirect, "
                        f"grid {sc.dims[0]}x{sc.dims[1]}x{sc.dims[2]}, {sc.n_subfields} subfields, "
                        f"MLP {sc.n_hidden}x{sc.hidden_width}, K={sc.samples_per_voxel}",
            "image": [sc.W, sc.H], "poses_per_step": 1, "n_subfields": sc.n_subfields,
            "precision": precision, "seed": args.config - 1,
            "l2": "explicit L2 flush (512 MiB memset) between timed iterations, outside the CUDA events"}


def time_config(r360, config, precision, steps=5, warmup=3, pinhole=None):
    """Short device-timed run of another BASELINE.json config (all its poses in one batch call).
    pinhole = (W, H, f): the same scene through the roaming (perspective) view instead of the panorama."""
    import torch
    from scenegen import make_scene
    sc = make_scene(config)
    scene = r360.scene_from(sc)
    scene.set_precision(precision)
    scene.use_current_torch_stream()
    B, W, H = len(sc.poses), sc.W, sc.H
    if pinhole:
        W, H, f = pinhole
        scene.set_camera("pinhole", f, f, W / 2.0, H / 2.0)
    poses = np.ascontiguousarray(np.stack([np.asarray(p, np.float32) for p in sc.poses]))
    rgb = torch.empty((B, H, W, 3), dtype=torch.float32, device="cuda")
    depth = torch.empty((B, H, W), dtype=torch.float32, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(warmup):
        scene.render_batch(poses, W, H, rgb, depth)
    torch.cuda.synchronize()
    ms, ms_mlp = 0.0, 0.0
    for _ in range(steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        scene.render_batch(poses, W, H, rgb, depth)
        e1.record()
        st = scene.stats()
        ms += e0.elapsed_time(e1)
        ms_mlp += st.ms_mlp
    ms /= steps
    ms_mlp /= steps
    fl = flop_per_sample(sc.hidden_width, sc.n_hidden)
    peaks = measured_peaks()
    out = {"config": config, "name": sc.name + (" (pinhole view)" if pinhole else ""), "image": [W, H], "poses": B, "n_subfields": sc.n_subfields,
           "mlp": [sc.n_hidden, sc.hidden_width], "K": sc.samples_per_voxel, "precision": precision,
           "ms_per_step": ms, "rays_per_s": B * W * H / (ms * 1e-3), "fps": B * 1e3 / ms,
           "samples_per_step": int(st.samples_emitted), "mlp_samples_per_s": st.samples_emitted / (ms_mlp * 1e-3),
           "ms_mlp": ms_mlp, "chunks": int(st.chunks)}
    if precision == "bf16":
        out["mlp_frac_of_bf16_sustained"] = st.samples_emitted * fl / (ms_mlp * 1e-3) / 1e12 / peaks["bf16_sustained"]
        # the sustained figure is cuBLAS under its own power throttle; a kernel that holds the full clock can pass it
        out["mlp_frac_of_bf16_burst"] = st.samples_emitted * fl / (ms_mlp * 1e-3) / 1e12 / peaks["bf16"]
    scene.close()
    del rgb, depth, flush
    torch.cuda.empty_cache()
    return out


def time_extras(r360, config):
    """Wall-clock of the stand-alone entry points (host arrays in, host arrays out) on a BASELINE.json scene."""
    import torch
    from scenegen import make_scene
    sc = make_scene(config, with_weights=False)
    out = {}

    def wall(fn, reps):
        fn()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            r = fn()
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) / reps, r

    dt, lab = wall(lambda: r360.assign_subfields(sc.occupancy, sc.dims, sc.box_min, sc.box_max, sc.occ_threshold,
                                                 sc.n_subfields), 2)
    out["assign_subfields"] = {"seconds": dt, "occupied_voxels": int((lab >= 0).sum()), "n": sc.n_subfields,
                               "what": "Algorithm 1 stage II (PAPER.md:147-154), r360_assign_subfields"}
    pose = np.asarray(sc.poses[0], np.float64).reshape(3, 4)
    vs = (np.array(sc.box_max) - np.array(sc.box_min)) / np.array(sc.dims)
    cell = np.floor((pose[:, 3] - np.array(sc.box_min)) / vs).astype(int)
    dt, plan = wall(lambda: r360.floorplan(sc.occupancy, sc.dims, sc.occ_threshold, (int(cell[0]), int(cell[1]))), 5)
    out["floorplan"] = {"seconds": dt, "cells": int(plan.size), "interior_cells": int((plan & 1).sum()),
                        "what": "floorplan estimation (PAPER.md:176-178), r360_floorplan"}
    W, H = 1024, 512
    depth = np.full((H, W), 2.5, np.float32)
    L0 = np.zeros(int(np.prod(sc.dims)), np.float32)
    dt, L = wall(lambda: r360.occupancy_fuse(L0, sc.dims, sc.box_min, sc.box_max, sc.poses[0], W, H, depth), 5)
    out["occupancy_fuse"] = {"seconds": dt, "image": [W, H], "voxels": int(L0.size), "voxels_updated": int((L != 0).sum()),
                             "what": "one observation of Eq. 6 (PAPER.md:117-128), r360_occupancy_fuse, synthetic depth"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--precision", default="auto", choices=["auto", "fp32", "bf16"])
    ap.add_argument("--ref-row-stride", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--all-configs", action="store_true",
                    help="also time BASELINE.json's other configs (short runs) and add them as other_configs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    use_dist = world > 1 or "TORCHELASTIC_RUN_ID" in os.environ      # under torchrun: always go through NCCL
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import __graft_entry__ as g
    import paper_2208_02705_b200 as r360
    if not os.path.exists(r360.lib_path()):
        g.build()
    from scenegen import make_scene
    sc = make_scene(args.config)
    scene = r360.scene_from(sc)
    precision = args.precision
    if precision == "auto":
        try:
            scene.set_precision("bf16")
            precision = "bf16"
        except r360.R360Error:
            precision = "fp32"
    scene.set_precision(precision)
    scene.use_current_torch_stream()
    # each rank renders its own pose: rank r yaws pose 0 by r * 2pi/world about the world up axis
    from paper_2208_02705_b200.shard import rank_pose
    pose = rank_pose(sc.poses[0], rank, world)
    W, H = sc.W, sc.H
    rgb = torch.empty((1, H, W, 3), dtype=torch.float32, device="cuda")
    depth = torch.empty((1, H, W), dtype=torch.float32, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        scene.render(pose, W, H, rgb, depth)
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stage = {k: 0.0 for k in ("ms_count", "ms_scan", "ms_emit", "ms_mlp", "ms_composite")}
    launches = 0
    barrier()
    for k in range(args.steps):
        flush.zero_()
        ev[k][0].record()
        scene.render(pose, W, H, rgb, depth)
        ev[k][1].record()
        st = scene.stats()                      # synchronises; per-stage CUDA events on the launch stream
        for key in stage:
            stage[key] += getattr(st, key)
        launches += st.kernel_launches
    barrier()
    clk = clocks.stop()
    ms_total = sum(a.elapsed_time(b) for a, b in ev)
    tt = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if use_dist:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ms_step = float(tt.item()) / args.steps
    rays_step = W * H * world
    value = rays_step / (ms_step * 1e-3)

    # end to end through the host-buffer entry point (pinned host buffers, H2D pose + D2H image per step)
    h_rgb = torch.empty((1, H, W, 3), dtype=torch.float32).pin_memory()
    h_depth = torch.empty((1, H, W), dtype=torch.float32).pin_memory()
    h_pose = torch.from_numpy(pose.copy()).pin_memory()
    for _ in range(2):
        scene.render_batch_host(h_pose.numpy(), W, H, h_rgb.numpy(), h_depth.numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        scene.render_batch_host(h_pose.numpy(), W, H, h_rgb.numpy(), h_depth.numpy())
    torch.cuda.synchronize()
    te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if use_dist:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = rays_step * args.steps / float(te.item())

    if rank == 0:
        peaks = measured_peaks()
        samples = st.samples_emitted
        ms_mlp = stage["ms_mlp"] / args.steps
        fl = flop_per_sample(sc.hidden_width, sc.n_hidden)
        ach = samples * fl / (ms_mlp * 1e-3) / 1e12
        if precision == "bf16":
            roof = {"bound": "tensor", "kernel": "k_mlp_tc", "achieved": ach, "peak": peaks["bf16_sustained"],
                    "unit": "TFLOP/s", "frac": ach / peaks["bf16_sustained"], "traffic": None,
                    "peak_source": peaks["source"] + " bf16 sustained (kernel timed inside a long step)"}
        else:
            roof = {"bound": "alu", "kernel": "k_mlp_fp32", "achieved": ach, "peak": ALU_PEAK_TFLOPS,
                    "unit": "TFLOP/s", "frac": ach / ALU_PEAK_TFLOPS, "traffic": None,
                    "peak_source": "derived: 148 SM x 128 FMA/clk x 2 x 1.965 GHz"}
        roof["flop_per_sample"] = fl
        if precision == "bf16" and args.config == 3:
            roof["traffic"] = ncu_traffic("k_mlp_tc")
        if precision == "bf16":
            # MEASURED_PEAKS.json's sustained figure is a power-throttled cuBLAS run (its clocks_under_load block);
            # the fraction of the burst figure is reported beside it
            roof["peak_burst"] = peaks["bf16"]
            roof["frac_of_burst"] = ach / peaks["bf16"]
            roof["executed_flop_per_sample"] = executed_flop_per_sample(sc.hidden_width, sc.n_hidden)
        roof["samples_per_launch"] = int(samples)
        roof["ms_per_launch"] = ms_mlp
        # the memory-side stages against the measured HBM copy bandwidth: algorithmic bytes
        rays, segs, Kk = W * H, int(st.segments), sc.samples_per_voxel
        tensor = precision == "bf16"
        stage_bytes = {
            "k_count": rays * 8 + segs * 10 + (rays * 64 if tensor else 0),
            "k_emit": rays * 8 + segs * 10 + segs * (40 if tensor else 24),
            "k_composite": segs * Kk * (8 if tensor else 16) + segs * 8 + rays * 24,   # tensor path: binary16 x4 per sample
        }
        stage_key = {"k_count": "ms_count", "k_emit": "ms_emit", "k_composite": "ms_composite"}
        hbm_stages = {}
        for kname, nbytes in stage_bytes.items():
            ms_k = stage[stage_key[kname]] / args.steps
            gbs = nbytes / (ms_k * 1e-3) / 1e9 if ms_k > 0 else 0.0
            hbm_stages[kname] = {"algorithmic_bytes": int(nbytes), "ms": ms_k, "achieved_gbs": gbs,
                                 "frac_of_hbm_peak": gbs / peaks["hbm"],
                                 # the committed ncu captures are of config 3 on the tensor path only
                                 "traffic": ncu_traffic(kname) if tensor and args.config == 3 else None}
        line = {"metric": "rays_per_second_equirect_render", "value": value, "unit": "rays/s", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "bf16" if precision == "bf16" else "f32",
                "data": "synthetic", "config": workload_config(sc, args, precision),
                "fps": 1e3 / ms_step * world, "mlp_samples_per_s": samples / (ms_mlp * 1e-3),
                "samples_per_frame": int(samples), "segments_per_frame": int(st.segments),
                "stage_ms": {k: v / args.steps for k, v in stage.items()},
                "clocks": clk, "roofline": roof, "hbm_stages": hbm_stages,
                "e2e": {"value": e2e_value, "unit": "rays/s", "h2d_bytes_per_step": 48 * world,
                        "d2h_bytes_per_step": W * H * 16 * world},
                "gpu_launches": int(launches)}
        if args.all_configs:
            scene.close()
            del rgb, depth
            line["other_configs"] = [time_config(r360, c, precision) for c in (1, 2, 4, 5) if c != args.config]
            # the paper times its perspective (roaming) view at 720p: same scene, 90 degree pinhole
            line["other_configs"].append(time_config(r360, args.config, precision, pinhole=(1280, 720, 640.0)))
            line["extras"] = time_extras(r360, args.config)
        if not args.no_cpu_baseline:
            cb = oracle_sample(sc, args.ref_row_stride)
            line["cpu_baseline"] = {"value": cb["rays_per_s"], "unit": "rays/s", "cores": cb["cores"],
                                    "kind": "oracle", "sample": cb["sample"]}
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
