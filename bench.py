#!/usr/bin/env python
"""bench.py — counterfactual state-renders/s of the whole hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg1|cfg2|cfg4|cfg0]

A step = one frame of the workload through every stage of the path:
closure, per-variant deformation + EWA projection, tile binning + radix sort, state-blocked
compositing of B states (images materialised in HBM) with the fused per-state distortion against the
full-state render of the same frame, and the per-group utility aggregation.

N > 1 (torchrun): frames are independent units; rank r renders frames r, r+N, ... — no data-path
collective ("weak" scaling: every rank does K steps).  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2606_17212_b200 import shard, synth  # noqa: E402

# FLOP accounting of the compositing kernel, FMA = 2 flop:
#   per (pixel, record) alpha evaluation : dx, dy (2) + u (1) + s (2) + q (1) + v (1) + q (2) + o*e (1)               = 10
#   per (pixel, record, state) update    : w = alpha*T (1) + T' = T - w (1) + 3 FMA (6) + the T' < 1e-4 compare (1) =  9
#   literal per-state model: 20 flop per logical (pixel, Gaussian, state) pair
FLOP_SHARED, FLOP_STATE, FLOP_LITERAL = 10.0, 9.0, 20.0
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # 74.4: SMs x FP32 lanes x 2 x max SM clock


def build_workload(name: str, n_frames: int):
    if name == "cfg0":
        wl = synth.workload_cfg0()
        wl.frames = wl.frames * n_frames
        wl.levels = wl.levels * n_frames
        e = np.zeros(0, np.int32)
        wl.idx_without, wl.idx_with, wl.group_id, wl.G = [e] * n_frames, [e] * n_frames, [e] * n_frames, 0
        return wl
    if name == "cfg1":
        return synth.workload_cfg1(n_frames=n_frames)
    if name == "cfg1r":   # cfg1 with the full representation: delta2/delta3 + scale/rotation/opacity refinements
        wl = synth.workload_cfg1(n_frames=n_frames)
        wl.scene = synth.with_attribute_refinements(synth.with_position_residuals(wl.scene))
        wl.name = "cfg1r_full_representation_800x800_B256"
        return wl
    if name == "cfg2":
        return synth.workload_cfg2(n_frames=n_frames)
    if name == "cfg3":
        return synth.workload_cfg3(n_views=max(1, min(8, n_frames)))
    if name == "cfg4":
        wl = synth.workload_cfg4()
        return wl
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md): an NVML polling thread
    (every 2 ms, so that even a 100 ms region gets dozens of samples); nvidia-smi is the fallback."""
    REASONS = (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("hw_thermal_slowdown", 0x40),
               ("sw_thermal_slowdown", 0x20))

    def __init__(self, index: int):
        self.index, self.rows, self.stop_flag, self.thread, self.err = index, [], False, None, None

    def _poll(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if vis:
                try:
                    idx = int(vis.split(",")[self.index])
                except (ValueError, IndexError):
                    pass
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            mx = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            while not self.stop_flag:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                try:
                    pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                except Exception:
                    pw = None
                self.rows.append((sm, mx, rs, pw))
                time.sleep(0.002)
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def start(self):
        self.thread = threading.Thread(target=self._poll, daemon=True)
        self.thread.start()
        time.sleep(0.05)   # let NVML initialise before the timed region starts

    def mark(self):
        """Samples taken before this call (NVML start-up, idle) are dropped."""
        self.rows.clear()

    def stop(self) -> dict:
        self.stop_flag = True
        if self.thread is not None:
            self.thread.join(timeout=2.0)
        if not self.rows:
            return self._smi_once()
        sm = [r[0] for r in self.rows]
        reasons = sorted({n for r in self.rows for n, bit in self.REASONS if r[2] & bit})
        pw = [r[3] for r in self.rows if r[3] is not None]
        return {"sm_mhz": float(np.median(sm)), "sm_min_mhz": float(min(sm)), "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons, "source": "nvml"}

    def _smi_once(self) -> dict:
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            o = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=20).stdout.strip().splitlines()[0]
            f = [x.strip() for x in o.split(",")]
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            return {"sm_mhz": float(f[0]), "sm_max_mhz": float(f[1]), "power_w_max": float(f[2]), "samples": 1,
                    "reasons": sorted(n for n, v in zip(names, f[3:7]) if v.lower().startswith("active")),
                    "source": f"nvidia-smi after the region (nvml: {self.err})"}
        except Exception as e:  # noqa: BLE001
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [f"unavailable: {self.err}; {e!r}"]}


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_sample(wl, frame: int, n_states: int):
    """Times the CPU oracle, as it stands, on the first n_states states of a frame (+ the full-state
    reference and the distortion).  Returns seconds."""
    from oracle import oracle as O
    cam, t = wl.frames[frame]
    osc = oracle_sample.cache.get(wl.name)
    if osc is None:
        oracle_sample.cache.clear()                       # one workload's scene at a time
        osc = oracle_sample.cache[wl.name] = O.OracleScene(wl.scene)
    lv = np.ascontiguousarray(wl.levels[frame][:n_states])
    t0 = time.perf_counter()
    full = np.full((1, wl.scene.C), 3, np.int8)
    both = np.concatenate([lv, full], axis=0)
    imgs, _ = osc.render_batch(cam, t, both)
    O.distortion(imgs[:-1], imgs[-1])
    return time.perf_counter() - t0, O.num_threads()


oracle_sample.cache = {}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = build_workload(args.workload, max(1, min(args.steps + args.warmup, 8)))
    cam0, _ = wl.frames[0]
    B = wl.levels[0].shape[0]
    n_s = min(args.ref_states, B)
    for k in range(args.warmup):
        oracle_sample(wl, k % len(wl.frames), n_s)
    tot, cores = 0.0, 1
    for k in range(args.steps):
        dt, cores = oracle_sample(wl, k % len(wl.frames), n_s)
        tot += dt
    value = n_s * args.steps / tot
    sample = f"{n_s} of {B} states per frame (+1 full-state reference render and the MSE/PSNR reduction), {args.steps} frames"
    line = {"impl": "reference", "metric": "counterfactual_state_renders_per_s", "value": value, "unit": "states/s",
            "mpix_states_per_s": value * cam0.W * cam0.H / 1e6, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (decisions in f32)", "data": "synthetic",
            "config": {"workload": wl.name, "states_per_frame": B, "resolution": [cam0.W, cam0.H],
                       "gaussians": wl.scene.N, "clusters": wl.scene.C},
            "cpu_baseline": {"value": value, "unit": "states/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "states/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ our arm
KERNEL_SOURCE = ROOT / "paper_2606_17212_b200" / "csrc" / "k_composite_q.cu"


def traffic_record(workload_name: str) -> dict:
    """roofline.traffic = DRAM bytes per launch of the dominant kernel from an ncu --set full capture, recorded in
    profiles/traffic.txt together with the SHA-256 of the kernel source it was taken on.  The number is only
    reported while the kernel source still has that hash; otherwise traffic is null and the reason is given."""
    import hashlib
    tp = ROOT / "profiles" / "traffic.txt"
    out = {"traffic": None, "traffic_source": None}
    if not tp.exists():
        return out
    sha_now = hashlib.sha256(KERNEL_SOURCE.read_bytes()).hexdigest() if KERNEL_SOURCE.exists() else None
    meta, val = {}, None
    for ln in tp.read_text().splitlines():
        f = ln.split()
        if ln.startswith("# ") and len(f) >= 3 and f[1].endswith(":"):
            meta[f[1][:-1]] = " ".join(f[2:])
        elif len(f) == 2 and not ln.startswith("#") and f[0] == workload_name:
            val = int(f[1])
    src = {"file": "profiles/traffic.txt", "commit": meta.get("commit"), "command": meta.get("command"),
           "kernel_source": str(KERNEL_SOURCE.relative_to(ROOT)), "kernel_source_sha256": meta.get("kernel_source_sha256"),
           "matches_current_source": sha_now is not None and sha_now == meta.get("kernel_source_sha256")}
    out["traffic_source"] = src
    if val is not None and src["matches_current_source"]:
        out["traffic"] = val
    elif val is not None:
        src["note"] = "the kernel source changed since the capture: traffic withheld"
    return out


def measure_ours(args, workload: str, steps: int, warmup: int, full: bool):
    """One workload through the C ABI.  full = the N = 1 bench line (repetitions, sustained pass, end-to-end call,
    the run without images); otherwise the compact sub-record of `workloads` (value, roofline, clocks, CPU sample)."""
    import torch
    from paper_2606_17212_b200 import build as gbuild
    gbuild.build()
    from paper_2606_17212_b200 import gsr

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but {world} rank(s) are running (WORLD_SIZE)")
    total_steps = steps + warmup
    n_frames = min(150, max(1, total_steps * world)) if workload in ("cfg1", "cfg1r") else min(8, max(1, total_steps))
    wl = build_workload(workload, n_frames)
    n_frames = len(wl.frames)
    scene = gsr.Scene(wl.scene)
    if args.state_block:
        gsr.set_option("state_block", args.state_block)
    cam0, _ = wl.frames[0]
    B, Cn, G = wl.levels[0].shape[0], wl.scene.C, wl.G
    W, H = cam0.W, cam0.H
    cams = [gsr.camera_struct(c) for c, _ in wl.frames]
    ts = [float(t) for _, t in wl.frames]
    dev = torch.device("cuda", local)
    lv_dev = [torch.from_numpy(np.ascontiguousarray(l)).to(dev) for l in wl.levels]
    iwo = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in wl.idx_without]
    iw = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in wl.idx_with]
    gid = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in wl.group_id]
    # ---- frames in flight: frame k runs on stream k mod F with its own workspace and outputs, so that the
    #      latency-bound projection / sort launches of one frame fill the SMs the compositing tail of another
    #      leaves idle.  F is capped so that the image buffers stay under 48 GB.
    img_bytes = B * H * W * 12
    F = max(1, min(args.frames_in_flight, max(1, int(48e9 // max(img_bytes, 1)))))
    bufs = []
    for _ in range(F):
        bufs.append({"ws": scene.new_workspace(cam0, B),
                     "out": torch.empty((B, H, W, 3), dtype=torch.float32, device=dev),
                     "ref": torch.empty((H, W, 3), dtype=torch.float32, device=dev),
                     "mse": torch.empty(B, dtype=torch.float64, device=dev),
                     "psnr": torch.empty(B, dtype=torch.float32, device=dev),
                     "util": torch.zeros((max(G, 1), 9), dtype=torch.float64, device=dev),
                     "stream": torch.cuda.Stream(device=dev)})
    ws = bufs[0]["ws"]

    def frame_of(step):
        return shard.frame_for_step(step, rank, world, n_frames)

    def frame_into(b, k, images):
        f = frame_of(k)
        scene.render_states_vs_full(cams[f], ts[f], lv_dev[f], b["ws"], b["ref"], b["mse"], b["psnr"],
                                    out=b["out"] if images else None)
        if G > 0:
            gsr.group_utility_into(b["mse"], b["psnr"], iwo[f], iw[f], gid[f], G, b["util"])

    def step(k, images=True):                    # pipelined: F frames in flight
        b = bufs[k % F]
        with torch.cuda.stream(b["stream"]):
            frame_into(b, k, images)

    def step_serial(k, images=True):             # one frame at a time on the current stream
        frame_into(bufs[0], k, images)

    def timed(fn, k0, K, pipelined=False, finish=None):
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        main = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(main)
        if pipelined:
            for b in bufs:
                b["stream"].wait_event(e0)
        for k in range(k0, k0 + K):
            fn(k)
        if pipelined:
            for b in bufs:
                main.wait_stream(b["stream"])
        if finish is not None:
            finish()                     # host threads: every call has returned (each synchronises its stream)
        e1.record(main)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        return shard.max_over_ranks(ms, device=dev)

    # ---- warm-up, then the timed region (device-resident inputs), clocks sampled during it
    for k in range(warmup):
        step(k)
    torch.cuda.synchronize()
    for b in bufs[:min(F, warmup)]:                  # the workspaces a warm-up step has written
        scene.status(b["ws"])
    l0 = gsr.launch_count()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.mark()
    # protocol of PAPER.md:142 ("5 warm-ups, 3 repetitions, Student-t 95 % CI"): the timed region of exactly
    # `steps` steps is repeated; `value` is the mean over the repetitions
    n_rep = 3 if full else 1
    ms_reps = []
    for r in range(n_rep):
        ms_reps.append(timed(step, warmup + r * steps, steps, pipelined=True))
        if r == 0:
            launches = gsr.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms = float(np.mean(ms_reps))
    value_reps = [B * steps * world / (m * 1e-3) for m in ms_reps]
    value = float(np.mean(value_reps))
    T975 = {1: 12.706, 2: 4.303, 3: 3.182, 4: 2.776}      # Student t, 97.5 %, n - 1 degrees of freedom
    ci95 = (T975[n_rep - 1] * float(np.std(value_reps, ddof=1)) / np.sqrt(n_rep)) if n_rep > 1 else None

    # ---- sustained pass: the same pipelined steps for >= 2 s, clocks and power sampled throughout, so that the
    #      number is also on record at the power-steady clock
    sustained = None
    if full:
        n_sus = int(np.ceil(2200.0 / max(ms / steps, 1e-3)))
        sus = ClockSampler(local)
        if rank == 0:
            sus.start()
            sus.mark()
        ms_sus = timed(step, warmup, n_sus, pipelined=True)
        sus_clocks = sus.stop() if rank == 0 else None
        sustained = {"value": B * n_sus * world / (ms_sus * 1e-3), "unit": "states/s", "steps": n_sus,
                     "seconds": ms_sus * 1e-3, "ms_per_step": ms_sus / n_sus, "clocks": sus_clocks}

    # ---- the same steps one frame at a time with CUDA events around every k_composite_q launch and around the
    #      memory-bound phases: what the roofline objects are computed from (events of overlapping streams
    #      would count co-running kernels twice)
    gsr.set_option("profile", 1)
    ms_serial = timed(step_serial, warmup, steps)
    comp_ms, comp_n = gsr.profile_read()
    proj_ms, sort_ms, ph_n = gsr.profile_read_phases()
    gsr.set_option("profile", 0)
    keys = scene.status(ws)

    # ---- the same path without materialising the images (distortion/utility only), reported beside it
    ms_noimg = timed(lambda k: step(k, images=False), warmup, steps, pipelined=True) if full else None

    e2e = None
    if full:
        # ---- end to end through the host-buffer C-ABI call: pinned host inputs, H2D + D2H inside the timed region
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_lv = [pin(l) for l in wl.levels]
        h_iwo, h_iw, h_gid = [pin(a) for a in wl.idx_without], [pin(a) for a in wl.idx_with], [pin(a) for a in wl.group_id]
        # F host threads, each with its own stream, workspace and pinned result buffers, call the (blocking) host
        # API round-robin: the same frames-in-flight pipeline as above, driven through the public call
        from concurrent.futures import ThreadPoolExecutor
        lanes = []
        for _ in range(F):
            h_mse = torch.empty(B, dtype=torch.float64).pin_memory()
            h_psnr = torch.empty(B, dtype=torch.float32).pin_memory()
            h_util = torch.zeros((max(G, 1), 9), dtype=torch.float64).pin_memory()
            lanes.append({"pins": (h_mse, h_psnr, h_util), "ws": None, "stream": torch.cuda.Stream(device=dev),
                          "host": (h_mse.numpy(), h_psnr.numpy(), h_util.numpy().view(gsr.UTILITY_DTYPE).reshape(-1)),
                          "pool": ThreadPoolExecutor(max_workers=1), "pending": []})

        def e2e_frame(lane, k):
            f = frame_of(k)
            torch.cuda.set_device(local)
            with torch.cuda.stream(lane["stream"]):
                r = scene.utility_frame_host(cams[f], ts[f], h_lv[f].numpy(), h_iwo[f].numpy(), h_iw[f].numpy(),
                                             h_gid[f].numpy(), G, workspace=lane["ws"], materialise=True, bufs=lane["host"])
            lane["ws"] = r[4]

        def step_e2e(k):
            lane = lanes[k % F]
            lane["pending"].append(lane["pool"].submit(e2e_frame, lane, k))

        def finish_e2e():
            for lane in lanes:
                for fut in lane["pending"]:
                    fut.result()
                lane["pending"].clear()

        for b in bufs:
            b["out"] = None
        torch.cuda.empty_cache()
        for k in range(max(min(warmup, 3), F)):
            step_e2e(k)
        finish_e2e()
        ms_e2e = timed(step_e2e, warmup, steps, finish=finish_e2e)
        for lane in lanes:
            lane["pool"].shutdown()
        n_pairs = int(wl.idx_without[0].size)
        e2e = {"value": B * steps * world / (ms_e2e * 1e-3), "unit": "states/s",
               "h2d_bytes_per_step": int(B * Cn + 3 * 4 * n_pairs), "d2h_bytes_per_step": int(B * 8 + B * 4 + G * 72),
               "ms_per_step": ms_e2e / steps,
               "host_threads": F,
               "note": "gsr_utility_frame_host: pinned host levels/pairs in, mse/psnr/utilities out; images materialised on device; %d host threads, one stream + workspace each" % F}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None
    for b in bufs:
        b["out"] = None
    torch.cuda.empty_cache()

    # ---- roofline of the dominant kernel (k_composite_q): counted work / CUDA-event time / FP32 peak
    bufs[0]["out"] = torch.empty((B, H, W, 3), dtype=torch.float32, device=dev)
    n_cnt = min(steps, 6)
    cnt = np.zeros(3, np.float64)
    for k in range(warmup, warmup + n_cnt):
        step_serial(k)
        cnt += scene.debug_pair_counts(ws)
    cnt *= steps / n_cnt                       # scaled to the timed region (frames are statistically alike)
    comp_s = comp_ms * 1e-3
    flop_alg = cnt[0] * FLOP_SHARED + cnt[1] * FLOP_STATE
    peak_meas = gsr.measure_fp32_peak()
    achieved = flop_alg / comp_s / 1e12 if comp_s > 0 else 0.0
    roofline = {"kernel": "k_composite_q", "bound": "alu", "achieved": achieved, "peak": peak_meas, "unit": "TFLOP/s",
                "frac": achieved / peak_meas if peak_meas else None, "traffic": None,
                "peak_kind": "measured here: FFMA-chain kernel (gsr_measure_fp32_peak); nominal %.1f" % NOMINAL_FP32_TFLOPS,
                "kernel_ms_per_launch": comp_ms / max(comp_n, 1), "kernel_launches": comp_n,
                "kernel_share_of_step": comp_ms / ms_serial,
                "measured_on": "the same %d steps run one frame at a time (%.3f ms/step), CUDA events around every launch" % (steps, ms_serial / steps),
                "alpha_evals_per_step": cnt[0] / steps, "state_updates_per_step": cnt[1] / steps,
                "logical_pairs_per_step": cnt[2] / steps,
                "literal_equiv_tflops": cnt[2] * FLOP_LITERAL / comp_s / 1e12 if comp_s > 0 else 0.0,
                "literal_equiv_frac": (cnt[2] * FLOP_LITERAL / comp_s / 1e12 / peak_meas) if comp_s > 0 and peak_meas else None,
                "image_write_gbs": B * H * W * 12 * steps / comp_s / 1e9 if comp_s > 0 else None}
    # ---- the memory-bound phases a1-a3 against the HBM roofline (algorithmic bytes per unit)
    K = (wl.scene.sh_degree + 1) ** 2
    n_rec = scene.V * wl.scene.N
    b_gauss = 48 + 2 * 16 * ((3 * K + 3) // 4) + 4 * ((3 * wl.scene.R + 3) // 4) + (24 if scene.V == 4 else 0)
    proj_bytes = wl.scene.N * b_gauss + n_rec * 88
    # a3 (k_sort.cu): count pass reads count + rect (12 B / record); the scatter reads them again with the depth
    # bits (16 B / record) and writes 8 B / key; the per-tile sort reads 8 B and writes 12 B / key
    sort_bytes = n_rec * 28 + keys * 28
    hbm_peak, hbm_kind = 6650.0, "fallback (B200_PROFILING.md)"
    mp = ROOT / "MEASURED_PEAKS.json"
    if mp.exists():
        try:
            hbm_peak, hbm_kind = float(json.loads(mp.read_text())["hbm_gbs"]), "MEASURED_PEAKS.json"
        except Exception:
            pass
    phases = None
    if ph_n > 0:
        pg = proj_bytes * ph_n / (proj_ms * 1e-3) / 1e9
        sg = sort_bytes * ph_n / (sort_ms * 1e-3) / 1e9
        phases = {"bound": "hbm", "peak": hbm_peak, "peak_kind": hbm_kind, "unit": "GB/s", "frames": ph_n,
                  "project": {"ms_per_frame": proj_ms / ph_n, "algorithmic_bytes": int(proj_bytes), "achieved": pg,
                              "frac": pg / hbm_peak},
                  "bin_sort": {"ms_per_frame": sort_ms / ph_n, "algorithmic_bytes": int(sort_bytes), "achieved": sg,
                               "frac": sg / hbm_peak, "launches_per_frame": 3,
                               "note": "counting sort by tile + one bitonic sort per tile segment (%d keys)" % keys},
                  "share_of_step": (proj_ms + sort_ms) / ms_serial}
    roofline.update(traffic_record(wl.name))

    # ---- backward (gsr_render_backward: the compositor; gsr_project_backward: projection, SH colour, Eq. (1) and the
    #      activation; SURVEY.md §8(f)-4 follow-on): forward + backward of the same frames, one frame in flight,
    #      dL/d(image) resident (a fixed random tensor: the kernels' work does not depend on its values)
    backward = None
    if full and not args.no_backward:
        n_b = min(steps, 6)
        gimg = torch.randn((B, H, W, 3), dtype=torch.float32, device=dev) * (2.0 / (3.0 * W * H))
        b0 = bufs[0]
        grec = torch.empty((scene.num_records(), 12), dtype=torch.float32, device=dev)
        chain = True                              # 2-record scenes: gsr_project_backward; cfg1r: gsr_project_backward_full
        gpar = [None]

        def fwd_bwd(k, mode=2):
            frame_into(b0, k, True)
            if mode >= 1:
                scene.render_backward(b0["ws"], b0["out"], gimg, grad=grec)
            if mode >= 2 and chain:
                f = frame_of(k)
                pb = scene.project_backward if scene.V == 2 else scene.project_backward_full
                gpar[0] = pb(cams[f], ts[f], grec, out=gpar[0])

        for k in range(2):
            fwd_bwd(warmup + k)
        ms_fbp = timed(fwd_bwd, warmup, n_b)
        ms_fb = timed(lambda k: fwd_bwd(k, 1), warmup, n_b)
        ms_f = timed(lambda k: fwd_bwd(k, 0), warmup, n_b)
        backward = {"value": B * n_b * world / (ms_fbp * 1e-3), "unit": "states/s (forward + backward)",
                    "ms_per_step_forward_backward": ms_fbp / n_b, "ms_per_step_forward": ms_f / n_b,
                    "ms_per_step_backward": (ms_fb - ms_f) / n_b,
                    "ms_per_step_project_backward": (ms_fbp - ms_fb) / n_b if chain else None, "steps": n_b,
                    "note": "gsr_render_states_vs_full + gsr_render_backward (grad [records, 12] summed over the %d "
                            "states) + gsr_project_backward (gradients of the scene's parameters), one frame in flight" % B}
        del gimg, grec

    # ---- CPU oracle on this box's cores, bounded sample of the same workload
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # cfg1 (the bench line): all 256 states of two frames, ~15 s of CPU work; sub-records: 16 states of two frames
        n_s = min(4 * args.ref_states, B) if full else min(16, B)
        f0, f1 = frame_of(warmup), frame_of(warmup + 1)
        dt0, cores = oracle_sample(wl, f0, n_s)
        dt1, _ = oracle_sample(wl, f1, n_s)
        dt = dt0 + dt1
        cpu = {"value": 2 * n_s / dt, "unit": "states/s", "cores": cores, "kind": "oracle",
               "sample": f"first {n_s} of {B} states of frames {f0} and {f1} (+ the full-state reference render and MSE/PSNR of each), {dt:.1f} s"}

    line = {"metric": "counterfactual_state_renders_per_s", "value": value, "unit": "states/s",
            "mpix_states_per_s": value * W * H / 1e6, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps, "ms_per_step_one_frame_in_flight": ms_serial / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "states_per_frame": B, "resolution": [W, H], "gaussians": wl.scene.N,
                       "clusters": Cn, "sh_degree": wl.scene.sh_degree, "R": wl.scene.R, "frames": n_frames,
                       "images_materialised": True, "frames_in_flight": F, "state_block": args.state_block or "default", "keys_per_frame": keys,
                       "l2": "per-step working set (%.2f GB of images written) exceeds the 126 MB L2; every step is a different frame" % (B * H * W * 12 / 1e9),
                       "parallelism": "frames sharded over ranks, no collective" if world > 1 else "1 GPU"},
            "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline, "memory_phases": phases,
            "cpu_baseline": cpu}
    if full:
        line.update({"repetitions": n_rep, "value_reps": value_reps, "value_ci95": ci95,
                     "ms_per_step_reps": [m / steps for m in ms_reps], "sustained": sustained,
                     "value_without_images": B * steps * world / (ms_noimg * 1e-3), "e2e": e2e, "backward": backward,
                     "context": {"paper_h100_pcie_utility_states_per_s": 1889.7,
                                 "note": "PAPER.md:150, other hardware, unstated resolution/scene: context only"}})
    if dist is not None:
        dist.destroy_process_group()
    scene.close()
    del bufs, lv_dev
    torch.cuda.empty_cache()
    return line


# ------------------------------------------------------------------------------------------------ atlas workload
def measure_atlas(args, steps: int, warmup: int, full: bool):
    """--workload atlas.  A step = one view of the partial-state atlas:
    utility sweep (2 x 4C x n_ctx states, fused distortion) -> Eq. (3)-(4) -> three policy orders -> frontier
    states at 4 matched budgets -> 8197 sampled states + 12 frontier states rendered (fused distortion, no
    images: 8209 x 800 x 800 x 12 B would be 63 GB) -> state bytes -> best sampled state per budget."""
    import torch
    from paper_2606_17212_b200 import build as gbuild
    gbuild.build()
    from paper_2606_17212_b200 import gsr

    assert int(os.environ.get("WORLD_SIZE", "1")) == 1, "the atlas workload is a 1-GPU bench line"
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n_views = max(1, min(steps + warmup, 4))
    wl = synth.workload_atlas(n_views=n_views)
    scene = gsr.Scene(wl.scene)
    Cn, G = wl.scene.C, wl.G
    cam0, _ = wl.frames[0]
    W, H = cam0.W, cam0.H
    cams = [gsr.camera_struct(c) for c, _ in wl.frames]
    ts = [float(t) for _, t in wl.frames]
    nb, n_pol = len(wl.budget_fracs), 3
    Bs, Ba = wl.sweep_levels[0].shape[0], wl.atlas_levels[0].shape[0]
    Bt = Ba + n_pol * nb
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    sweep = [to_dev(l) for l in wl.sweep_levels]
    iwo, iw, gid = [to_dev(a) for a in wl.idx_without], [to_dev(a) for a in wl.idx_with], [to_dev(a) for a in wl.group_id]
    batch = [torch.cat([to_dev(l), torch.zeros((n_pol * nb, Cn), dtype=torch.int8, device=dev)]) for l in wl.atlas_levels]
    raw = to_dev(wl.raw_bytes)
    wire = gsr.group_wire_bytes(raw)
    total_wire = int(wire.sum().item())
    budgets = to_dev(np.asarray([int(f * total_wire) for f in wl.budget_fracs], np.int64))
    ws = scene.new_workspace(cam0, Bt)
    ref = torch.empty((H, W, 3), dtype=torch.float32, device=dev)
    mse_s, psnr_s = torch.empty(Bs, dtype=torch.float64, device=dev), torch.empty(Bs, dtype=torch.float32, device=dev)
    mse_a, psnr_a = torch.empty(Bt, dtype=torch.float64, device=dev), torch.empty(Bt, dtype=torch.float32, device=dev)
    util = torch.zeros((G, 9), dtype=torch.float64, device=dev)
    cost = torch.empty(Bt, dtype=torch.int64, device=dev)
    best = torch.empty(nb, dtype=torch.int32, device=dev)
    n_frames = len(wl.frames)

    def step(k):
        f = k % n_frames
        scene.render_states_vs_full(cams[f], ts[f], sweep[f], ws, ref, mse_s, psnr_s, out=None)
        gsr.group_utility_into(mse_s, psnr_s, iwo[f], iw[f], gid[f], G, util)
        score = util[:, 7].contiguous()                      # risk-adjusted utility in dB (Eq. 4)
        for p in range(n_pol):
            order, _ = gsr.frontier_order(score, wire, p)
            gsr.frontier_states(order, wire, budgets, levels_out=batch[f][Ba + p * nb: Ba + (p + 1) * nb])
        scene.render_states_vs_full(cams[f], ts[f], batch[f], ws, ref, mse_a, psnr_a, out=None)
        gsr.state_bytes(batch[f], wire, out=cost)
        gsr.best_state_under_budget(psnr_a[:Ba], cost[:Ba], budgets, out=best)

    def timed(fn, k0, K):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(k0, k0 + K):
            fn(k)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    for k in range(warmup):
        step(k)
    scene.status(ws)
    gsr.set_option("profile", 1)
    l0 = gsr.launch_count()
    sampler = ClockSampler(0)
    sampler.start()
    sampler.mark()
    ms = timed(step, warmup, steps)
    clocks = sampler.stop()
    launches = gsr.launch_count() - l0
    comp_ms, comp_n = gsr.profile_read()
    gsr.set_option("profile", 0)
    scene.status(ws)
    states_per_step = Bs + Bt
    value = states_per_step * steps / (ms * 1e-3)

    # end to end: pinned host levels in, every result of the step back on the host
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_sweep, h_atlas = [pin(l) for l in wl.sweep_levels], [pin(l) for l in wl.atlas_levels]
    h_out = {"psnr": torch.empty(Bt, dtype=torch.float32).pin_memory(), "cost": torch.empty(Bt, dtype=torch.int64).pin_memory(),
             "best": torch.empty(nb, dtype=torch.int32).pin_memory(), "util": torch.empty((G, 9), dtype=torch.float64).pin_memory()}

    def step_e2e(k):
        f = k % n_frames
        sweep[f].copy_(h_sweep[f], non_blocking=True)
        batch[f][:Ba].copy_(h_atlas[f], non_blocking=True)
        step(k)
        h_out["psnr"].copy_(psnr_a, non_blocking=True)
        h_out["cost"].copy_(cost, non_blocking=True)
        h_out["best"].copy_(best, non_blocking=True)
        h_out["util"].copy_(util, non_blocking=True)
        torch.cuda.current_stream().synchronize()

    e2e = None
    if full:
        step_e2e(0)
        ms_e2e = timed(step_e2e, warmup, steps)
        e2e = {"value": states_per_step * steps / (ms_e2e * 1e-3), "unit": "states/s",
               "h2d_bytes_per_step": int((Bs + Ba) * Cn), "d2h_bytes_per_step": int(Bt * 12 + nb * 4 + G * 72),
               "ms_per_step": ms_e2e / steps}

    # roofline of the dominant kernel, counted work of the two render calls of one step
    cnt = np.zeros(3, np.float64)
    f = warmup % n_frames
    scene.render_states_vs_full(cams[f], ts[f], sweep[f], ws, ref, mse_s, psnr_s, out=None)
    cnt += scene.debug_pair_counts(ws)
    scene.render_states_vs_full(cams[f], ts[f], batch[f], ws, ref, mse_a, psnr_a, out=None)
    cnt += scene.debug_pair_counts(ws)
    comp_s = comp_ms * 1e-3 / steps
    peak = gsr.measure_fp32_peak()
    achieved = (cnt[0] * FLOP_SHARED + cnt[1] * FLOP_STATE) / comp_s / 1e12
    roofline = {"kernel": "k_composite_q", "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": None,
                "peak_kind": "measured here: FFMA-chain kernel (gsr_measure_fp32_peak); nominal %.1f" % NOMINAL_FP32_TFLOPS,
                "kernel_ms_per_launch": comp_ms / max(comp_n, 1), "kernel_launches": comp_n,
                "kernel_share_of_step": comp_ms / ms,
                "alpha_evals_per_step": cnt[0], "state_updates_per_step": cnt[1],
                "logical_pairs_per_step": cnt[2], "literal_equiv_tflops": cnt[2] * FLOP_LITERAL / comp_s / 1e12}

    psnr_h, best_h = psnr_a.cpu().numpy(), best.cpu().numpy()
    result = {"budget_fracs": list(wl.budget_fracs),
              "sampled_oracle_psnr_db": [float(psnr_h[i]) if i >= 0 else None for i in best_h],
              "utility_order_psnr_db": [float(v) for v in psnr_h[Ba:Ba + nb]],
              "nominal_order_psnr_db": [float(v) for v in psnr_h[Ba + nb:Ba + 2 * nb]],
              "byte_greedy_psnr_db": [float(v) for v in psnr_h[Ba + 2 * nb:Ba + 3 * nb]]}
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        osc = O.OracleScene(wl.scene)
        n_s = min(args.ref_states if full else 16, Ba)
        cam, t = wl.frames[f]
        t0 = time.perf_counter()
        imgs, _ = osc.render_batch(cam, t, np.concatenate([wl.atlas_levels[f][:n_s], np.full((1, Cn), 3, np.int8)]))
        O.distortion(imgs[:-1], imgs[-1])
        dt = time.perf_counter() - t0
        cpu = {"value": n_s / dt, "unit": "states/s", "cores": O.num_threads(), "kind": "oracle",
               "sample": f"first {n_s} of {Ba} atlas states of view {f} (+ full-state reference and MSE/PSNR), {dt:.1f} s"}
    line = {"metric": "counterfactual_state_renders_per_s", "value": value, "unit": "states/s",
            "mpix_states_per_s": value * W * H / 1e6, "n_gpus": 1, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "states_per_step": states_per_step, "sweep_states": Bs, "atlas_states": Ba,
                       "frontier_states": n_pol * nb, "resolution": [W, H], "gaussians": wl.scene.N, "clusters": Cn,
                       "images_materialised": False,
                       "l2": "each step projects, sorts and composites a different view; no output is re-read"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
            "atlas": result}
    scene.close()
    return line



def measure_train(args, steps: int, warmup: int, full: bool):
    """--workload train: the forward-plus-backward render step at the size of the paper's Table 2 ("2.7M primitives",
    128 worlds).  A step = one frame: B states and the full state rendered (images
    materialised, MSE fused), gsr_distortion_backward (dL/d(image) of mean_b MSE + 0.20 (1 - SSIM) against the
    full-state render), gsr_render_backward, gsr_project_backward -> the gradients of the scene's
    parameters.
    Reports world-frames/s (a world-frame = one rendered receiver-state image, the paper's unit) with three
    repetitions and a Student-t 95 % interval, and the split of the step.  The paper's scene, resolution and masks are
    not given: context for BASELINE.md row 2, not a comparison."""
    import torch
    from paper_2606_17212_b200 import build as gbuild
    gbuild.build()
    from paper_2606_17212_b200 import gsr

    assert int(os.environ.get("WORLD_SIZE", "1")) == 1, "the train workload is a 1-GPU bench line"
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n_frames = max(1, min(steps + warmup, 3))
    wl = synth.workload_train(n_frames=n_frames, B=args.train_worlds, n_gaussians=args.train_gaussians)
    scene = gsr.Scene(wl.scene)
    cam0, _ = wl.frames[0]
    W, H, B = cam0.W, cam0.H, wl.levels[0].shape[0]
    cams = [gsr.camera_struct(c) for c, _ in wl.frames]
    ts = [float(t) for _, t in wl.frames]
    lv = [torch.from_numpy(np.ascontiguousarray(l)).to(dev) for l in wl.levels]
    ws = scene.new_workspace(cam0, B)
    out = torch.empty((B, H, W, 3), dtype=torch.float32, device=dev)
    ref = torch.empty((H, W, 3), dtype=torch.float32, device=dev)
    mse, psnr = torch.empty(B, dtype=torch.float64, device=dev), torch.empty(B, dtype=torch.float32, device=dev)
    wgt = torch.full((B,), 1.0 / B, dtype=torch.float64, device=dev)
    gimg = torch.empty((B, H, W, 3), dtype=torch.float32, device=dev)
    grec = torch.empty((scene.num_records(), 12), dtype=torch.float32, device=dev)
    dws = torch.empty(int(gsr.lib().gsr_distortion_backward_workspace_bytes(H, W)), dtype=torch.uint8, device=dev)
    gpar = [None]

    def step(k, mode=3):
        f = k % n_frames
        scene.render_states_vs_full(cams[f], ts[f], lv[f], ws, ref, mse, psnr, out=out)
        if mode >= 1:
            gsr.distortion_backward(out, ref, wgt, 0.20, out=gimg, workspace=dws)
        if mode >= 2:
            scene.render_backward(ws, out, gimg, grad=grec)
        if mode >= 3:
            gpar[0] = scene.project_backward(cams[f], ts[f], grec, out=gpar[0])

    def timed(fn, k0, K):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(k0, k0 + K):
            fn(k)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    for k in range(warmup):
        step(k)
    keys = scene.status(ws)
    l0 = gsr.launch_count()
    sampler = ClockSampler(0)
    sampler.start()
    sampler.mark()
    reps = [timed(step, warmup + r * steps, steps) for r in range(3 if full else 1)]
    clocks = sampler.stop()
    launches = (gsr.launch_count() - l0) // len(reps)
    ms_fb = timed(lambda k: step(k, 2), warmup, steps)
    ms_fd = timed(lambda k: step(k, 1), warmup, steps)
    ms_f = timed(lambda k: step(k, 0), warmup, steps)
    vals = [B * steps / (m * 1e-3) for m in reps]
    value = float(np.mean(vals))
    T975 = {1: 12.706, 2: 4.303, 3: 3.182, 4: 2.776}      # Student t, 97.5 %, n - 1 degrees of freedom
    ci = float(T975[len(vals) - 1] * np.std(vals, ddof=1) / np.sqrt(len(vals))) if len(vals) > 1 else None
    ms = float(np.mean(reps))
    line = {"metric": "training_render_world_frames_per_s", "value": value, "unit": "world-frames/s (forward + backward)",
            "value_reps": vals, "value_ci95": ci, "n_gpus": 1, "steps": steps, "warmup": warmup, "ms_per_step": ms / steps,
            "ms_per_step_forward": ms_f / steps, "ms_per_step_distortion_backward": (ms_fd - ms_f) / steps,
            "ms_per_step_backward": (ms_fb - ms_fd) / steps, "ms_per_step_project_backward": (ms - ms_fb) / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "worlds": B, "resolution": [W, H], "gaussians": wl.scene.N,
                       "clusters": wl.scene.C, "sh_degree": wl.scene.sh_degree, "R": wl.scene.R, "frames": n_frames,
                       "keys_per_frame": int(keys), "images_materialised": True,
                       "l2": "per-step working set (%.2f GB of images written, %.2f GB of dL/d(image) read) exceeds the "
                             "126 MB L2; every step is a different frame" % (B * H * W * 12 / 1e9, B * H * W * 12 / 1e9)},
            "clocks": clocks, "gpu_launches": int(launches),
            "paper": {"value": 360.46, "unit": "world-frames/s", "where": "PAPER.md:238-249, Table 2, 128 worlds, H100 PCIe, "
                      "2.7M primitives, scene replicated per world; scene / resolution / masks not given: context only"}}
    scene.close()
    del out, gimg, grec, ref
    return line


SUB_WORKLOADS = ("cfg2", "cfg3", "cfg4", "atlas", "train")


def run_ours(args):
    """The N = 1 bench line: configs[1] in full (repetitions, CI, sustained pass, end-to-end, roofline, CPU sample) and
    — SURVEY.md §8(d), BASELINE.md "what we will measure" — a compact sub-record for each other workload."""
    if args.workload == "atlas":
        line = measure_atlas(args, args.steps, args.warmup, full=True)
    elif args.workload == "train":
        line = measure_train(args, max(1, min(args.steps, 6)), args.warmup, full=True)
    else:
        line = measure_ours(args, args.workload, args.steps, args.warmup, full=True)
    if line is None:                      # ranks other than 0
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.workload == "cfg1" and world == 1 and not args.no_sub_workloads:
        subs = {}
        for name in SUB_WORKLOADS:
            t0 = time.perf_counter()
            try:
                if name == "train":
                    sub = measure_train(args, 2, 3, full=False)
                else:
                    sub = measure_atlas(args, 2, 2, full=False) if name == "atlas" else measure_ours(args, name, 3, 3, full=False)
                keep = ("metric", "value", "unit", "mpix_states_per_s", "steps", "warmup", "ms_per_step", "ms_per_step_forward",
                        "ms_per_step_distortion_backward", "ms_per_step_backward", "ms_per_step_project_backward", "config", "clocks", "gpu_launches",
                        "cpu_baseline", "paper")
                rec = {k: sub[k] for k in keep if k in sub}
                r = sub.get("roofline")
                if r:
                    rec["roofline"] = {k: r[k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac",
                                                         "kernel_share_of_step") if k in r}
                rec["wall_s"] = time.perf_counter() - t0
                subs[name] = rec
            except Exception as e:  # noqa: BLE001  a sub-record must never cost the headline line
                subs[name] = {"error": repr(e)}
        line["workloads"] = subs
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=60)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg1", choices=["cfg0", "cfg1", "cfg1r", "cfg2", "cfg3", "cfg4", "atlas", "train"])
    ap.add_argument("--train-worlds", type=int, default=128, help="--workload train: states per frame (the paper's worlds)")
    ap.add_argument("--train-gaussians", type=float, default=2.7e6, help="--workload train: primitives")
    ap.add_argument("--ref-states", type=int, default=64, help="states per frame the CPU oracle renders")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-backward", action="store_true", help="skip the forward + backward timing")
    ap.add_argument("--no-sub-workloads", action="store_true",
                    help="cfg1 only: skip the compact cfg2 / cfg3 / cfg4 / atlas sub-records")
    ap.add_argument("--state-block", type=int, default=0, help="states per compositing CTA (0 = library default)")
    ap.add_argument("--frames-in-flight", type=int, default=4,
                    help="frames pipelined on separate CUDA streams, each with its own workspace and outputs")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without torchrun: start the N ranks here (one process per GPU, NCCL only for the barrier and
        # the max-over-ranks time); a box with fewer GPUs fails loudly instead of timing one GPU
        import torch
        n_dev = torch.cuda.device_count()
        if n_dev < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but this box has {n_dev} CUDA device(s)")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1",
               f"--nproc-per-node={args.gpus}", "--local-addr", "127.0.0.1", str(Path(__file__).resolve()), *sys.argv[1:]]
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # the init log (on stderr) lets the driver count the ranks
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        raise SystemExit(subprocess.call(cmd))
    run_ours(args)


if __name__ == "__main__":
    main()
