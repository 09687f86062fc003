#!/usr/bin/env python
"""bench.py -- throughput of the fisheye plane-sweep hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5|C3|P|P3|PH|PM] [--impl ours|reference]

A "step" is one pass of the whole hot path (footprint pack + fused sweep S1..S12) over one synchronized
frame set of the workload: BASELINE.json configs[4] (C5, the throughput stream: config-3 rig moving 0.5 m per frame,
192 fronto + 64 ground planes, 9x9 ZNCC, filters and masks on) by default, or configs[2] (C3) with --workload C3, or
one of the paper's own workload shapes: P = five cameras at full resolution, P3 =
three of them, PH = half resolution, PM = the multi-scale estimator (fsw_compute_depth_multires_batch).
`value` = finite (pixel, plane, view) cost evaluations per second, inputs resident in HBM; `e2e` = the same through
fsw_compute_depth_host (pinned host buffers, copies inside the timed region).  N > 1 (torchrun): frame sets are
independent, so each rank runs the same number of steps on its own frames -- no data-path collective, "weak".
--impl reference times the CPU oracle (oracle/) on a bounded crop of the same workload, rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOP_PER_EVAL = 70.0   # algorithmic FP32 work of one (pixel, plane, view) cost evaluation
N_STAGED = 32          # distinct frame sets resident on the device (the C5 stream length)
METRIC = "plane-sweep cost evals/sec (pixel x plane x view)"
# dram__bytes_read.sum + dram__bytes_write.sum and issue-slot utilisation of one sweep launch, from the committed ncu
# captures (profiles/), each with the hash of the kernel source it was taken on (kernel_source_hash()): a figure whose
# hash no longer matches paper_1809_06132_b200/csrc/fsw_sweep.cuh is reported as null, not as a stale number
NCU_CAPTURES = {
    ("C5", 8): {"kernel_hash": "dd1a26c10355", "dram_bytes": 155.2e6, "issue_active_pct": 68.6, "fma_pipe_pct": 36.2,
                "alu_pipe_pct": 36.8, "source": "profiles/r2_sweep_kernel.md (ncu --set full of one 8-set sweep launch)"},
    ("C3", 8): {"kernel_hash": "dd1a26c10355", "dram_bytes": 154.0e6, "issue_active_pct": 67.7, "fma_pipe_pct": 35.3,
                "alu_pipe_pct": 36.6, "source": "profiles/r2_sweep_kernel.md (ncu --set full of one 8-set sweep launch)"},
    ("P", 8): {"kernel_hash": "dd1a26c10355", "dram_bytes": 84.7e6, "issue_active_pct": 66.6, "fma_pipe_pct": 35.3,
               "alu_pipe_pct": 38.0, "source": "profiles/r2_sweep_kernel.md (ncu --set full of one 8-set sweep launch)"},
}


def kernel_source_hash():
    import hashlib
    with open(os.path.join(ROOT, "paper_1809_06132_b200", "csrc", "fsw_sweep.cuh"), "rb") as fh:
        return hashlib.sha256(fh.read()).hexdigest()[:12]


def ncu_capture(workload, batch):
    """the committed capture of this workload's sweep launch; a launch of another size than the captured one (20 steps
    run as 7 + 7 + 6) gets the captured DRAM traffic scaled by the number of frame sets -- the traffic is the images in
    and the maps out of every frame set -- and says so in its source"""
    cap = NCU_CAPTURES.get((workload, batch))
    if cap is None:
        for (w, b), c in NCU_CAPTURES.items():
            if w == workload:
                cap = dict(c, dram_bytes=c["dram_bytes"] * batch / b,
                           source=c["source"] + "; captured with %d frame sets per launch, traffic scaled to %d" % (b, batch))
                break
    if cap is None or cap["kernel_hash"] != kernel_source_hash():
        return None
    return cap


def batch_sizes(steps, batch):
    """`steps` frame sets in ceil(steps / batch) launches of nearly equal size (20 steps, batch 8 -> 7 + 7 + 6): an
    under-filled last launch would leave the persistent grid unbalanced."""
    n_calls = max(1, -(-steps // batch))
    base, extra = divmod(steps, n_calls)
    return [base + (1 if i < extra else 0) for i in range(n_calls)]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=128)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--workload", default="C5", choices=["C5", "C3", "P", "P3", "PH", "PM"])
    ap.add_argument("--batch", type=int, default=8,
                    help="frame sets per sweep launch (fsw_compute_depth_batch); 1 = one launch per frame set")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-baseline-seconds", type=float, default=10.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload_config(name):
    import synth
    if name == "P3":   # the three-camera configuration of PAPER.md:280, :294
        return synth.make_config(6, cameras=(0, 1, 2))
    cfg = synth.make_config({"C5": 5, "C3": 3, "P": 6, "PH": 8, "PM": 7}[name])
    if name == "C3":  # the C3 scene, but as a stream of N_STAGED frame sets like C5 so that inputs exceed L2
        cfg = dict(cfg, n_frames=N_STAGED, step_m=0.5, mask_seed=None)
    return cfg


def workload_label(name):
    if name == "P":
        return ("paper workload shape (PAPER.md:224,249; SURVEY 8(f) 2): 5 fisheye cams (4 matching views, rotated) "
                "1024x544 u8, 64 fronto + 30 ground planes, 9x9 ZNCC, filters")
    if name == "P3":
        return ("paper workload shape, three-camera configuration (PAPER.md:280,294): 3 fisheye cams (2 matching views, "
                "rotated) 1024x544 u8, 64 fronto + 30 ground planes, 9x9 ZNCC, filters")
    if name == "PH":
        return ("paper workload shape at half resolution (PAPER.md:249): 5 fisheye cams 512x272 u8, 64 fronto + 30 ground "
                "planes, 7x7 ZNCC, filters")
    if name == "PM":
        return ("paper workload shape, multi-scale (PAPER.md:88-90,249): 5 fisheye cams 1024x544 u8; 512x272 full field of "
                "view 7x7 + 572x332 centre crop 9x9, 64 fronto + 30 ground planes in both passes, filters")
    return ("BASELINE.json configs[4]: 32-frame stream, 3 fisheye cams 1280x1024 u8, 192 fronto + 64 ground planes, "
            "9x9 ZNCC, filters + masks" if name == "C5" else
            "BASELINE.json configs[2]: 3 fisheye cams 1280x1024 u8, 96 fronto + 32 ground planes, 9x9 ZNCC, filters")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def summary(self):
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ---------------------------------------------------------------------------------------------------------------------
def cropped_rig(cfg, crop_w, crop_h):
    """The workload's rig restricted to a centred crop_w x crop_h window of every camera (principal point shifted):
    a bounded sample of the same workload for the CPU legs."""
    cams = []
    W, H = cfg["cams"][0]["width"], cfg["cams"][0]["height"]
    x0, y0 = (W - crop_w) // 2, (H - crop_h) // 2
    for c in cfg["cams"]:
        c2 = dict(c)
        c2.update(width=crop_w, height=crop_h, cx=c["cx"] - x0, cy=c["cy"] - y0)
        cams.append(c2)
    return cams, (x0, y0)


def is_multires(cfg):
    return "families_low" in cfg


def oracle_sample(cfg, frame_images, mask, crop_w, crop_h, keep=False):
    """Runs the oracle as it stands on a centred crop_w x crop_h window of the frame set (the whole frame set when the
    window is the image); returns (seconds, n_eval, maps)."""
    import oracle
    cams, (x0, y0) = cropped_rig(cfg, crop_w, crop_h)
    imgs = [np.ascontiguousarray(im[y0:y0 + crop_h, x0:x0 + crop_w]) for im in frame_images]
    m = None if mask is None else np.ascontiguousarray(mask[y0:y0 + crop_h, x0:x0 + crop_w])
    t0 = time.perf_counter()
    if is_multires(cfg):
        pl = dict(cfg["params_low"], horizon_row=cfg["params_low"]["horizon_row"] - y0)
        pc = dict(cfg["params_crop"], horizon_row=cfg["params_crop"]["horizon_row"] - y0)
        cx0, cy0, cw, ch = cfg["crop"]   # the crop of the multi-scale pass, clipped to the sampled window
        ax0, ay0 = max(cx0 - x0, 0), max(cy0 - y0, 0)
        ax1, ay1 = min(cx0 + cw - x0, crop_w), min(cy0 + ch - y0, crop_h)
        out = oracle.compute_depth_multires(cams, cfg["ref_index"], cfg["families_low"], cfg["families_crop"], pl, pc,
                                            (ax0, ay0, ax1 - ax0, ay1 - ay0), imgs, m, keep_cost=keep)
    else:
        params = dict(cfg["params"], horizon_row=cfg["params"]["horizon_row"] - y0)
        out = oracle.compute_depth(cams, cfg["ref_index"], cfg["families"], params, imgs, m, keep_cost=keep)
    return time.perf_counter() - t0, int(out["n_eval"]), out


def run_reference(args, rank):
    """--impl reference: the oracle, unmodified, on the host cores; each step = one cropped frame set."""
    if rank != 0:
        return
    import oracle
    import synth
    cfg = workload_config(args.workload)
    oracle.build()
    total_steps = args.steps + args.warmup
    # size the crop so that the whole run stays within a few minutes (oracle ~ 1e7 evals/s per 8 cores)
    budget_s = 150.0
    planes_views = sum(f["n_planes"] for f in cfg.get("families", cfg.get("families_crop"))) * (len(cfg["cams"]) - 1)
    est_rate = 1.2e6 * max(oracle.num_threads(), 1)
    px = max(48 * 36, int(budget_s / max(total_steps, 1) * est_rate / planes_views))
    crop_h = int(min(640, max(36, (px / (4.0 / 3.0)) ** 0.5))) // 4 * 4
    crop_w = int(min(848, crop_h * 4 // 3)) // 4 * 4
    frames = {}
    times, evals = [], []
    for s in range(total_steps):
        f = s % N_STAGED
        if f not in frames:
            frames[f] = synth.render_frame(cfg, f)
        mask = None if cfg.get("mask_seed") is None else synth.make_mask(cfg["cams"][0]["width"], cfg["cams"][0]["height"], cfg["mask_seed"] + f)
        dt, ne, _ = oracle_sample(cfg, frames[f], mask, crop_w, crop_h)
        if s >= args.warmup:
            times.append(dt)
            evals.append(ne)
    total = float(sum(times))
    value = float(sum(evals)) / total if total > 0 else 0.0
    sample = "centred %dx%d crop of each frame set (principal point shifted), all planes and views" % (crop_w, crop_h)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "evals/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / max(len(times), 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(args.workload), "sample": sample},
        "cpu_baseline": {"value": value, "unit": "evals/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
def run_ours(args, rank, local_rank, world):
    import torch
    import synth
    import paper_1809_06132_b200 as fsw

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    cfg = workload_config(args.workload)
    W, H = cfg["cams"][0]["width"], cfg["cams"][0]["height"]

    # ---- inputs: N_STAGED distinct frame sets per rank, resident on the device (and pinned on the host for e2e) ----
    from paper_1809_06132_b200 import shard
    host_frames, host_masks = [], []
    for f in shard.frames_for_rank(0, N_STAGED, rank, world):
        host_frames.append(synth.render_frame(cfg, f))
        if cfg.get("mask_seed") is not None:
            host_masks.append(synth.make_mask(W, H, cfg["mask_seed"] + f))
    dev_frames = [[torch.from_numpy(im).to(dev) for im in fr] for fr in host_frames]
    dev_masks = [torch.from_numpy(m).to(dev) for m in host_masks] or [None] * N_STAGED
    rig = fsw.Rig(cfg["cams"], cfg["ref_index"])
    multires = is_multires(cfg)
    if multires:
        planes_low, planes = fsw.PlaneSet(cfg["families_low"]), fsw.PlaneSet(cfg["families_crop"])
        n_nominal = (W // 2) * (H // 2) * planes_low.n_planes * (rig.n_cams - 1) + \
            cfg["crop"][2] * cfg["crop"][3] * planes.n_planes * (rig.n_cams - 1)
    else:
        planes = fsw.PlaneSet(cfg["families"])
        n_nominal = W * H * planes.n_planes * (rig.n_cams - 1)
    ctx = fsw.Context(rig, local_rank)
    # every frame set gets its own output maps so that the bytes touched per pass exceed the 126 MB L2
    outs = [dict(depth=torch.empty((H, W), dtype=torch.float32, device=dev),
                 best_cost=torch.empty((H, W), dtype=torch.float32, device=dev),
                 second_cost=torch.empty((H, W), dtype=torch.float32, device=dev),
                 plane_index=torch.empty((H, W), dtype=torch.int16, device=dev),
                 valid_reason=torch.empty((H, W), dtype=torch.uint8, device=dev)) for _ in range(N_STAGED)]

    B = max(1, min(args.batch, N_STAGED))

    def call_one(c, images, mask, out, host=False):
        """one frame set per call: fsw_compute_depth(_host) or fsw_compute_depth_multires(_host)"""
        if multires:
            return c.compute_depth_multires(planes_low, planes, cfg["params_low"], cfg["params_crop"], cfg["crop"], images,
                                            mask, host=host, out=out)
        return c.compute_depth(planes, cfg["params"], images, mask, host=host, out=out)

    def call_batch(c, image_sets, masks, outs_, host=False, want=fsw.Context.ALL):
        """several frame sets per call: fsw_compute_depth_batch(_host) or fsw_compute_depth_multires_batch(_host)"""
        if multires:
            return c.compute_depth_multires_batch(planes_low, planes, cfg["params_low"], cfg["params_crop"], cfg["crop"],
                                                  image_sets, masks, want=want, host=host, outs=outs_)
        return c.compute_depth_batch(planes, cfg["params"], image_sets, masks, want=want, host=host, outs=outs_)

    def step(i):
        f = i % N_STAGED
        call_one(ctx, dev_frames[f], dev_masks[f], outs[f])

    def run_steps(first, n, host=False):
        """steps first .. first+n-1 in launches of nearly equal size, at most B consecutive frame sets each (the stream
        is processed in order).  host: through the *_host calls, alternating between two contexts on two streams
        (fsw_context_set_host_async) so that the copies of one batch overlap the sweep of the other; every batch still
        does its own host-to-device copies, kernels and device-to-host copy of the depth maps, in that order, on its
        stream."""
        i = first
        for call, nb in enumerate(batch_sizes(n, B)):
            fs = [(i + j) % N_STAGED for j in range(nb)]
            if host:
                lane = call % 2
                with torch.cuda.stream(e2e_streams[lane]):
                    if nb == 1:
                        call_one(e2e_ctx[lane], pin_frames[fs[0]], pin_masks[fs[0]], pin_outs[lane][0], host=True)
                    else:
                        call_batch(e2e_ctx[lane], [pin_frames[f] for f in fs], [pin_masks[f] for f in fs],
                                   pin_outs[lane][:nb], host=True, want=("depth",))
            elif nb == 1:
                step(i)
            else:
                call_batch(ctx, [dev_frames[f] for f in fs], [dev_masks[f] for f in fs], [outs[f] for f in fs])
            i += nb

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------------------------------
    run_steps(0, args.warmup)
    # one untimed call of every launch size the timed loop will use: the context sizes its scratch (footprint images,
    # set table) on first use, and an allocation inside the timed region would synchronize the device
    for nb in sorted(set(batch_sizes(args.steps, B))):
        run_steps(0, nb)
    torch.cuda.synchronize()
    n_eval_step = []
    launches = 0
    for f in range(min(N_STAGED, args.steps)):   # per-frame N_eval from the kernel's counter (untimed pass)
        step(f)
        c = ctx.last_counters()
        n_eval_step.append(c["n_eval"])
    sampler = ClockSampler(physical_gpu_index(local_rank))
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record(stream)
    run_steps(0, args.steps)
    ev1.record(stream)
    torch.cuda.synchronize()
    sampler.stop_flag = True
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches_per_step = ctx.last_counters()["n_launches"]  # kernels of one call of the timed loop
    sizes = batch_sizes(args.steps, B)                      # frame sets per call of the timed loop
    n_calls = len(sizes)
    Bt = sizes[0]
    launches = launches_per_step * n_calls
    evals_total = float(sum(n_eval_step[i % len(n_eval_step)] for i in range(args.steps)))

    # ---- the sweep kernel alone: CUDA events around its launches on the same stream (fsw_context_set_timing) ------
    ctx.set_timing(True)
    sweep_ms, sweep_evals = [], []
    for i in range(0, max(Bt, min(args.steps, 2 * N_STAGED) // Bt * Bt), Bt):   # launches of the size the timed loop used
        run_steps(i, Bt)
        sweep_ms.append(ctx.last_counters()["sweep_ms"])
        sweep_evals.append(sum(n_eval_step[(i + j) % len(n_eval_step)] for j in range(Bt)))
    ctx.set_timing(False)
    sweep_ms_avg = float(np.mean(sweep_ms))
    evals_per_launch = float(np.mean(sweep_evals))
    # latency of a single frame set (one launch per frame set), for context
    torch.cuda.synchronize()
    ev0.record(stream)
    for i in range(8):
        step(i)
    ev1.record(stream)
    torch.cuda.synchronize()
    ms_single = ev0.elapsed_time(ev1) / 8

    # ---- end to end: host buffers through fsw_compute_depth_host ---------------------------------------------------
    pin_frames = [[torch.from_numpy(im).pin_memory() for im in fr] for fr in host_frames]
    pin_masks = [torch.from_numpy(m).pin_memory() for m in host_masks] or [None] * N_STAGED
    pin_outs = [[dict(depth=torch.empty((H, W), dtype=torch.float32).pin_memory()) for _ in range(B)] for _ in range(2)]
    h2d = sum(int(t.numel() * t.element_size()) for t in pin_frames[0]) + (W * H if host_masks else 0)
    d2h = W * H * 4
    # two contexts (each owns its staging buffers) on two streams; the host calls return without synchronizing
    e2e_ctx = [fsw.Context(rig, local_rank), fsw.Context(rig, local_rank)]
    e2e_streams = [torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)]
    for c in e2e_ctx:
        c.set_host_async(True)

    run_steps(0, min(4 * B, N_STAGED), host=True)
    e2e_steps = args.steps
    barrier()
    ev0.record(stream)
    for st in e2e_streams:
        st.wait_event(ev0)
    run_steps(0, e2e_steps, host=True)
    for st in e2e_streams:
        done = torch.cuda.Event()
        done.record(st)
        stream.wait_event(done)
    ev1.record(stream)
    torch.cuda.synchronize()
    barrier()
    ms_e2e = ev0.elapsed_time(ev1)
    launches += launches_per_step * n_calls

    # ---- max over ranks ----------------------------------------------------------------------------------------------
    (ms_total, ms_e2e), (evals_all,) = shard.reduce_timing([ms_total, ms_e2e], [evals_total], dev)

    if rank == 0:
        from paper_1809_06132_b200.probe import measure_fp32_peak
        fp32_tflops, _ = measure_fp32_peak(local_rank)
        value = evals_all / (ms_total * 1e-3)
        e2e_value = evals_all / (ms_e2e * 1e-3)
        achieved = evals_per_launch * FLOP_PER_EVAL / (sweep_ms_avg * 1e-3) / 1e12
        cap = ncu_capture(args.workload, Bt)
        n_cam_bytes = sum(int(t.numel() * t.element_size()) for t in dev_frames[0])
        line = {
            "metric": METRIC, "value": value, "unit": "evals/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args.workload), "frames_staged_per_gpu": N_STAGED,
                       "n_eval_per_step": evals_total / args.steps, "n_nominal_per_step": n_nominal,
                       "l2": "inputs, footprint images and outputs rotate over %d distinct frame sets (%.0f MB per pass) "
                             "> 126 MB L2" % (N_STAGED, N_STAGED * (n_cam_bytes * 9 + W * H + W * H * 15) / 1e6),
                       "frame_sets_per_launch": sizes, "ms_single_frame_set_launch": ms_single,
                       "parallelism": "frame sets sharded over %d GPU(s), no collective" % world},
            "depth_maps_per_s": world * args.steps / (ms_total * 1e-3),
            # what a real-time pipeline sees: one frame set per call (25 frame sets per second arrive)
            "single_frame_set": {"ms_per_map": ms_single, "depth_maps_per_s": 1e3 / ms_single,
                                 "evals_per_s": evals_total / args.steps / (ms_single * 1e-3)},
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_value, "unit": "evals/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e / e2e_steps, "depth_maps_per_s": world * e2e_steps / (ms_e2e * 1e-3),
                    "how": "fsw_compute_depth_%sbatch_host on pinned host buffers: every batch copies its images and masks "
                           "to the device, runs the kernels and copies its depth maps back, on one of two streams "
                           "(two contexts, fsw_context_set_host_async) so that copies overlap the other batch's sweep"
                           % ("multires_" if multires else "")},
            "gpu_launches": launches,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": fp32_tflops, "unit": "TFLOP/s",
                         "frac": achieved / fp32_tflops if fp32_tflops else None,
                         "traffic": cap["dram_bytes"] if cap else None,
                         "traffic_source": cap["source"] if cap else None,
                         "ncu_issue_active_pct": cap["issue_active_pct"] if cap else None,
                         "ncu_fma_pipe_pct": cap["fma_pipe_pct"] if cap else None,
                         "ncu_alu_pipe_pct": cap["alu_pipe_pct"] if cap else None,
                         "kernel_source_hash": kernel_source_hash(),
                         "frame_sets_per_launch": Bt, "evals_per_launch": evals_per_launch,
                         "kernel": "fsw::sweep_kernel<%d,...>%s" % (
                             cfg.get("params", cfg.get("params_crop"))["window"],
                             " (both sweeps of the multi-scale call)" if multires else ""),
                         "kernel_ms": sweep_ms_avg,
                         "flop_per_eval": FLOP_PER_EVAL,
                         "peak_source": "FFMA-chain kernel measured in this run (MEASURED_PEAKS.json has no FP32 figure); "
                                        "nominal 148 SM x 128 lanes x 2 x clock"},
        }
        if not args.no_cpu_baseline:
            step(0)
            torch.cuda.synchronize()
            gpu0 = {k: v.cpu().numpy() for k, v in outs[0].items()}
            line["cpu_baseline"], line["parity"] = cpu_baseline(cfg, host_frames, host_masks, args.cpu_baseline_seconds, gpu0)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def cpu_baseline(cfg, frames, masks, seconds, gpu_maps0=None):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the workload: whole frame sets
    of the stream (every plane and view), one after the other, until `seconds` of CPU work are done (at most 6).
    The oracle's maps of frame set 0 are also held against the GPU's (oracle/compare.py): the parity statistics of
    this very run go into the bench line."""
    import oracle
    from oracle.compare import compare_maps, depth_conditioning
    oracle.build()
    cores = oracle.num_threads()
    W, H = cfg["cams"][0]["width"], cfg["cams"][0]["height"]
    total_t, total_e, n = 0.0, 0, 0
    parity = None
    while n < min(6, len(frames)) and total_t < seconds:
        dt, ne, maps = oracle_sample(cfg, frames[n], masks[n] if masks else None, W, H, keep=(n == 0 and gpu_maps0 is not None))
        if n == 0 and gpu_maps0 is not None:
            if is_multires(cfg):
                st = compare_maps(maps, gpu_maps0, (maps["cost_lo"], maps["cost_hi"]))
            else:
                cond = depth_conditioning(maps, oracle.plane_table(cfg["families"])[0])
                st = compare_maps(maps, gpu_maps0, maps["cost"], depth_cond=cond)
            keys = ("index_exact_frac", "index_match_frac", "max_dc1", "max_dc2", "frac_ddepth_over_tol",
                    "depth_worst_ratio_to_bound", "fragile_frac", "valid_mismatch_nonfragile", "n_oracle_valid")
            parity = {k: st[k] for k in keys}
            parity["frame_set"] = 0
            maps = None
        total_t += dt
        total_e += ne
        n += 1
    base = {"value": total_e / total_t, "unit": "evals/s", "cores": cores, "kind": "oracle", "seconds": total_t,
            "sample": "frame sets 0..%d of the workload at full size (%dx%d), all planes and views" % (n - 1, W, H)}
    return base, parity


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
