"""Times the hot path on every BASELINE.json config (C1..C5) and on the paper's own workload shape (config 6).

    python -m paper_1809_06132_b200.time_configs [--reps 20]

Prints one markdown table row per config: milliseconds per depth map (CUDA events on the launching stream, device
resident inputs, 3 warm-up calls), finite cost evaluations per map (the kernel's counter) and evaluations per second.
C1..C4 and 6 are single calls (one frame set per launch: the latency figure); C5 and the last row of 6 run 8 frame sets
per launch like bench.py.  Config 6 is also timed on the two three-camera subsets of PAPER.md:280 (fig:camconfiguration:
"3 Cameras (C1)" = leftmost, central, rightmost; "3 Cameras (C2)" = the three central cameras; the paper reports that
they "save about 17% of run time"): a subset is simply a rig built from those cameras.
Inputs come from the seeded generator `synth` (no files are read)."""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch
    import synth
    import paper_1809_06132_b200 as fsw

    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=20)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("time_configs needs a CUDA device: the hot path has no CPU fallback")
    stream = torch.cuda.current_stream()

    def timed(fn, reps):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    print("| config | call | ms per depth map | finite cost evaluations per map | evaluations / s |")
    print("|---|---|---|---|---|")
    # (config index, camera subset or None, label suffix); the rig of config 6 is (reference = central, outer left,
    # outer right, inner left, inner right)
    runs = [(i, None, "") for i in (1, 2, 3, 4, 5, 6)] + [(6, (0, 1, 2), " 3 cameras (C1)"), (6, (0, 3, 4), " 3 cameras (C2)")]
    for idx, subset, suffix in runs:
        cfg = synth.make_config(idx)
        if subset is not None:
            cfg = dict(cfg, cams=[cfg["cams"][i] for i in subset], name=cfg["name"] + suffix)
        rig = fsw.Rig(cfg["cams"], cfg["ref_index"])
        ctx = fsw.Context(rig, 0)
        W, H = cfg["cams"][0]["width"], cfg["cams"][0]["height"]
        n_frames = 8 if idx >= 5 else 1
        frames = [[torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, f)] for f in range(n_frames)]
        if subset is not None:
            rows_filter = lambda rows: rows[-1:]  # the batched row only
        else:
            rows_filter = lambda rows: rows
        if idx == 4:
            pl, pc = fsw.PlaneSet(cfg["families_low"]), fsw.PlaneSet(cfg["families_crop"])
            mask = torch.from_numpy(synth.make_mask(W, H, cfg["mask_seed"])).cuda()
            fn = lambda: ctx.compute_depth_multires(pl, pc, cfg["params_low"], cfg["params_crop"], cfg["crop"], frames[0], mask)
            rows = [("fsw_compute_depth_multires", fn, 1)]
        else:
            planes = fsw.PlaneSet(cfg["families"])
            masks = [None] * n_frames
            if cfg.get("mask_seed") is not None:
                masks = [torch.from_numpy(synth.make_mask(W, H, cfg["mask_seed"] + f)).cuda() for f in range(n_frames)]
            rows = [("fsw_compute_depth", lambda: ctx.compute_depth(planes, cfg["params"], frames[0], masks[0]), 1)]
            if n_frames > 1:
                rows.append(("fsw_compute_depth_batch, 8 frame sets",
                             lambda: ctx.compute_depth_batch(planes, cfg["params"], frames, masks), n_frames))
        for label, fn, n in rows_filter(rows):
            ms = timed(fn, args.reps) / n
            n_eval = ctx.last_counters()["n_eval"] / n
            print("| %s %dx%d | %s | %.4f | %.4g | %.3g |" % (cfg["name"], W, H, label, ms, n_eval, n_eval / (ms * 1e-3)))
        ctx.close()


if __name__ == "__main__":
    main()
