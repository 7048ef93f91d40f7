#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (the 5 C-ABI calls of include/mg.h) over one
synthetic frame.  Prints ONE JSON line (see the contract in DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

value = Gaussian-pixel blends per second (forward + backward blends of the frame, exact counts from
oracle/work_counts.json, divided by the device time of a whole step), inputs resident in HBM.
e2e    = the same with host buffers: pinned-host -> device copies of every input and device -> host reads
         of the image and all gradients inside the timed region.
roofline = the dominant kernel (largest share of the step), FP32-ALU bound, against the FP32 peak measured on this
         chip by mg_measure_fp32_peak (the figure derived from the unit counts is printed beside it); `rooflines` has
         one entry per C-ABI call (HBM-bound calls against MEASURED_PEAKS.json's copy bandwidth).
cpu_baseline / --impl reference = the oracle, as it stands, on the host cores, on a bounded sample of tiles.
N > 1: one process per GPU (torchrun), replicas only -- no collective on the data path.
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

# Algorithmic work per unit -- the ONE place these constants live (counted once from the oracle's
# O10/O11 arithmetic).  Work the method does not require is not charged: under reading 5 the forward pass never looks
# at an entry with M = 0, and the backward pass owes such an entry dL/dM only.
FLOP_PAIR = 13             # per pair evaluation: 2 sub, 6 quadratic form, mul, min, 2 compares (+1 MUFU not counted)
FLOP_BLEND_FWD = 11        # per unmasked blend, forward: M alpha, T' (fma), compare, a T, 3 fma
FLOP_BLEND_BWD = 59        # per unmasked blend, backward (49 + 10 adds of the per-entry reduction)
FLOP_BLEND_BWD_MASKED = 12  # per masked blend, backward: g.c (5), g.c - g.b, T x, alpha X accumulate (2), its reduction add, 2 compares
BYTES_PRE = (301, 109)     # mg_preprocess, per visible / per culled Gaussian
BYTES_PRE_BWD = (513, 240)  # mg_preprocess_bwd, per visible / per culled Gaussian
BYTES_SORT_KEY = 22        # mg_bin_sort, per duplicated key, this scheme; the floor of any scheme is 4
# dram__bytes_read.sum + dram__bytes_write.sum per launch, summed over the kernels of each call: written by
# `python ncu_summary.py` from the `ncu --set full` capture named in profiles/r03_final.md (section 3)
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r03_traffic.json")
# kernels of libmg launched per step (memsets and copies not counted), see binsort.cu for the sort's list
KERNELS_PER_STEP = {"preprocess": 1, "bin_sort": 2 + 4 + 5 + 6, "render_fwd": 1, "render_bwd": 1,
                    "preprocess_bwd": 2}


def ncu_traffic(cfg):
    """{call: bytes per launch} for this config from the tracked ncu summary, or {} if there is none."""
    if not os.path.exists(TRAFFIC_JSON):
        return {}
    return json.load(open(TRAFFIC_JSON)).get(str(cfg), {})


def algorithmic_work(wc, N):
    """Per call: (bound, work per launch, unit).  Flops for the blend kernels, bytes for the HBM-bound calls."""
    vis, cul = wc["visible"], N - wc["visible"]
    fwd_flop = ((wc["fwd_pair_evals"] - wc["fwd_pair_evals_masked"]) * FLOP_PAIR
                + (wc["fwd_blends"] - wc["fwd_blends_masked"]) * FLOP_BLEND_FWD)
    bwd_flop = (wc["bwd_pair_evals"] * FLOP_PAIR + (wc["bwd_blends"] - wc["bwd_blends_masked"]) * FLOP_BLEND_BWD
                + wc["bwd_blends_masked"] * FLOP_BLEND_BWD_MASKED)
    return {"preprocess": ("hbm", vis * BYTES_PRE[0] + cul * BYTES_PRE[1]),
            "bin_sort": ("hbm", wc["R"] * BYTES_SORT_KEY),
            "render_fwd": ("alu", fwd_flop), "render_bwd": ("alu", bwd_flop),
            "preprocess_bwd": ("hbm", vis * BYTES_PRE_BWD[0] + cul * BYTES_PRE_BWD[1])}


def work_counts(cfg):
    p = os.path.join(ROOT, "oracle", "work_counts.json")
    data = json.load(open(p)) if os.path.exists(p) else {}
    return data.get(str(cfg))


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def mark(self, timeout=5.0):
        """Wait until nvidia-smi has started emitting, then remember where the timed region begins."""
        t0 = time.time()
        while self.proc is not None and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.02)
        self.first = len(self.rows)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        rows = self.rows[getattr(self, "first", 0):] or self.rows[-1:]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(cfg, n_tiles_target=None, seed=0):
    """Time the oracle on a bounded sample of the workload: every k-th tile.  Returns (blends, seconds, info)."""
    import oracle as orc
    from paper_2412_20522_b200 import scenes

    sc = scenes.make(cfg)
    cam = sc.camera
    gw, gh = orc.grid(cam)
    ntiles = gw * gh
    if n_tiles_target is None:
        n_tiles_target = ntiles if ntiles <= 5000 else ntiles // 2  # config 3: the whole frame, ~10-20 s of CPU work
    stride = max(1, ntiles // n_tiles_target)
    sel = np.zeros(ntiles, np.uint8)
    sel[seed % stride::stride] = 1
    frac = float(sel.sum()) / ntiles
    arrs = (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)
    g = sc.dL_dimage().astype(np.float64)
    t0 = time.perf_counter()
    pre = orc.preprocess(cam, *arrs)
    t1 = time.perf_counter()
    ids, ranges = orc.bin_sort(cam, pre["depths"].astype(np.float32), pre["rects"], pre["tiles_touched"], sel)
    t2 = time.perf_counter()
    fwd = orc.render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks)
    t3 = time.perf_counter()
    rb = orc.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, g)
    t4 = time.perf_counter()
    orc.preprocess_bwd(cam, *arrs, rb["dL_dmeans2d"], rb["dL_dconic"], rb["dL_dopacity"], rb["dL_drgb"])
    t5 = time.perf_counter()
    blends = fwd["blends"] + rb["blends"]
    # per-Gaussian steps run on the whole scene; charge the sample its share of them
    seconds = (t3 - t2) + (t4 - t3) + (t2 - t1) + frac * ((t1 - t0) + (t5 - t4))
    which = "the whole frame" if stride == 1 else f"every {stride}th tile"
    info = (f"{int(sel.sum())} of {ntiles} tiles ({which}) of config {cfg}: oracle bin_sort+render_fwd+render_bwd "
            f"on those tiles ({t2 - t1:.1f}+{t3 - t2:.1f}+{t4 - t3:.1f} s) + {frac:.4f} x (preprocess {t1 - t0:.1f} s + "
            f"preprocess_bwd {t5 - t4:.1f} s)")
    return blends, seconds, info


def max_over_ranks(value, world, device):
    """MAX over ranks of a per-rank scalar (the contract's multi-GPU timing rule).  nccl on cuda, gloo on cpu."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def bench_mask_head(sc, g, hbm_gbs, reps=20):
    """SURVEY.md 8(f) row f1, measured like the hot path (CUDA events, warm, inputs resident): the mask head at the
    bench workload's N.  Algorithmic bytes per Gaussian: sample 24 (2 scores + 2 uniforms in, mask + soft out),
    loss 12, backward 16, prune rule 89 (10 draws), compaction 4 x 61 floats in + the kept rows out."""
    import torch

    from paper_2412_20522_b200 import binding as mg
    from paper_2412_20522_b200 import scenes

    n = sc.N
    scores_np, u_np, u10_np, gm_np = scenes.mask_head_inputs(n)
    t = lambda a: torch.from_numpy(a).cuda()
    scores, u, u10, dmask = t(scores_np), t(u_np), t(u10_np), t(gm_np)
    masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    dscores = torch.empty(n, 2, device="cuda")
    stats = torch.zeros(3, dtype=torch.float64, device="cuda")
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    src = [g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], scores]
    dst = [torch.empty_like(x) for x in src]
    ws = torch.empty(mg.mg_compact_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64).pin_memory()
    calls = {
        "mask_sample": lambda: mg.mg_mask_sample(scores, u, 1.0, masks, soft),
        "mask_loss": lambda: mg.mg_mask_loss(masks, 0.1, dmask, stats),
        "mask_sample_bwd": lambda: mg.mg_mask_sample_bwd(soft, dmask, 1.0, dscores),
        "mask_prune_keep": lambda: mg.mg_mask_prune_keep(scores, u10, keep),
        "compact": lambda: mg.mg_compact(keep, src, dst, ws, n_out),
    }
    out = {}
    for name, fn in calls.items():
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out[name] = e0.elapsed_time(e1) / reps
    kept = int(n_out[0])
    row = sum(x.numel() // n for x in src) * 4
    nbytes = {"mask_sample": 24 * n, "mask_loss": 12 * n, "mask_sample_bwd": 16 * n, "mask_prune_keep": 89 * n,
              "compact": n * (row + 1 + 4) + kept * row}
    return {"N": n, "kept_by_prune_rule": kept,
            "ms": {k: round(v, 4) for k, v in out.items()},
            "gb_per_s": {k: round(nbytes[k] / (out[k] * 1e-3) / 1e9, 1) for k in out},
            "frac_of_hbm_peak": {k: round(nbytes[k] / (out[k] * 1e-3) / 1e9 / hbm_gbs, 3) for k in out},
            "peak_gb_per_s": hbm_gbs}


def bench_inference(sc, g, m, reps=30):
    """forward-only rendering (preprocess + bin_sort + render_fwd, every mask = 1), the setting
    of the paper's FPS numbers (one RTX 4090, real captures) -- on the bench scene with all
    Gaussians, and on the survivors after compacting away the Gaussians the scene's masks switch off."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    def fps(gd, n):
        fr = mg.Frame(sc.camera, n)
        ones = torch.ones(n, device="cuda")
        fr.forward(gd, ones)
        torch.cuda.synchronize()

        def once():
            fr.preprocess(gd); fr.bin_sort(); fr.render_fwd(ones)
        for _ in range(3):
            once()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            once()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        return {"N": n, "R": fr.R, "ms_per_frame": round(ms, 4), "fps": round(1e3 / ms, 1)}

    out = {"all_gaussians": fps(g, sc.N)}
    keep = (m != 0).to(torch.uint8)
    names = ["means", "log_scales", "quats", "opacity_logits", "sh"]
    src = [g[k] for k in names]
    dst = [torch.empty_like(t) for t in src]
    ws = torch.empty(mg.mg_compact_workspace_bytes(sc.N), dtype=torch.uint8, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64).pin_memory()
    mg.mg_compact(keep, src, dst, ws, n_out)
    torch.cuda.synchronize()
    nk = int(n_out[0])
    out["compacted_survivors"] = fps({k: t[:nk].contiguous() for k, t in zip(names, dst)}, nk)
    out["paper_context"] = "3DGS 187.8 -> MaskGaussian 384.7 FPS on Mip-NeRF360 (3.2 M -> 1.2 M Gaussians), one RTX 4090, PAPER.md:138-141"
    return out


def bench_cameras(sc, g, m, steps=10):
    """BASELINE.json configs[4]: "Forward+backward are timed over 20 cameras on a circle".  ms per frame (all five
    calls) for every camera of the scene; buffers sized for the largest R."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    fr = mg.Frame(sc.cameras[0], sc.N)
    Rs = []
    for cam in sc.cameras:
        fr.set_camera(cam)
        fr.preprocess(g)
        torch.cuda.current_stream().synchronize()
        Rs.append(int(fr.R_host[0]))
    fr.reserve(max(Rs))
    ms = []
    for ci, cam in enumerate(sc.cameras):
        fr.set_camera(cam)
        gimg = torch.from_numpy(sc.dL_dimage(ci)).cuda()
        for _ in range(2):
            fr.step(g, m, gimg)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            fr.step(g, m, gimg)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1) / steps)
        assert int(fr.R_host[1]) == Rs[ci]
    return {"cameras": len(ms), "ms_per_frame_mean": float(np.mean(ms)), "ms_per_frame_max": float(np.max(ms)),
            "ms_per_frame_min": float(np.min(ms)), "R_min": min(Rs), "R_max": max(Rs)}


def bench_cameras_two_in_flight(sc, g, m, sweeps=3):
    """The cameras of the scene as INDEPENDENT views (BASELINE.json configs[4]: 20 cameras on a circle; also the
    inference setting) with two frames in flight: camera k runs on stream k % 2 with its own Frame, so
    the latency-bound mg_bin_sort and the HBM-bound mg_preprocess of one view run under the issue-bound blend kernels
    of the other.  A throughput figure over independent views -- never the training-iteration number (an iteration's
    calls depend on one another).  Timed against the same sweep on one stream, in the same run; every view of the
    two-stream run is then compared bit for bit (sorted ids, tile ranges, n_contrib, image, final_T) with the
    sequential one."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    cams = sc.cameras
    frs = [mg.Frame(cams[0], sc.N) for _ in range(3)]  # two in flight + one for the sequential sweep
    Rs = []
    for cam in cams:
        frs[0].set_camera(cam)
        frs[0].preprocess(g)
        torch.cuda.current_stream().synchronize()
        Rs.append(int(frs[0].R_host[0]))
    for f in frs:
        f.reserve(max(Rs))
    gimgs = [torch.from_numpy(sc.dL_dimage(ci)).cuda() for ci in range(len(cams))]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()

    def one(fr, ci):
        fr.set_camera(cams[ci])
        fr.step(g, m, gimgs[ci])

    def sweep_seq():
        for ci in range(len(cams)):
            one(frs[2], ci)

    def sweep_two(first=0, last=None):
        for ci in range(first, len(cams) if last is None else last):
            with torch.cuda.stream(streams[ci % 2]):
                one(frs[ci % 2], ci)

    def join():
        cur = torch.cuda.current_stream()
        for st in streams:
            cur.wait_stream(st)

    sweep_seq(); sweep_two(); join()  # warm-up of both forms
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(sweeps):
        sweep_seq()
    e1.record()
    torch.cuda.synchronize()
    ms_seq = e0.elapsed_time(e1) / (sweeps * len(cams))
    e0.record()
    for st in streams:
        st.wait_event(e0)
    for _ in range(sweeps):
        sweep_two()
    join()
    e1.record()
    torch.cuda.synchronize()
    ms_two = e0.elapsed_time(e1) / (sweeps * len(cams))
    # every view, two at a time, against the sequential frame
    same = True
    for ci in range(0, len(cams) - 1, 2):
        sweep_two(ci, ci + 2)
        join()
        torch.cuda.synchronize()
        for k in (0, 1):
            one(frs[2], ci + k)
            torch.cuda.synchronize()
            a, b, R = frs[k], frs[2], Rs[ci + k]
            same = same and int(a.R_host[1]) == R == int(b.R_host[1])
            same = same and torch.equal(a.sorted_ids[:R], b.sorted_ids[:R]) and torch.equal(a.tile_ranges, b.tile_ranges)
            same = same and torch.equal(a.n_contrib, b.n_contrib) and torch.equal(a.image, b.image) and torch.equal(a.final_T, b.final_T)
    assert same, "two frames in flight changed an output"
    del frs
    torch.cuda.empty_cache()
    return {"ms_per_frame_sequential": round(ms_seq, 4), "ms_per_frame_two_in_flight": round(ms_two, 4),
            "gain": round(1.0 - ms_two / ms_seq, 4), "frames_timed_each": sweeps * len(cams),
            "outputs_bit_identical_to_sequential": bool(same),
            "note": "throughput over independent views on two streams; not a training-iteration figure"}


def bench_render_loss(sc, hbm_gbs, reps=30):
    """SURVEY.md 8(f) row f3 at the bench image size.  Algorithmic bytes per image element: 12 (image and target in,
    gradient out); the two-kernel scheme moves 44 (three derivative maps written and read back)."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    cam = sc.camera
    rng = np.random.default_rng(3)
    img = torch.from_numpy(rng.uniform(0, 1, (3, cam.height, cam.width)).astype(np.float32)).cuda()
    tgt = torch.from_numpy(rng.uniform(0, 1, (3, cam.height, cam.width)).astype(np.float32)).cuda()
    grad = torch.empty_like(img)
    stats = torch.zeros(3, dtype=torch.float64, device="cuda")
    ws = torch.empty(mg.mg_render_loss_workspace_bytes(cam.width, cam.height), dtype=torch.uint8, device="cuda")
    fn = lambda: mg.mg_render_loss(img, tgt, 0.2, grad, stats, ws)
    for _ in range(3):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    n = img.numel()
    return {"image": [cam.width, cam.height], "ms": round(ms, 4), "algorithmic_gb_per_s": round(12 * n / (ms * 1e-3) / 1e9, 1),
            "moved_gb_per_s": round(44 * n / (ms * 1e-3) / 1e9, 1), "frac_of_hbm_peak": round(12 * n / (ms * 1e-3) / 1e9 / hbm_gbs, 4),
            "note": "13 MB per plane set: L2-resident, launch- and latency-bound at this size"}


def bench_optimizer(sc, g, fr, hbm_gbs, reps=10):
    """SURVEY.md 8(f) row f4 at the bench workload's N: the statistics after a backward pass and one fused Adam step
    over the 59 floats per Gaussian + 2 mask scores (28 B per parameter float: p, g, m, v in; p, m, v out), dense and
    restricted to the Gaussians visible in the view."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    n = sc.N
    scores = torch.zeros(n, 2, device="cuda")
    params = [g["means"].clone(), g["log_scales"].clone(), g["quats"].clone(), g["opacity_logits"].clone(), g["sh"].clone(), scores]
    grads = [fr.dL_dmeans, fr.dL_dlog_scales, fr.dL_dquats, fr.dL_dopacity_logits, fr.dL_dsh, torch.zeros_like(scores)]
    groups = [(p, gr, torch.zeros_like(p), torch.zeros_like(p), 1e-4) for p, gr in zip(params, grads)]
    acc, den, mxr = (torch.zeros(n, device="cuda") for _ in range(3))
    nfl = sum(p.numel() for p in params)
    vis = int((fr.radii > 0).sum())
    calls = {"adam_step": (lambda: mg.mg_adam_step(groups, 0.9, 0.999, 1e-15, 3), 28 * nfl),
             "adam_step_visible_only": (lambda: mg.mg_adam_step(groups, 0.9, 0.999, 1e-15, 3, fr.radii), 28 * (nfl // n) * vis + 4 * n),
             "density_stats": (lambda: mg.mg_density_stats(fr.dL_dmeans2d, fr.radii, (1.0, 1.0), acc, den, mxr), 4 * n + 32 * vis)}
    out = {"N": n, "visible": vis, "param_floats": nfl, "ms": {}, "gb_per_s": {}, "frac_of_hbm_peak": {}}
    for name, (fn, nbytes) in calls.items():
        for _ in range(2):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        out["ms"][name] = round(ms, 4)
        out["gb_per_s"][name] = round(nbytes / (ms * 1e-3) / 1e9, 1)
        out["frac_of_hbm_peak"][name] = round(nbytes / (ms * 1e-3) / 1e9 / hbm_gbs, 3)
    return out


def bench_training_iteration(sc, g, fr, reps=10):
    """One whole training iteration on the bench workload, the eleven C-ABI calls of DESIGN.md section 11 back to back
    on one stream: mask_sample, preprocess, bin_sort, render_fwd, render_loss, render_bwd, mask_loss, mask_sample_bwd,
    preprocess_bwd, density_stats, adam_step (all 59 floats per Gaussian + the 2 mask scores).  Parameters do change from
    iteration to iteration (lr 1e-5: the scene stays the bench scene to within the noise of a few steps); the uniforms
    are one fixed draw.  The sum of the rows timed one by one is printed beside it for comparison."""
    import torch

    from paper_2412_20522_b200 import binding as mg

    n, cam = sc.N, sc.camera
    gen = torch.Generator(device="cuda")
    gen.manual_seed(7)
    uniforms = torch.rand(n, 2, device="cuda", generator=gen).clamp_(1e-7, 1 - 1e-7)
    scores = torch.zeros(n, 2, device="cuda")
    scores[:, 1] = torch.randn(n, device="cuda", generator=gen)
    names = ("means", "log_scales", "quats", "opacity_logits", "sh")
    params = {k: g[k].clone() for k in names}
    masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    dL_dscores = torch.empty(n, 2, device="cuda")
    fr.forward(params, torch.ones(n, device="cuda"))
    fr.reserve(int(fr.R * 1.1))
    target = fr.image.clone()
    dL_dimage = torch.empty_like(fr.image)
    lstats, mstats = (torch.zeros(3, dtype=torch.float64, device="cuda") for _ in range(2))
    ws = torch.empty(mg.mg_render_loss_workspace_bytes(cam.width, cam.height), dtype=torch.uint8, device="cuda")
    acc, den, mxr = (torch.zeros(n, device="cuda") for _ in range(3))
    grads = dict(means=fr.dL_dmeans, log_scales=fr.dL_dlog_scales, quats=fr.dL_dquats, opacity_logits=fr.dL_dopacity_logits,
                 sh=fr.dL_dsh)
    groups = [(params[k], grads[k], torch.zeros_like(params[k]), torch.zeros_like(params[k]), 1e-5) for k in names]
    groups.append((scores, dL_dscores, torch.zeros_like(scores), torch.zeros_like(scores), 1e-5))
    it = [0]

    def iteration():
        it[0] += 1
        mg.mg_mask_sample(scores, uniforms, 1.0, masks, soft)
        fr.preprocess(params)  # no host sync inside the iteration: the sort buffers keep a 10 % reserve (below)
        fr.bin_sort()
        fr.render_fwd(masks)
        mg.mg_render_loss(fr.image, target, 0.2, dL_dimage, lstats, ws)
        fr.render_bwd(masks, dL_dimage)
        fr.preprocess_bwd(params)
        mg.mg_mask_loss(masks, 5e-4, fr.dL_dmask, mstats)
        mg.mg_mask_sample_bwd(soft, fr.dL_dmask, 1.0, dL_dscores)
        mg.mg_density_stats(fr.dL_dmeans2d, fr.radii, (cam.width / 2, cam.height / 2), acc, den, mxr)
        mg.mg_adam_step(groups, 0.9, 0.999, 1e-15, it[0])

    for _ in range(3):
        iteration()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        iteration()
    e1.record()
    torch.cuda.synchronize()
    assert int(fr.R_host[1]) <= fr.R_capacity, "R outgrew the reserve during the timed iterations"
    return {"ms": round(e0.elapsed_time(e1) / reps, 4), "calls": 11, "iterations_timed": reps,
            "loss_render": float(lstats[2]), "mean_mask": float(mstats[2])}


def n_threads():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count()


def run_reference(args, rank, world):
    if rank != 0:
        return
    import oracle as orc

    orc.lib()
    for _ in range(min(args.warmup, 1)):
        oracle_sample(args.config, n_tiles_target=16)
    tot_b, tot_s, info = 0, 0.0, ""
    steps = min(args.steps, 3)
    for s in range(steps):
        b, sec, info = oracle_sample(args.config, seed=s)
        tot_b += b
        tot_s += sec
    v = tot_b / tot_s
    line = {"impl": "reference", "metric": "gaussian_pixel_blends_per_s", "value": v, "unit": "blends/s",
            "n_gpus": args.gpus, "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * tot_s / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "sample": info},
            "cpu_baseline": {"value": v, "unit": "blends/s", "cores": n_threads(), "kind": "oracle", "sample": info},
            "e2e": {"value": v, "unit": "blends/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_name(cfg):
    return {1: "configs[0] tiny: 1k Gaussians, 128x128, SH0", 2: "configs[1] small: 100k Gaussians, 512x512, SH3",
            3: "configs[2] outdoor: 3M Gaussians, 1297x840, SH3 (north_star target)",
            4: "configs[3] indoor: 2.8M Gaussians, 1264x832, SH3",
            5: "configs[4] stress: 6M Gaussians, 1920x1080, SH3, camera 0"}[cfg]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--all-cameras", action="store_true", help="also time every camera of the scene (config 5: 20)")
    ap.add_argument("--no-config5", action="store_true", help="skip the config 5 (20 cameras) entry of next_rows")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as `python bench.py --gpus N`: become N ranks, one per GPU (replicas)
        import socket

        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port", str(port),
                                  os.path.abspath(__file__)] + sys.argv[1:])
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    from paper_2412_20522_b200 import binding as mg
    from paper_2412_20522_b200 import scenes

    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    mg.lib()
    args.warmup = max(args.warmup, 3)

    sc = scenes.make(args.config)
    cam = sc.camera
    g, m = mg.upload(sc)
    gimg_np = sc.dL_dimage()
    gimg = torch.from_numpy(gimg_np).cuda()
    fr = mg.Frame(cam, sc.N)
    fr.forward(g, m)           # sizes the sort buffers from the exact R (one sync, outside the timed region)
    fr.backward(g, m, gimg)
    torch.cuda.synchronize()
    R = fr.R
    wc = work_counts(args.config)
    if wc is not None:
        assert wc["R"] == R or abs(wc["R"] - R) < 1e-4 * R, (wc["R"], R)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        fr.step(g, m, gimg)
    barrier()
    names = ["preprocess", "bin_sort", "render_fwd", "render_bwd", "preprocess_bwd"]
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(args.steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.mark()
    barrier()
    for s in range(args.steps):
        e = ev[s]
        e[0].record(); fr.preprocess(g)
        e[1].record(); fr.bin_sort()
        e[2].record(); fr.render_fwd(m)
        e[3].record(); fr.render_bwd(m, gimg)
        e[4].record(); fr.preprocess_bwd(g)
        e[5].record()
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = ev[0][0].elapsed_time(ev[-1][5])
    per_call = {n: float(np.mean([ev[s][i].elapsed_time(ev[s][i + 1]) for s in range(args.steps)])) for i, n in enumerate(names)}
    assert int(fr.R_host[1]) == R
    total_ms = max_over_ranks(total_ms, world, "cuda")
    ms_step = total_ms / args.steps

    # ---- e2e: host buffers, H2D of every input + D2H of image and gradients inside the timed region
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    host_in = {k: pin(getattr(sc, k)) for k in ("means", "log_scales", "quats", "opacity_logits", "sh")}
    host_m, host_g = pin(sc.masks), pin(gimg_np)
    out_names = ["image", "dL_dmask", "dL_dmeans", "dL_dlog_scales", "dL_dquats", "dL_dopacity_logits", "dL_dsh"]
    host_out = {k: torch.empty(getattr(fr, k).shape, dtype=torch.float32).pin_memory() for k in out_names}
    h2d = sum(t.numel() * 4 for t in host_in.values()) + host_m.numel() * 4 + host_g.numel() * 4
    d2h = sum(t.numel() * 4 for t in host_out.values())

    def e2e_step():
        for k, t in host_in.items():
            g[k].copy_(t, non_blocking=True)
        m.copy_(host_m, non_blocking=True)
        gimg.copy_(host_g, non_blocking=True)
        fr.step(g, m, gimg)
        for k, t in host_out.items():
            t.copy_(getattr(fr, k), non_blocking=True)

    e2e_step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.e2e_steps):
        e2e_step()
    e1.record()
    barrier()
    e2e_serial_ms = e0.elapsed_time(e1) / args.e2e_steps

    # The same work, software-pipelined over three streams and two sets of device buffers: the H2D copies of step
    # i+1 and the D2H reads of step i-1 overlap the kernels of step i (PCIe is full duplex), every step still moves
    # all of its inputs in and all of its results out.
    fr2 = mg.Frame(cam, sc.N)
    g2, m2 = mg.upload(sc)
    gimg2 = gimg.clone()
    fr2.forward(g2, m2)
    fr2.backward(g2, m2, gimg2)
    host_out2 = {k: torch.empty_like(t).pin_memory() for k, t in host_out.items()}
    torch.cuda.synchronize()
    bufs = [(fr, g, m, gimg, host_out), (fr2, g2, m2, gimg2, host_out2)]
    s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_cmp = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def pipelined(n):
        for i in range(n):
            b = i % 2
            f_, g_, m_, gi_, ho_ = bufs[b]
            with torch.cuda.stream(s_in):
                if i >= 2:
                    s_in.wait_event(ev_cmp[b])  # the kernels of step i-2 have consumed these input buffers
                for k, t in host_in.items():
                    g_[k].copy_(t, non_blocking=True)
                m_.copy_(host_m, non_blocking=True)
                gi_.copy_(host_g, non_blocking=True)
                ev_in[b].record(s_in)
            with torch.cuda.stream(s_cmp):
                s_cmp.wait_event(ev_in[b])
                if i >= 2:
                    s_cmp.wait_event(ev_out[b])  # the results of step i-2 have left these output buffers
                f_.step(g_, m_, gi_)
                ev_cmp[b].record(s_cmp)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_cmp[b])
                for k, t in ho_.items():
                    t.copy_(getattr(f_, k), non_blocking=True)
                ev_out[b].record(s_out)

    pipelined(2)
    barrier()
    n_pipe = max(args.e2e_steps, 4) * 2
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s_in)
    pipelined(n_pipe)
    s_out.wait_stream(s_cmp)
    e1.record(s_out)
    barrier()
    e2e_ms = e0.elapsed_time(e1) / n_pipe
    assert torch.equal(host_out["image"], host_out2["image"])  # both buffer sets produced the same frame
    e2e_ms = max_over_ranks(e2e_ms, world, "cuda")
    e2e_serial_ms = max_over_ranks(e2e_serial_ms, world, "cuda")

    # The link's own ceiling, measured the same way (pinned host memory, the 576 MB SH array in, the 576 MB SH gradient
    # out): each direction alone, then both at once on two streams.  e2e moves 733 MB each way per step, so
    # 733 MB / (the both-at-once rate) is the floor of an e2e step on this box whatever the kernels do.
    def copy_rate(do_in, do_out, reps=3):
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0.record()
        sa.wait_event(t0); sb.wait_event(t0)
        for _ in range(reps):
            if do_in:
                with torch.cuda.stream(sa):
                    g["sh"].copy_(host_in["sh"], non_blocking=True)
            if do_out:
                with torch.cuda.stream(sb):
                    host_out["dL_dsh"].copy_(fr.dL_dsh, non_blocking=True)
        torch.cuda.current_stream().wait_stream(sa)
        torch.cuda.current_stream().wait_stream(sb)
        t1.record()
        torch.cuda.synchronize()
        return reps * host_in["sh"].numel() * 4 / (t0.elapsed_time(t1) * 1e-3) / 1e9  # GB/s per direction

    link = {"h2d_alone_gb_per_s": round(copy_rate(True, False), 1), "d2h_alone_gb_per_s": round(copy_rate(False, True), 1),
            "both_at_once_gb_per_s_each_way": round(copy_rate(True, True), 1)}
    link["floor_ms_per_step"] = round(max(h2d, d2h) / (link["both_at_once_gb_per_s_each_way"] * 1e9) * 1e3, 2)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    blends = (wc["fwd_blends"] + wc["bwd_blends"]) if wc else None
    value = world * blends / (ms_step * 1e-3) if blends else None
    e2e_value = world * blends / (e2e_ms * 1e-3) if blends else None

    # ---- rooflines: every call against the peak that bounds it; `roofline` = the dominant kernel's entry
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peaks = json.load(open(peaks_path)) if os.path.exists(peaks_path) else {}
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    hbm_gbs = float(peaks.get("hbm_gbs", 6540.8))
    hbm_source = "MEASURED_PEAKS.json hbm_gbs (copy, burst)" if "hbm_gbs" in peaks else "fallback of B200_PROFILING.md"
    fp32_derived = 148 * 128 * 2 * sm_max * 1e6 / 1e12  # TFLOP/s from the guide's unit counts (context)
    fp32_meas = mg.mg_measure_fp32_peak(0.05)             # timed on this chip, now (MEASURED_PEAKS.json has no FP32 entry)
    fp32_peak = max(fp32_meas["ffma_sustained"], fp32_meas["ffma2_sustained"])
    roofline, rooflines = None, None
    if wc:
        traffic = ncu_traffic(args.config)
        rooflines = {}
        tot = sum(per_call.values())
        for call, (bound, work) in algorithmic_work(wc, sc.N).items():
            sec = per_call[call] * 1e-3
            if bound == "alu":
                ach, peak, unit = work / sec / 1e12, fp32_peak, "TFLOP/s"
            else:
                # An HBM-bound call is credited with the bytes it had to move AND did move: the per-Gaussian constants
                # charge every row, but a kernel may skip rows that need no work (mg_preprocess_bwd does not touch the
                # SH rows of Gaussians without a gradient), and bytes nobody read are not bandwidth.  `frac` therefore
                # uses min(algorithmic, ncu DRAM traffic); both fractions are printed beside it.
                moved = traffic.get(call)
                charged = min(work, moved) if moved else work
                ach, peak, unit = charged / sec / 1e9, hbm_gbs, "GB/s"
                extra = {"charged_bytes": charged, "frac_algorithmic": work / sec / 1e9 / peak,
                         "frac_moved": (moved / sec / 1e9 / peak) if moved else None}
                if call == "bin_sort":  # the scheme's own byte count says nothing about the scheme: 4 B per key is any sort's floor
                    extra["frac_of_4B_per_key_floor"] = wc["R"] * 4 / sec / 1e9 / peak
            rooflines[call] = {"bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                               "traffic": traffic.get(call), "work_per_launch": work, "ms": per_call[call],
                               "share_of_step": per_call[call] / tot}
            if bound != "alu":
                rooflines[call].update(extra)
        dom = max(("render_fwd", "render_bwd"), key=lambda n: per_call[n])
        survey = wc[dom[7:] + "_pair_evals"] * FLOP_PAIR + wc[dom[7:] + "_blends"] * (FLOP_BLEND_BWD if dom == "render_bwd" else FLOP_BLEND_FWD)
        roofline = dict(rooflines[dom], kernel=dom + "_kernel",
                        traffic_unit="bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, profiles/r03_final.md)",
                        flop_per_launch=rooflines[dom]["work_per_launch"],
                        flop_counting="masked and unmasked work charged separately (bench.py FLOP_*, DESIGN.md 7.6)",
                        frac_by_survey_constants=survey / (per_call[dom] * 1e-3) / 1e12 / fp32_peak,
                        peak_source="measured: mg_measure_fp32_peak, dependent-free FMA chains on every SM, >= 50 ms, sustained",
                        peak_measured=fp32_meas, peak_derived=fp32_derived, hbm_peak_source=hbm_source)

    next_rows = None
    if world == 1:
        next_rows = {"mask_head": bench_mask_head(sc, g, hbm_gbs), "inference": bench_inference(sc, g, m),
                     "render_loss": bench_render_loss(sc, hbm_gbs), "optimizer": bench_optimizer(sc, g, fr, hbm_gbs)}
        ti = bench_training_iteration(sc, g, fr)
        nr = next_rows
        ti["sum_of_rows_ms"] = round(ms_step + nr["render_loss"]["ms"] + nr["optimizer"]["ms"]["adam_step"] + nr["optimizer"]["ms"]["density_stats"]
                                     + sum(nr["mask_head"]["ms"][k] for k in ("mask_sample", "mask_loss", "mask_sample_bwd")), 4)
        next_rows["training_iteration"] = ti
        next_rows["training_iteration_ms"] = ti["ms"]
        if args.all_cameras:
            next_rows["all_cameras"] = bench_cameras(sc, g, m)
        if args.config == 3 and not args.no_config5:
            # BASELINE.json configs[4]: "Forward+backward are timed over 20 cameras on a circle" -- in the default record
            sc5 = scenes.make(5)
            g5, m5 = mg.upload(sc5)
            next_rows["config5"] = dict(bench_cameras(sc5, g5, m5, steps=5), workload=workload_name(5).replace(", camera 0", ", its 20 cameras"))
            next_rows["config5"]["two_in_flight"] = bench_cameras_two_in_flight(sc5, g5, m5)

    cpu = None
    if not args.no_cpu_baseline:
        b, sec, info = oracle_sample(args.config)
        cpu = {"value": b / sec, "unit": "blends/s", "cores": n_threads(), "kind": "oracle", "sample": info}

    gw, gh = mg.grid(cam)
    launches = args.steps * sum(KERNELS_PER_STEP.values())
    line = {"metric": "gaussian_pixel_blends_per_s", "value": value, "unit": "blends/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "N": sc.N, "width": cam.width, "height": cam.height,
                       "sh_degree": cam.sh_degree, "R": R, "l2": "inputs (708 MB of Gaussians + sort buffers) exceed the 126 MB L2; no flush",
                       "parallelism": "replicas only" if world > 1 else "1 GPU"},
            "ms_per_frame": ms_step, "ms_per_call": per_call,
            "pair_evals_per_s": (world * (wc["fwd_pair_evals"] + wc["bwd_pair_evals"]) / (ms_step * 1e-3)) if wc else None,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "blends/s", "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "how": "pinned host buffers; H2D of all inputs and D2H of image + all gradients every step, software-pipelined over 3 streams and 2 buffer sets",
                    "ms_per_step_unpipelined": e2e_serial_ms,
                    "gb_per_s_each_way": round(max(h2d, d2h) / (e2e_ms * 1e-3) / 1e9, 1), "link_ceiling": link},
            "gpu_launches": launches, "roofline": roofline, "rooflines": rooflines, "cpu_baseline": cpu,
            "next_rows": next_rows}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
