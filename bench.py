"""bench.py -- frames/s and Gsamples/s of the bricked ray-casting hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c2|c1|c0]
                    [--impl ours|reference] [--no-variants] [--no-cpu-baseline]

A step is ONE FRAME: one pass of the whole hot path (view set-up + visibility sort, per-brick
ray casting, sort-last compositing: rows a2..a9 of SURVEY.md sec. 8) for one view of the
workload's 36-view cycle, on a synthetic radio-spectral-cube stand-in already resident in HBM
as ghost-padded bricks (row a1, built once before the timed region, as in the paper:
PAPER.md:146 loads the data once, :150 renders per view). DESIGN.md "Measurement" states the
recipe, the algorithmic bytes and the roofline.

Default workload = BASELINE.json configs[3] ("c3"): 4096x4096x1536 float32 (~103 GB) in 512^3
ghost-padded bricks, 1920x1080, 36-view turntable, ALPHA, step 1.0, early termination 0.99 --
the configuration the metric ("frames/sec and Gsamples/s at 1920x1080 on 1 B200") and
north_star's target (">= 100 GB in-core cube at 1920x1080") are quoted on.

N > 1 (torchrun): frames are independent units, so each rank holds its own copy of the cube
and renders K frames of the cycle (different view offsets); no data-path collective; the
aggregate is N*K frames over the slowest rank's time ("scaling": "weak").

Prints ONE JSON line (rank 0).
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402  (seeded inputs only)

METRIC = "frames/s at 1920x1080 (with Gsamples/s and roofline fraction beside it)"


# ----------------------------------------------------------------------------- workloads
def workload(name):
    """Shapes, cameras and classification of BASELINE.json's configs."""
    c = dict(synth.CONFIGS[name])
    c["name"] = name
    c["seed"] = synth.BASE_SEED + int(name[1:]) + {"n": 10, "s": 20}.get(name[0], 0)
    c.setdefault("kind", 0)
    fr = synth.Framing(c["nx"], c["ny"], c["nz"], c["width"], c["height"])
    if name == "c2":  # "1920x1080 perspective output, 36 seeded views"
        c["views"] = [fr.seeded(c["seed"], k) for k in range(36)]
        c["view_kind"] = "36 seeded rotations"
    else:             # "36-frame turntable about the spectral axis"
        c["views"] = [fr.turntable(k) for k in range(36)]
        c["view_kind"] = "36-view turntable, elevation 20 deg"
    c["proj"] = fr.proj(False)
    c["tau"] = 0.99
    return c


def views_for_rank(rank, world, nviews):
    """Rank r starts its cycle at view r*nviews/world: ranks render different frames."""
    off = (rank * nviews) // max(world, 1)
    return [(off + k) % nviews for k in range(nviews)]


def aggregate(local_ms, frames_per_rank, world, all_reduce_max=None):
    """Whole-job frames/s: all ranks' frames over the SLOWEST rank's device time."""
    ms = all_reduce_max(local_ms) if all_reduce_max is not None else local_ms
    return frames_per_rank * world / (ms * 1e-3), ms


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: NVML polled every ~10 ms
    from a thread (the frames of the default workload take ~1 ms each, too short for the
    profiling recipe's `nvidia-smi -lms 200` line, which is the fallback)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index, self.thread, self.stop_flag = index, None, False
        self.sm, self.smax, self.reasons = [], None, set()

    def _poll(self):
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        while not self.stop_flag:
            self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
            try:
                mask = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
            except Exception:
                mask = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
            for bit, name in self.REASONS.items():
                if mask & bit:
                    self.reasons.add(name)
            time.sleep(0.01)

    def start(self):
        import threading
        self.stop_flag = False
        self.thread = threading.Thread(target=self._safe_poll, daemon=True)
        self.thread.start()
        time.sleep(0.05)

    def _safe_poll(self):
        try:
            self._poll()
        except Exception as e:  # NVML missing: fall back to one nvidia-smi query
            self.error = repr(e)

    def stop(self):
        self.stop_flag = True
        if self.thread is not None:
            self.thread.join(timeout=5)
        if not self.sm:
            try:
                q = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=clocks.sm,clocks.max.sm",
                                    "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=20).stdout
                a, b = (float(x) for x in q.strip().split(","))
                self.sm, self.smax = [a], b
            except Exception:
                return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.smax, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


# ----------------------------------------------------------------------------- product arm
def build_volume(vr, wl, tf):
    """Row a1: generate the cube on the device slab by slab (synth's CUDA twin) and upload it."""
    import torch
    # first launches of a kernel pay CUDA's lazy module loading (~1 ms): take it on a toy volume
    toy = vr.Volume(48, 40, 36, 16, wl["ghost"])
    toy.upload(torch.zeros((36, 40, 48), dtype=torch.float32, device="cuda"))
    toy.minmax()
    toy.close()
    cube = synth.Cube(wl["seed"], wl["nx"], wl["ny"], wl["nz"], wl["nsrc"], wl["ramp"], wl.get("kind", 0))
    # the store is mapped brick by brick (VR_LAYOUT_TILED_RELEASABLE: the same tiled layout for every kernel), so that the
    # LAST variant can hand it back array by array and render through the texture arm alone (vr_volume_release_store)
    try:
        g = vr.Volume(wl["nx"], wl["ny"], wl["nz"], wl["brick"], wl["ghost"], layout=vr.LAYOUT_TILED_RELEASABLE)
        g.releasable = True
    except vr.VrError:
        g = vr.Volume(wl["nx"], wl["ny"], wl["nz"], wl["brick"], wl["ghost"])
        g.releasable = False
    plane = wl["nx"] * wl["ny"] * 4
    nzs = max(1, min(wl["nz"], (4 << 30) // plane))  # 4 GiB slabs: 64 planes of config 3
    buf = torch.empty((nzs, wl["ny"], wl["nx"]), dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    evs = []
    for z0 in range(0, wl["nz"], nzs):
        nk = min(nzs, wl["nz"] - z0)
        cube.fill_device(buf[:nk].data_ptr(), 0, 0, z0, wl["nx"], wl["ny"], nk, st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.upload(buf[:nk], origin=(0, 0, z0))
        e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    del buf
    torch.cuda.empty_cache()
    g.set_transfer_function(tf, *tf_range(wl))
    g.set_early_termination(wl["tau"])
    # row a1 (once per cube): every source voxel read once, every padded brick cell written once
    pad = 1
    for n in (wl["nx"], wl["ny"], wl["nz"]):
        nb = -(-n // wl["brick"])
        pad *= n + 2 * wl["ghost"] * nb
    up_bytes = 4 * (wl["nx"] * wl["ny"] * wl["nz"] + pad)
    up_ms = sum(a.elapsed_time(b) for a, b in evs)
    g.upload_stats = {"kernel": "vr_upload_tma442_kernel (TMA box loads; vr_upload_tile442_kernel where the source is not 16-byte aligned)", "launches": len(evs), "ms": round(up_ms, 3), "bytes": up_bytes,
                      "gb_per_s": round(up_bytes / (up_ms * 1e-3) / 1e9, 1)}
    # every per-view buffer and table the frames below need, taken now: vr_render then never allocates or synchronises
    g.reserve_views(wl["views"], [wl["proj"]] * len(wl["views"]), wl["width"], wl["height"])
    torch.cuda.synchronize()
    # rows f1 + R19 (once per upload): one streaming read of the padded brick store gives the per-brick and the macro-cell ranges
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    lo, hi = g.minmax()
    e1.record()
    torch.cuda.synchronize()
    mm_ms = e0.elapsed_time(e1)
    g.minmax_stats = {"kernel": "vr_range_kernel (+ init, decode, reduce: 4 launches)", "ms": round(mm_ms, 3), "bytes": 4 * pad,
                      "gb_per_s": round(4 * pad / (mm_ms * 1e-3) / 1e9, 1), "data_min": float(lo), "data_max": float(hi)}
    return g, cube


def build_part(vr, wl, cube, tf, box):
    """A part handle of the workload's cube (row f3), filled with its region (bricks + ghost layers) only."""
    import torch
    from paper_1205_0282_b200 import sortlast
    dims = (wl["nx"], wl["ny"], wl["nz"])
    st = torch.cuda.current_stream().cuda_stream
    p = vr.Volume(*dims, wl["brick"], wl["ghost"], part=box)
    (x0, y0, z0), (sx, sy, sz) = sortlast.part_region(dims, wl["brick"], wl["ghost"], box)
    nzs = max(1, min(sz, (4 << 30) // (sx * sy * 4)))
    buf = torch.empty((nzs, sy, sx), dtype=torch.float32, device="cuda")
    for k0 in range(0, sz, nzs):
        nk = min(nzs, sz - k0)
        cube.fill_device(buf[:nk].data_ptr(), x0, y0, z0 + k0, sx, sy, nk, st)
        p.upload(buf[:nk], origin=(x0, y0, z0 + k0))
    torch.cuda.synchronize()
    del buf
    p.set_transfer_function(tf, *tf_range(wl))
    p.set_early_termination(wl["tau"])
    return p


def sortlast_report(vr, g, wl, cube, tf, nparts, order, K, Wm):
    """Row f3 measured on ONE GPU, the parts one after the other (no rank waits for another): each part of the k-d
    partition is created, filled with its region (bricks + ghost layers) and renders the K frames of the cycle as
    partial frames packed by rectangle (vr_render_part_pieces), stage events per frame; then the N pieces of one view are merged
    (vr_composite_parts, the work the N ranks share by stripes). The exchange itself needs N GPUs: its volume is
    reported from the geometry (the paper's M + epsilon), not timed."""
    import torch
    from paper_1205_0282_b200 import sortlast
    dims = (wl["nx"], wl["ny"], wl["nz"])
    Wp, Hp = wl["width"], wl["height"]
    boxes, tree = sortlast.kd_partition(dims, wl["brick"], nparts)
    out = torch.empty((Hp, Wp, 4), dtype=torch.float32, device="cuda")
    K = min(K, 64)  # frames whose stage events the library keeps
    frame_ms = np.zeros((nparts, K))
    pieces, rects, store_gb, ray_ms = [], [], [], []
    view0 = wl["views"][order[Wm % len(order)]]
    for r, box in enumerate(boxes):
        p = build_part(vr, wl, cube, tf, box)
        p.minmax()
        # what a rank does per frame: set-up, ray table, ray cast, and stage-1 compositing straight into the
        # rectangle-packed piece it sends (vr_render_part_pieces; here one piece = the part's whole rectangle)
        def part_frame(vi):
            rc = vr.part_rect(dims, wl["brick"], box, wl["views"][vi], wl["proj"], Wp, Hp)
            piece = out.view(-1)[:(rc[3] - rc[1]) * (rc[2] - rc[0]) * 4].view(rc[3] - rc[1], rc[2] - rc[0], 4)
            p.render_part_pieces(wl["views"][vi], wl["proj"], Wp, Hp, wl["step"], 0, [rc], [piece])
            return rc, piece

        for k in range(Wm):
            part_frame(order[k % len(order)])
        p.set_timing(1)  # the library's own stage events: device time of each frame's kernels, no host gaps
        torch.cuda.synchronize()
        for k in range(K):
            part_frame(order[(Wm + k) % len(order)])
        torch.cuda.synchronize()
        stg = p.debug_stage_times(K)
        frame_ms[r] = stg.sum(axis=1)
        ray_ms.append(round(float(stg[:, 1].mean()), 4))
        p.set_timing(0)
        rc, piece = part_frame(order[Wm % len(order)])
        torch.cuda.synchronize()
        pieces.append(piece.clone())
        rects.append(rc)
        nb = int(np.prod([box[1][a] - box[0][a] for a in range(3)]))
        store_gb.append(round(nb * (wl["brick"] + 2 * wl["ghost"]) ** 3 * 4 / 1e9, 2))
        p.close()
        torch.cuda.empty_cache()
    po = sortlast.part_order(tree, wl["brick"], view0, wl["proj"])
    merged = torch.empty((Hp, Wp, 4), dtype=torch.float32, device="cuda")
    for _ in range(3):
        g.composite_parts(0, pieces, rects, po, Wp, Hp, merged)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(20):
        g.composite_parts(0, pieces, rects, po, Wp, Hp, merged)
    e1.record()
    torch.cuda.synchronize()
    merge_ms = e0.elapsed_time(e1) / 20
    whole = torch.empty((Hp, Wp, 4), dtype=torch.float32, device="cuda")
    g.render(view0, wl["proj"], Wp, Hp, wl["step"], 0, whole)
    torch.cuda.synchronize()
    rdr = sortlast.SortLastRenderer(dims, wl["brick"], wl["ghost"], backend=object(), rank=0, world=nparts)
    moved = [rdr.exchange_bytes(wl["views"][v], wl["proj"], Wp, Hp) for v in sorted(set(order))]
    slowest = frame_ms.max(axis=0)  # per frame: the part every other rank waits for
    return {"parts": nparts, "boxes_bricks": [[b1[a] - b0[a] for a in range(3)] for b0, b1 in boxes], "store_gb_per_part": store_gb,
            "part_frame_ms": {"mean": round(float(frame_ms.mean()), 4), "slowest_part_mean": round(float(slowest.mean()), 4),
                              "per_part_mean": [round(float(x), 4) for x in frame_ms.mean(axis=1)], "per_part_raycast_mean": ray_ms},
            "render_bound_frames_per_s": round(1e3 / float(slowest.mean()), 1),
            "merge_ms_whole_frame": round(merge_ms, 4), "merge_launches": 1,
            "merged_vs_single_handle_max_abs": float((merged - whole).abs().max()),
            "exchange_bytes_per_frame": int(np.mean(moved)), "frame_bytes": Wp * Hp * 16,
            "what": "one GPU, parts rendered one after the other; frame time of a part = device time of its set-up, ray-cast and "
                    "stage-1 compositing kernels (stage events); render_bound_frames_per_s = 1 / mean over frames of the slowest "
                    "part's frame time, before the exchange, which is not timed here"}


def run_bricks_sharded(args, vr, wl, tf, mode_id, rank, world, local_rank, dist, reduce_max):
    """`--sharding bricks` (row f3): ONE cube over all ranks, every frame rendered by all of them (sort-last,
    paper_1205_0282_b200.sortlast). Strong scaling: the cube and the frames are fixed as N grows. Each rank fills
    only its own region (bricks + ghost layers) from the device generator. Timed like the frame-sharded arm:
    barrier + synchronise on both sides, CUDA events, maximum over ranks. The default on N > 1 ranks (north_star's bench
    line is the one-GPU cube; on one GPU this arm is the world of one and has to be asked for)."""
    import torch
    from paper_1205_0282_b200 import sortlast
    dims = (wl["nx"], wl["ny"], wl["nz"])
    cube = synth.Cube(wl["seed"], wl["nx"], wl["ny"], wl["nz"], wl["nsrc"], wl["ramp"], wl.get("kind", 0))
    rdr = sortlast.SortLastRenderer(dims, wl["brick"], wl["ghost"], rank=rank, world=world)
    (x0, y0, z0), (sx, sy, sz) = rdr.region()
    st = torch.cuda.current_stream().cuda_stream
    nzs = max(1, min(sz, (4 << 30) // (sx * sy * 4)))
    buf = torch.empty((nzs, sy, sx), dtype=torch.float32, device="cuda")
    for k0 in range(0, sz, nzs):
        nk = min(nzs, sz - k0)
        cube.fill_device(buf[:nk].data_ptr(), x0, y0, z0 + k0, sx, sy, nk, st)
        rdr.upload(buf[:nk], (x0, y0, z0 + k0))
    torch.cuda.synchronize()
    del buf
    rdr.set_transfer_function(tf, *tf_range(wl))
    rdr.set_early_termination(wl["tau"])
    lo, hi = rdr.minmax()
    # rows a1 / a5 on a part: the faster arm where it fits beside the part's store (a rank holds 1 / N of the cube) - float32
    # arrays for ALPHA values, 8-bit arrays as the exact MIP filter; falls back to the hand-rolled sampler (tests/test_gpu_sortlast.py)
    part_sampler = "manual"
    want = {"auto": "texture" if mode_id == 0 else "texture_byte", "manual": None}.get(args.sampler, args.sampler)
    if want and args.tf in ("ramp", "translucent"):
        try:
            rdr.backend.volume.set_sampler(sampler_id(vr, want))
            part_sampler = want
        except vr.VrError:
            pass
    W, H, K, Wm = wl["width"], wl["height"], args.steps, args.warmup
    nv = len(wl["views"])
    sampler = ClockSampler(local_rank) if rank == 0 else None
    for k in range(Wm):
        rdr.render(wl["views"][k % nv], wl["proj"], W, H, wl["step"], mode_id)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    l0 = rdr.backend.volume.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(K):
        frame = rdr.render(wl["views"][(Wm + k) % nv], wl["proj"], W, H, wl["step"], mode_id)
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    ms = reduce_max(e0.elapsed_time(e1))
    clocks = sampler.stop() if sampler else None
    launches = rdr.backend.volume.launch_count() - l0
    # end to end: the finished frame also travels to pinned host memory on rank 0, every step
    host = torch.empty((H, W, 4), dtype=torch.float32).pin_memory() if rank == 0 else None
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(K):
        frame = rdr.render(wl["views"][(Wm + k) % nv], wl["proj"], W, H, wl["step"], mode_id)
        if rank == 0:
            host.copy_(frame, non_blocking=True)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    e2e_ms = reduce_max((time.perf_counter() - t0) * 1e3)
    moved = int(np.mean([rdr.exchange_bytes(wl["views"][(Wm + k) % nv], wl["proj"], W, H, mode_id) for k in range(K)]))
    cfg = config_of(wl, args)
    cfg["sharding"] = "bricks: k-d partition into %d parts (row f3), one cube over all ranks, sort-last exchange" % world
    return {"metric": METRIC, "value": round(K / (ms * 1e-3), 3), "unit": "frames/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": round(ms / K, 4), "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": cfg, "gpu_launches": int(launches),
            "e2e": {"value": round(K / (e2e_ms * 1e-3), 3), "unit": "frames/s", "h2d_bytes_per_step": 128 * world,
                    "d2h_bytes_per_step": W * H * 16,
                    "what": "SortLastRenderer.render on every rank + the merged frame copied to pinned host memory on rank 0"},
            "clocks": clocks, "exchange_bytes_per_frame": moved, "frame_bytes": W * H * 16, "sampler": part_sampler + " (rank 0's part)",
            "data_range": [float(lo), float(hi)], "roofline": None, "cpu_baseline": None}


def tf_range(wl):
    """Data range the transfer function spans: [-3, 10] sigma for the spectral cubes, [0, 20] for density cubes."""
    return (0.0, synth.NBODY_VMAX) if wl.get("kind", 0) == synth.NBODY else (synth.TF_VMIN, synth.TF_VMAX)


def pick_tf(wl, name):
    if wl.get("kind", 0) == synth.NBODY:  # zero-opacity toe: empty space is exactly transparent (R16)
        t = synth.tf_density()
        if name == "translucent":
            t[:, 3] /= 64.0
        return t
    if name == "threshold":  # noise hidden: zero opacity below 3.5 sigma (macro-cell skipping, R19)
        return synth.tf_threshold()
    return synth.tf_ramp() if name == "ramp" else synth.tf_translucent()


def count_pass(g, vr, wl, mode, view_ids, out, cells_every):
    """Instrumented frames (never timed): samples per view, and for every `cells_every`-th view
    the distinct brick-store cells / 32-byte sectors its samples read (algorithmic bytes)."""
    import torch
    res = {}
    for n, vi in enumerate(view_ids):
        want_cells = cells_every > 0 and n % cells_every == 0
        g.set_counting(2 if want_cells else 1)
        g.render(wl["views"][vi], wl["proj"], wl["width"], wl["height"], wl["step"], mode, out)
        torch.cuda.synchronize()
        s = g.debug_stats()
        assert s["overflow"] == 0
        res[vi] = s
    g.set_counting(0)
    return res


def timed_device(g, wl, mode, order, K, W, out, dist=None):
    """K frames back to back on one stream, CUDA events at both ends, stage events inside."""
    import torch
    for k in range(W):
        g.render(wl["views"][order[k % len(order)]], wl["proj"], wl["width"], wl["height"], wl["step"], mode, out)
    g.set_timing(1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    l0 = g.launch_count()
    e0.record()
    for k in range(K):
        g.render(wl["views"][order[(W + k) % len(order)]], wl["proj"], wl["width"], wl["height"], wl["step"], mode, out)
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - l0
    nst = min(K, 64)
    stages = g.debug_stage_times(nst)                       # last nst frames, oldest first
    stage_views = [order[(W + k) % len(order)] for k in range(K - nst, K)]
    g.set_timing(0)
    return ms, launches, stages, stage_views


def timed_e2e(g, wl, mode, order, K, W, host_bufs, dist=None, pipelined=True):
    """Same frames through the host-buffer entries: per frame the matrices go host->device (as
    kernel arguments) and the finished RGBA frame comes back into pinned host memory; both
    inside the timed region. pipelined: vr_render_host_async (frame i's copy overlaps frame
    i+1's rendering, two frames in flight, three rotating pinned buffers) and one
    vr_render_host_wait before the closing event; else vr_render_host, which waits per frame."""
    import torch

    def frame(k):
        view = wl["views"][order[k % len(order)]]
        if pipelined:
            g.render_host_async(view, wl["proj"], wl["width"], wl["height"], wl["step"], mode, host_bufs[k % len(host_bufs)])
        else:
            g.render_host(view, wl["proj"], wl["width"], wl["height"], wl["step"], mode, out=host_bufs[0])

    for k in range(W):
        frame(k)
    g.render_host_wait()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(K):
        frame(W + k)
    g.render_host_wait()
    torch.cuda.synchronize()
    ms = (time.perf_counter() - t0) * 1e3
    if dist is not None:
        dist.barrier()
    return ms


def traffic_of(workload, mode, tf):
    """DRAM bytes (read + write) of ONE ray-cast launch from the committed `ncu --set full`
    capture of this workload (profiles/r2_traffic.csv, written from the .ncu-rep files as
    profiles/r2_traffic.md describes), or None. QUOTED from that capture of one view, not measured in this run
    (the line says so: `traffic_source`)."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "r2_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if (row["workload"], row["mode"], row["tf"]) == (workload, mode, tf):
                    return int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
    except Exception:
        pass
    return None


def roofline_of(counts, stages, stage_views, peak_gbs, peak_src, traffic=None):
    """Ray-cast kernel (the dominant one): algorithmic bytes = 4 B x distinct brick-store cells
    its samples read + the sub-image bytes it writes, over the views the
    counting pass covered; duration = that kernel's device time for the same views inside the
    timed region (library stage events on the render stream). `lines_*`: the same with the
    distinct 128-byte lines of the brick store instead of the cells - what DRAM must deliver
    for this layout at least."""
    by_view = {}
    for (ms_setup, ms_ray, ms_comp), vi in zip(stages, stage_views):
        by_view.setdefault(vi, []).append(float(ms_ray))
    alg, lines, ms, n = 0.0, 0.0, 0.0, 0
    for vi, s in counts.items():
        if s["cells_touched"] >= 0 and vi in by_view:
            alg += 4.0 * s["cells_touched"] + s["subimage_bytes"]
            lines += 128.0 * s["lines_touched"] + s["subimage_bytes"]
            ms += float(np.mean(by_view[vi]))
            n += 1
    if n == 0 or ms <= 0:
        return None
    achieved = alg / (ms * 1e-3) / 1e9
    lines_gbs = lines / (ms * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": "vr_raycast_kernel", "achieved": round(achieved, 1), "peak": peak_gbs, "unit": "GB/s",
            "frac": round(achieved / peak_gbs, 4), "traffic": traffic,
            "traffic_source": "quoted: dram__bytes_read.sum + dram__bytes_write.sum of one launch in the committed ncu capture "
                              "(profiles/r2_traffic.csv), not measured in this run" if traffic else None,
            "peak_source": peak_src,
            "algorithmic_bytes_per_launch": round(alg / n), "launch_ms": round(ms / n, 4), "views_counted": n,
            "lines_bytes_per_launch": round(lines / n), "lines_gbs": round(lines_gbs, 1),
            "lines_frac": round(lines_gbs / peak_gbs, 4)}


# Issued instructions one sample NEEDS, whatever the kernel: ALPHA 8 loads + 7 lerp FMA + 7 differences
# + 6 position adds + 3 weights + classification (scale, index, fraction, 2 shared loads, 4 FMA) + opacity (2 MUFU, 3 FP) +
# blending (5 FP) + termination and loop control (~5) = 55; MIP drops classification, opacity and blending: 30.
ALGORITHMIC_INSTRUCTIONS = {"alpha": 55, "mip": 30}
SM_COUNT, SCHEDULERS_PER_SM = 148, 4


def roofline_alu(gsamples_per_s, mode, sm_mhz, traffic=None):
    """Issue-slot bound of the sample loop, the bound of DENSELY sampled views (configs 0, 1, 2, 4: >= 0.6 samples per
    voxel, every line is reused from L1/L2 and DRAM idles). The peak uses the ALGORITHMIC work of a sample (SURVEY.md sec.
    8(d): 8 loads, 7 lerps, the position update, one LUT lerp with 2 shared loads, one pow on 2 MUFU, ~8 FMA of blending:
    50-60 issued instructions; ALGORITHMIC_INSTRUCTIONS = 55 for ALPHA, 30 for MIP, which has no classification, opacity
    or blending), NOT this kernel's own SASS count: peak = SMs x 4 warp schedulers x max SM clock x 32 lanes / that count.
    `frac` is then the distance from what the method needs, whatever the sampler (the texture arm issues fewer)."""
    clock = (sm_mhz or 1965.0) * 1e6
    peak = SM_COUNT * SCHEDULERS_PER_SM * clock * 32.0 / ALGORITHMIC_INSTRUCTIONS[mode] / 1e9
    return {"bound": "alu", "kernel": "vr_raycast_kernel", "achieved": round(gsamples_per_s, 2), "peak": round(peak, 1),
            "unit": "Gsamples/s", "frac": round(gsamples_per_s / peak, 4), "traffic": traffic,
            "peak_source": "%d SMs x %d schedulers x %.0f MHz (max SM clock) x 32 lanes / %d ALGORITHMIC instructions per sample "
                           "(SURVEY.md 8(d): 50-60 for ALPHA)" % (SM_COUNT, SCHEDULERS_PER_SM, clock / 1e6, ALGORITHMIC_INSTRUCTIONS[mode])}


def measured_peak():
    try:
        p = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(p["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


# ----------------------------------------------------------------------------- oracle legs
def oracle_volume(wl, tf):
    """The CPU oracle as it stands (oracle/, test infrastructure) on the same seeded cube:
    dense on the host when the cube is small, procedural voxels otherwise (no 103 GB host copy)."""
    import oracle
    cube = synth.Cube(wl["seed"], wl["nx"], wl["ny"], wl["nz"], wl["nsrc"], wl["ramp"], wl.get("kind", 0))
    nvox = wl["nx"] * wl["ny"] * wl["nz"]
    if nvox <= 512 ** 3:
        o = oracle.Volume(wl["nx"], wl["ny"], wl["nz"], wl["brick"], wl["ghost"], data=cube.fill_host())
        how = "dense host cube"
    else:
        o = oracle.Volume(wl["nx"], wl["ny"], wl["nz"], wl["brick"], wl["ghost"], voxel_fn=cube.voxel_fn())
        how = "procedural voxels"
    o.set_transfer_function(tf, *tf_range(wl))
    o.set_early_termination(wl["tau"])
    o._cube = cube
    return o, how


def sample_pixels(wl, n, salt):
    W, H = wl["width"], wl["height"]
    return np.array([[int(synth.u01(wl["seed"] + salt, 31, k) * W), int(synth.u01(wl["seed"] + salt, 32, k) * H)]
                     for k in range(n)], dtype=np.int32)


def oracle_sample_rate(o, wl, mode_id, view, npix, salt, cores):
    """Seconds, samples taken, for `npix` seeded pixels of one view."""
    pix = sample_pixels(wl, npix, salt)
    t0 = time.perf_counter()
    r = o.render(view, wl["proj"], wl["width"], wl["height"], wl["step"], mode_id, pixels=pix, nthreads=cores)
    dt = time.perf_counter() - t0
    return dt, int(r["counts"][:, 0].sum())


def cpu_baseline(wl, tf, mode_id, budget_s=15.0):
    """Oracle timed on the host cores on a bounded seeded pixel sample of the same frames,
    extrapolated to frames/s (sample pixels -> all W*H pixels). Baseline only."""
    cores = synth.default_threads()
    o, how = oracle_volume(wl, tf)
    dt, _ = oracle_sample_rate(o, wl, mode_id, wl["views"][0], 512, 1, cores)       # calibration
    per_pixel = max(dt / 512, 1e-7)
    views = [0, 9, 18, 27]
    npix = int(max(256, min(wl["width"] * wl["height"], budget_s / len(views) / per_pixel)))
    tot_t, tot_s = 0.0, 0
    for n, vi in enumerate(views):
        dt, ns = oracle_sample_rate(o, wl, mode_id, wl["views"][vi], npix, 2 + n, cores)
        tot_t += dt
        tot_s += ns
    frame_s = tot_t / len(views) * (wl["width"] * wl["height"] / float(npix))
    return {"value": 1.0 / frame_s, "unit": "frames/s", "cores": cores, "kind": "oracle",
            "sample": "%d seeded pixels of each of views %s (%s), extrapolated to %dx%d pixels" % (
                npix, views, how, wl["width"], wl["height"]),
            "msamples_per_s": tot_s / tot_t / 1e6}


def run_reference(args, wl, tf, mode_id):
    """--impl reference: the oracle IS the reference arm of this tier. Each step is a bounded
    seeded pixel sample of one frame of the cycle; value = extrapolated frames/s."""
    cores = synth.default_threads()
    o, how = oracle_volume(wl, tf)
    dt, _ = oracle_sample_rate(o, wl, mode_id, wl["views"][0], 512, 1, cores)
    per_pixel = max(dt / 512, 1e-7)
    total = max(1, args.steps + args.warmup)
    npix = int(max(256, min(wl["width"] * wl["height"], 90.0 / total / per_pixel)))
    for k in range(args.warmup):
        oracle_sample_rate(o, wl, mode_id, wl["views"][k % 36], npix, 100 + k, cores)
    t, ns = 0.0, 0
    for k in range(args.steps):
        dt, s = oracle_sample_rate(o, wl, mode_id, wl["views"][(args.warmup + k) % 36], npix, 200 + k, cores)
        t += dt
        ns += s
    scale = wl["width"] * wl["height"] / float(npix)
    ms_per_step = t / args.steps * scale * 1e3
    fps = 1e3 / ms_per_step
    sample = "%d seeded pixels per step (%s), extrapolated to %dx%d pixels" % (npix, how, wl["width"], wl["height"])
    return {"impl": "reference", "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_of(wl, args),
            "gsamples_per_s": ns / t / 1e9,
            "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def config_of(wl, args):
    what = "density cube: zero + %d extended halos" % wl["nsrc"] if wl.get("kind", 0) else \
        "noise + %d Gaussian sources%s" % (wl["nsrc"], " + spectral ramp" if wl["ramp"] else "")
    return {"workload": "%s: %dx%dx%d float32 cube (%s), %d^3 bricks + %d ghost, %dx%d, %s, %s, step %.1f, tf %s, "
                        "early termination %.2f%s" % (
                            wl["name"], wl["nx"], wl["ny"], wl["nz"], what, wl["brick"], wl["ghost"], wl["width"], wl["height"],
                            wl["view_kind"], args.mode.upper(), wl["step"], args.tf, wl["tau"],
                            (", fused traversal" if getattr(args, "traversal", "sort_last") == "fused" else "") +
                            (", texture sampler" if getattr(args, "sampler_asked", "auto") == "texture" else "")),
            "baseline_config_index": int(wl["name"][1:]) if wl["name"][0] == "c" else None,
            "cube_gb": round(wl["nx"] * wl["ny"] * wl["nz"] * 4 / 1e9, 2),
            "l2_policy": "inputs larger than L2 (every frame streams a new view's share of the cube); no explicit flush",
            "frames": "one frame per step, cycling the 36 views"}


# ----------------------------------------------------------------------------- config 4
def run_c4(args, vr, peak, peak_src, sampler):
    """BASELINE.json configs[4]: (i) the 1024^3 cube of config 2 rendered at 512^2 .. 4096^2 in
    ALPHA mode (seeded views, ramp TF, tau 0.99); (ii) the compositing microbenchmark: 64 seeded
    premultiplied full-frame 4096^2 RGBA layers composited in a seeded visibility order
    (vr_composite, row a9 alone). The roofline object is the compositing kernel's: pure HBM
    streaming, algorithmic bytes = every layer pixel read once + the frame written once."""
    import torch
    K, Wm = args.steps, args.warmup
    st = torch.cuda.current_stream().cuda_stream
    # (ii) first, while HBM is empty: 64 x 268 MB layers
    W = H = 4096
    n = 64
    layers = []
    for l in range(n):
        t = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
        synth.layer_device(synth.BASE_SEED + 4, l, 0, W * H, t.data_ptr(), st)
        layers.append(t)
    rects = [(0, 0, W, H)] * n
    order = synth.permutation(synth.BASE_SEED + 4, n)
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    for _ in range(Wm):
        vr.composite(layers, rects, order, W, H, out)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    torch.cuda.synchronize()
    sampler.start()
    ev[0].record()
    for k in range(K):
        vr.composite(layers, rects, order, W, H, out)
        ev[k + 1].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    comp_ms = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(K)])
    comp_bytes = (n + 1) * W * H * 16
    achieved = comp_bytes / (comp_ms.mean() * 1e-3) / 1e9
    comp = {"layers": n, "width": W, "height": H, "ms": round(float(comp_ms.mean()), 4), "ms_min": round(float(comp_ms.min()), 4),
            "bytes": comp_bytes, "gb_per_s": round(achieved, 1), "launches": K}
    roof = {"bound": "hbm", "kernel": "vr_composite_kernel", "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
            "frac": round(achieved / peak, 4), "traffic": traffic_of("c4", "composite", "-"), "peak_source": peak_src,
            "algorithmic_bytes_per_launch": comp_bytes, "launch_ms": round(float(comp_ms.mean()), 4)}
    del layers, out
    torch.cuda.empty_cache()

    # (i) resolution sweep on config 2's cube
    wl = workload("c2")
    sweep, launches = [], K
    g = None
    if args.c4_part != "composite":
        g, _ = build_volume(vr, wl, synth.tf_ramp())
        if args.sampler in ("auto", "texture"):  # auto: the faster arm on this cube (ALPHA, ramp TF; the second copy fits)
            g.set_sampler(vr.SAMPLER_TEXTURE)
            args.sampler = "texture"
    for res in ((512, 1024, 2048, 4096) if g is not None else ()):
        w = dict(wl)
        w["width"] = w["height"] = res
        fr = synth.Framing(w["nx"], w["ny"], w["nz"], res, res)
        w["views"] = [fr.seeded(w["seed"], k) for k in range(36)]
        w["proj"] = fr.proj(False)
        img = torch.empty((res, res, 4), dtype=torch.float32, device="cuda")
        ids = list(range(36))
        timed = sorted(set(ids[(Wm + k) % 36] for k in range(K)))
        counts = count_pass(g, vr, w, 0, timed, img, 0)
        ms, nl, stages, _ = timed_device(g, w, 0, ids, K, Wm, img)
        launches += nl
        samples = sum(counts[ids[(Wm + k) % 36]]["samples"] for k in range(K))
        ray_gs = samples / K / (float(stages[:, 1].mean()) * 1e-3) / 1e9
        sweep.append({"width": res, "height": res, "frames_per_s": round(K / (ms * 1e-3), 3),
                      "roofline_alu": roofline_alu(ray_gs, "alpha", None),
                      "gsamples_per_s": round(samples / (ms * 1e-3) / 1e9, 3), "samples_per_frame": int(samples / K),
                      "stage_ms": {"setup": round(float(stages[:, 0].mean()), 4), "raycast": round(float(stages[:, 1].mean()), 4),
                                   "composite": round(float(stages[:, 2].mean()), 4)}})
        del img
    if g is not None:
        g.close()
    top = sweep[-1] if sweep else {"frames_per_s": round(1e3 / float(comp_ms.mean()), 3), "gsamples_per_s": None}
    return {"metric": METRIC, "value": top["frames_per_s"], "unit": "frames/s", "n_gpus": 1, "steps": K, "warmup": Wm,
            "ms_per_step": round(1e3 / top["frames_per_s"], 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "c4: value = frames/s of config 2's 1024^3 cube at 4096x4096 (ALPHA, step 0.5, ramp TF, tau 0.99, "
                                   "36 seeded views); `sweep` = the same at 512^2..4096^2; `compositing` = 64 seeded premultiplied "
                                   "4096^2 RGBA layers through vr_composite in a seeded order",
                       "baseline_config_index": 4,
                       "l2_policy": "inputs larger than L2 (17 GB of layers per compositing launch; 4.3 GB cube); no explicit flush"},
            "gsamples_per_s": top["gsamples_per_s"], "gpu_launches": launches, "sweep": sweep, "compositing": comp,
            "roofline": roof, "clocks": clocks, "e2e": None, "cpu_baseline": None}


# ----------------------------------------------------------------------------- DRAM probe
def run_probe_dram(vr, gib):
    """What a 4-byte load that misses L2 costs: for every load flavour, L2
    fetch-granularity limit and locality pattern, loads per second of one probe launch (CUDA events inside
    vr_debug_probe_dram). DRAM bytes per load need ncu: the same command under
    `ncu --metrics dram__bytes_read.sum,gpu__time_duration.sum` lists the launches in the order of `cases`
    (two launches per case: warm-up, then the timed one)."""
    import torch
    buf = torch.zeros((gib << 30) // 4, dtype=torch.float32, device="cuda")
    peak, peak_src = measured_peak()
    cases = []

    def case(flavour, span, group, gran=0, ctas=148 * 8, lpt=256):
        nonlocal buf
        ms, loads = vr.debug_probe_dram(buf, flavour, span, group, lpt, ctas, gran)
        cases.append({"flavour": vr.PROBE_FLAVOURS[flavour], "span_bytes": span, "group": group, "l2_fetch_granularity": gran or "default",
                      "ctas": ctas, "loads": loads, "ms": round(ms, 4), "gloads_per_s": round(loads / (ms * 1e-3) / 1e9, 2),
                      "gbs_if_128B_per_load": round(loads * 128 / (ms * 1e-3) / 1e9, 1)})

    for f in range(11):  # every load a random line (the ld.global flavours; the texture unit's are `--probe tex`)
        case(f, 128, 1)
    for gran in (32, 64, 128):                 # cudaLimitMaxL2FetchGranularity
        case(1, 128, 1, gran)
        case(6, 128, 1, gran)
    case(1, 128, 1, 128)                       # leave the limit at its largest value for what follows
    for span, group in ((256, 2), (512, 2), (512, 4), (1024, 2), (1024, 8), (2048, 2), (4096, 2), (4096, 8), (65536, 2), (65536, 8)):
        case(1, span, group)                   # locality: `group` lines of one aligned block
        case(6, span, group)
    for ctas in (148 * 2, 148 * 4, 148 * 16, 148 * 32):  # memory-level parallelism
        case(1, 128, 1, 0, ctas)
    # address range: does the miss rate depend on how many 2 MB pages the lines are spread over (TLB reach), beyond what the
    # L2 hit rate of a smaller range explains? (sub-ranges of the same buffer)
    whole = buf
    for mib in (256, 512, 1024, 2048, 4096, 8192):
        if mib << 20 < whole.numel() * 4:
            buf = whole[:(mib << 20) // 4]
            case(1, 128, 1, 0, 148 * 32)
            cases[-1]["range_mib"] = mib
    buf = whole
    del buf
    return {"probe": "dram", "buffer_gib": gib, "hbm_peak_gbs": peak, "hbm_peak_source": peak_src, "cases": cases}


def sampler_id(vr, name):
    return {"manual": vr.SAMPLER_MANUAL, "texture": vr.SAMPLER_TEXTURE, "texture_half": vr.SAMPLER_TEXTURE_HALF, "texture_byte": vr.SAMPLER_TEXTURE_BYTE}[name]


def run_probe_tex(vr):
    """The same question for the texture unit (profiles/r2_probe_dram.md, second part): random fetches through texture
    objects - tex1Dfetch over linear memory (4 and 16 bytes), tex3D point fetches of float4 texels and linear-filtered
    float fetches from a 3-D CUDA array the probe allocates - beside ld.global.nc, over 4 GiB, at two grid sizes."""
    import torch
    buf = torch.zeros((4 << 30) // 4, dtype=torch.float32, device="cuda")
    cases = []
    for ctas in (148 * 8, 148 * 32):
        for f in (1, 11, 12, 13, 14):
            ms, loads = vr.debug_probe_dram(buf, f, 128, 1, 256, ctas, 0)
            cases.append({"flavour": vr.PROBE_FLAVOURS[f], "ctas": ctas, "loads": loads, "ms": round(ms, 4),
                          "gloads_per_s": round(loads / (ms * 1e-3) / 1e9, 2)})
    return {"probe": "tex", "buffer_gib": 4, "cases": cases}


# ----------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=36)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c0", "c1", "c2", "c3", "c4", "n1", "s3"])
    ap.add_argument("--mode", default="alpha", choices=["alpha", "mip"])
    ap.add_argument("--tf", default="ramp", choices=["ramp", "translucent", "threshold"])
    ap.add_argument("--traversal", default="sort_last", choices=["sort_last", "fused"],
                    help="main arm: per-brick sub-images + compositing (the headline path) or the fused traversal (row f2)")
    ap.add_argument("--cells-every", type=int, default=6, help="count distinct cells on every n-th view of the cycle (0 = never)")
    ap.add_argument("--c4-part", default="both", choices=["both", "composite"],
                    help="--workload c4: `composite` runs only the compositing microbenchmark (profiling)")
    ap.add_argument("--sharding", default="auto", choices=["auto", "frames", "bricks"],
                    help="bricks = ONE cube over all ranks, sort-last with a rectangle-packed exchange (the paper's design, "
                         "PAPER.md:136, :178-184; row f3; strong scaling); frames = every rank holds the whole cube and renders its "
                         "own frames (replicas, weak scaling). auto (default): bricks when launched on N > 1 ranks - with the "
                         "replica figure beside it as `replicas` - and the one-GPU line otherwise")
    ap.add_argument("--sortlast-parts", type=int, default=8,
                    help="row f3 report: parts of the k-d partition rendered one after the other on this GPU (0 = skip)")
    ap.add_argument("--sampler", default="auto", choices=["auto", "manual", "texture", "texture_half", "texture_byte"],
                    help="row a5: manual = hand-rolled float32 tri-linear from the tiled store; texture = the texture-object arm "
                         "(ALPHA frames; a second copy of the bricks as 3-D CUDA arrays). auto (default): 'whichever ncu shows is "
                         "faster' (north_star; DESIGN.md section 9) - the texture arm for ALPHA frames with a smooth table, on a "
                         "second copy where it fits beside the store, else on the RELEASED store (vr_volume_release_store, the "
                         "run's last leg, which then supplies the headline with the hand-rolled figures beside it as "
                         "`hand_rolled`); manual for MIP, stepped tables and the fused traversal's default")
    ap.add_argument("--release-store", action="store_true",
                    help="profiling: hand the float32 store back right after the build (vr_volume_release_store) and render the main "
                         "arm through the texture arm alone; implies --sampler texture --no-variants --cells-every 0")
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--probe", default=None, choices=["dram", "tex"],
                    help="dram: the DRAM fetch-granularity probe (vr_debug_probe_dram) instead of a workload; tex: the same for "
                         "fetches through texture objects; one JSON line")
    ap.add_argument("--probe-gib", type=int, default=16, help="--probe dram: size of the probed buffer")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.sampler_asked = args.sampler  # `config` names the sampler only when the caller chose it (both arms print the same config)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    wl = workload(args.workload if args.workload != "c4" else "c2")
    tf = pick_tf(wl, args.tf)
    mode_id = 0 if args.mode == "alpha" else 1

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args, wl, tf, mode_id)), flush=True)
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("NCCL_DEBUG", "INFO")  # the communicator's own log (rings / NVLS, transports) goes to stderr
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local_rank))

    from paper_1205_0282_b200 import build as vr_build
    if rank == 0:
        vr_build.build()
        synth._build.build()
    if dist is not None:
        dist.barrier()
    import paper_1205_0282_b200 as vr

    def reduce_max(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    if args.probe:
        if rank == 0:
            print(json.dumps(run_probe_dram(vr, args.probe_gib) if args.probe == "dram" else run_probe_tex(vr)), flush=True)
        return 0

    if args.workload == "c4":
        if world > 1:
            raise SystemExit("bench.py: --workload c4 is a single-GPU microbenchmark")
        peak, peak_src = measured_peak()
        print(json.dumps(run_c4(args, vr, peak, peak_src, ClockSampler(local_rank))), flush=True)
        return 0

    if args.sharding == "auto":
        args.sharding = "bricks" if world > 1 else "frames"
        auto = True
    else:
        auto = False
    if args.sharding == "bricks":
        line = run_bricks_sharded(args, vr, wl, tf, mode_id, rank, world, local_rank, dist, reduce_max)
        if auto and world > 1:  # beside it: N replicas of the whole cube, each rendering its own frames
            torch.cuda.empty_cache()
            g, _ = build_volume(vr, wl, tf)
            out = torch.empty((wl["height"], wl["width"], 4), dtype=torch.float32, device="cuda")
            order = views_for_rank(rank, world, len(wl["views"]))
            ms = timed_device(g, wl, mode_id, order, args.steps, args.warmup, out, dist)[0]
            fps, ms_max = aggregate(ms, args.steps, world, reduce_max)
            g.close()
            line["replicas"] = {"value": round(fps, 3), "unit": "frames/s", "scaling": "weak", "ms_per_step": round(ms_max / args.steps, 4),
                                "what": "every rank holds the whole cube and renders its own frames of the cycle; no data-path "
                                        "collective; all ranks' frames over the slowest rank's device time"}
        if rank == 0:
            print(json.dumps(line), flush=True)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    t_build = time.perf_counter()
    g, cube = build_volume(vr, wl, tf)
    t_build = time.perf_counter() - t_build
    promote = False  # auto: the texture arm on the released store becomes the headline (the run's last leg)
    if args.sampler == "auto":
        args.sampler = "manual"
        fits = torch.cuda.mem_get_info()[0] > 1.15 * wl["nx"] * wl["ny"] * wl["nz"] * 4  # a second copy fits (c0 - c2, n1)
        fits_byte = torch.cuda.mem_get_info()[0] > 0.3 * wl["nx"] * wl["ny"] * wl["nz"] * 4  # byte arrays fit (c3 too)
        if args.mode == "mip" and args.traversal == "sort_last" and fits_byte and not args.release_store:
            args.sampler = "texture_byte"  # exact MIP: byte arrays rule samples out, the float32 store supplies the values
        if args.mode == "alpha" and args.traversal == "sort_last" and args.tf in ("ramp", "translucent") and not args.release_store:
            if fits:
                args.sampler = "texture"
            else:
                promote = bool(getattr(g, "releasable", False)) and not args.no_variants and world == 1
    if args.release_store:
        if args.sampler == "texture_half":
            g.set_sampler(vr.SAMPLER_TEXTURE_HALF)  # the store is turned into float16 arrays
        else:
            args.sampler = "texture"
        g.release_store()
        args.no_variants, args.cells_every = True, 0
    elif args.sampler != "manual":
        g.set_sampler(sampler_id(vr, args.sampler))
    W, H, K, Wm = wl["width"], wl["height"], args.steps, args.warmup
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    host_bufs = [torch.empty((H, W, 4), dtype=torch.float32).pin_memory() for _ in range(3)]
    order = views_for_rank(rank, world, len(wl["views"]))
    timed_views = sorted(set(order[(Wm + k) % len(order)] for k in range(K)))

    def measure(mode, with_e2e, sampler):
        counts = count_pass(g, vr, wl, mode, timed_views, out, args.cells_every)
        if sampler:
            sampler.start()
        ms, launches, stages, stage_views = timed_device(g, wl, mode, order, K, Wm, out, dist)
        e2e_ms = timed_e2e(g, wl, mode, order, K, Wm, host_bufs, dist, True) if with_e2e else None
        e2e_sync_ms = timed_e2e(g, wl, mode, order, K, Wm, host_bufs, dist, False) if with_e2e else None
        clocks = sampler.stop() if sampler else None
        samples = sum(counts[order[(Wm + k) % len(order)]]["samples"] for k in range(K))
        return dict(ms=ms, launches=launches, stages=stages, stage_views=stage_views, e2e_ms=e2e_ms, e2e_sync_ms=e2e_sync_ms, clocks=clocks,
                    samples=samples, counts=counts)

    peak, peak_src = measured_peak()
    g.set_traversal(vr.FUSED if args.traversal == "fused" else vr.SORT_LAST)
    m = measure(mode_id, True, ClockSampler(local_rank) if rank == 0 else None)
    g.set_traversal(vr.SORT_LAST)
    fps, ms_max = aggregate(m["ms"], K, world, reduce_max)
    e2e_fps, e2e_ms_max = aggregate(m["e2e_ms"], K, world, reduce_max)
    e2e_sync_fps, _ = aggregate(m["e2e_sync_ms"], K, world, reduce_max)

    line = {"metric": METRIC, "value": round(fps, 3), "unit": "frames/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": round(ms_max / K, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": config_of(wl, args),
            "gsamples_per_s": round(m["samples"] * world / (ms_max * 1e-3) / 1e9, 3),
            "samples_per_frame": int(m["samples"] / K),
            "gpu_launches": int(m["launches"]),
            "e2e": {"value": round(e2e_fps, 3), "unit": "frames/s", "h2d_bytes_per_step": 128, "d2h_bytes_per_step": W * H * 16,
                    "what": "vr_render_host_async + one vr_render_host_wait: matrices from host memory, every finished RGBA frame "
                            "copied to pinned host memory inside the timed region (frame i's copy overlaps frame i+1's rendering); "
                            "host wall clock around K frames with a device synchronise on both sides; the cube stays resident in "
                            "HBM (in-core rendering, PAPER.md:146,206)",
                    "synchronous_value": round(e2e_sync_fps, 3),
                    "synchronous_what": "vr_render_host: the caller waits for each frame's copy before queueing the next"},
            "clocks": m["clocks"],
            "sampler": ("texture_byte: 8-bit 3-D CUDA arrays as the exact MIP filter in front of the hand-rolled sampler" if args.sampler == "texture_byte"
                        else "texture_half: float16 copies of the float32 voxels in 3-D CUDA arrays (sampling only; ALPHA inside 2e-3, MIP exact)" if args.sampler == "texture_half"
                        else "texture: 3-D CUDA arrays behind texture objects, a second copy beside the store" if args.sampler == "texture"
                        else "manual: hand-rolled float32 tri-linear from the 4x4x2 micro-tiled store") +
                       (" (chosen by --sampler auto)" if args.sampler_asked == "auto" else ""),
            "stage_ms": {"setup": round(float(m["stages"][:, 0].mean()), 4), "raycast": round(float(m["stages"][:, 1].mean()), 4),
                         "composite": round(float(m["stages"][:, 2].mean()), 4)},
            # the paper's estimator: frame time per rotation angle, then its 75th percentile
            # over the angles; here one device-timed frame per view of the cycle (stage events summed)
            "frame_ms": {"p50": round(float(np.percentile(m["stages"].sum(axis=1), 50)), 4),
                         "p75": round(float(np.percentile(m["stages"].sum(axis=1), 75)), 4),
                         "min": round(float(m["stages"].sum(axis=1).min()), 4),
                         "max": round(float(m["stages"].sum(axis=1).max()), 4), "views": int(len(m["stages"]))},
            "roofline": roofline_of(m["counts"], m["stages"], m["stage_views"], peak, peak_src,
                                    traffic_of(args.workload, args.mode, args.tf + ("" if args.traversal == "sort_last" else "/fused") +
                                               ("/" + args.sampler if args.sampler != "manual" else ""))),
            "build_s": round(t_build, 1), "upload": dict(g.upload_stats, frac_of_hbm_peak=round(g.upload_stats["gb_per_s"] / peak, 4)),
            "minmax": dict(g.minmax_stats, frac_of_hbm_peak=round(g.minmax_stats["gb_per_s"] / peak, 4))}
    # which roofline bounds the ray-cast kernel: DRAM for the sparsely sampled 103 GB cube (0.03 samples per
    # voxel), issue slots for the densely sampled small cubes; the other one is reported beside it
    smax = (m["clocks"] or {}).get("sm_max_mhz") if rank == 0 else None
    ray_gs = m["samples"] / K / (float(m["stages"][:, 1].mean()) * 1e-3) / 1e9
    alu = roofline_alu(ray_gs, args.mode, smax, traffic_of(args.workload, args.mode, args.tf))
    if args.workload in ("c3", "s3"):
        line["roofline_alu"] = alu
    else:
        line["roofline_hbm"], line["roofline"] = line["roofline"], alu
    # row f1: bricks the transfer function makes transparent are skipped (exactly); report what that buys
    culled = [s["bricks_culled"] for s in m["counts"].values()]
    if max(culled) > 0 and args.traversal == "sort_last" and world == 1:
        g.set_culling(False)
        ms_off, _, st_off, _ = timed_device(g, wl, mode_id, order, K, Wm, out, dist)
        g.set_culling(True)
        line["culling"] = {"bricks": g.nbricks, "bricks_culled_mean": round(float(np.mean(culled)), 1),
                           "frames_per_s_culling_off": round(K / (ms_off * 1e-3), 3),
                           "raycast_ms_culling_off": round(float(st_off[:, 1].mean()), 4)}
    cs = [s for s in m["counts"].values() if s["cells_touched"] >= 0]
    if cs:
        line["touched_per_frame"] = {"cells_gb": round(np.mean([4.0 * s["cells_touched"] for s in cs]) / 1e9, 3),
                                     "sectors_gb": round(np.mean([32.0 * s["sectors_touched"] for s in cs]) / 1e9, 3),
                                     "lines_gb": round(np.mean([128.0 * s["lines_touched"] for s in cs]) / 1e9, 3),
                                     "subimage_gb": round(np.mean([s["subimage_bytes"] for s in cs]) / 1e9, 4)}

    if not args.no_variants and world == 1:
        variants = []
        # sort-last (the headline path) with the other transfer function / mode, then the fused traversal
        # (row f2: one ray through all bricks, global early termination, no sub-images, no compositing)
        other = "manual" if args.sampler == "texture" else "texture"  # the other arm of rows a1 / a5, on the same frames
        # MIP: 8-bit arrays as the exact filter (they fit beside the 103 GB cube too), and the hand-rolled sampler beside it
        mip_s = "texture_byte" if args.sampler_asked == "auto" else args.sampler
        for vmode, vtf, vtrav, vsamp in (("alpha", "translucent", "sort_last", args.sampler), ("mip", "ramp", "sort_last", mip_s),
                                         ("mip", "ramp", "sort_last", "manual"),
                                         # float16 copies of the voxels for sampling (half the fetched bytes; fits beside the 103 GB cube)
                                         ("alpha", "ramp", "sort_last", "texture_half"), ("alpha", "translucent", "sort_last", "texture_half"),
                                         ("alpha", "ramp", "sort_last", other), ("alpha", "translucent", "sort_last", other),
                                         ("alpha", "ramp", "fused", args.sampler), ("alpha", "translucent", "fused", args.sampler),
                                         ("alpha", "threshold", "sort_last", args.sampler), ("alpha", "threshold", "fused", args.sampler),
                                         ("alpha", "ramp, early termination off", "sort_last", args.sampler)):
            if vtrav == "sort_last" and vmode == args.mode and vtf == args.tf and vsamp == args.sampler:
                if vmode == "mip":
                    continue  # the main arm itself
                vtf = "ramp"
            if vmode == "mip" and vsamp == "manual" and mip_s == "manual":
                continue
            if vsamp == "texture_half" and args.sampler == "texture_half":
                continue  # the main arm and its first variant already
            if vmode == "alpha" and vsamp == "texture_byte":
                vsamp = "manual"  # byte arrays serve MIP only
            try:
                g.set_sampler(sampler_id(vr, vsamp))
            except vr.VrError as e:  # the 103 GB cube: no room for a second copy of the bricks as 3-D arrays
                variants.append({"mode": vmode, "tf": vtf, "traversal": vtrav, "sampler": vsamp, "unavailable": str(e)})
                continue
            noert = vtf.endswith("early termination off")  # the paper's protocol: with and without
            g.set_transfer_function(pick_tf(wl, "ramp" if noert else vtf), *tf_range(wl))
            g.set_early_termination(2.0 if noert else wl["tau"])
            g.set_traversal(vr.FUSED if vtrav == "fused" else vr.SORT_LAST)
            v = measure(0 if vmode == "alpha" else 1, False, None)
            extra = {}
            if vtf == "threshold":  # the same frames (bit-identical) without brick culling and macro-cell skipping
                g.set_culling(False)
                ms_off = timed_device(g, wl, 0, order, K, Wm, out, dist)[0]
                g.set_culling(True)
                extra = {"frames_per_s_skipping_off": round(K / (ms_off * 1e-3), 3)}
            g.set_traversal(vr.SORT_LAST)
            g.set_early_termination(wl["tau"])
            variants.append({"mode": vmode, "tf": vtf, "traversal": vtrav, "sampler": ("manual" if (vtf == "threshold" and vsamp == "texture") else vsamp) +
                                        (" (MIP: the arrays as an exact filter in front of the hand-rolled sampler)" if vmode != "alpha" and vsamp != "manual" else "") +
                                        (" (a stepped table keeps the hand-rolled sampler)" if vtf == "threshold" and vsamp == "texture" else ""),
                             "frames_per_s": round(K / (v["ms"] * 1e-3), 3), **extra,
                             "gsamples_per_s": round(v["samples"] / (v["ms"] * 1e-3) / 1e9, 3),
                             "samples_per_frame": int(v["samples"] / K),
                             "stage_ms": {"setup": round(float(v["stages"][:, 0].mean()), 4),
                                          "raycast": round(float(v["stages"][:, 1].mean()), 4),
                                          "composite": round(float(v["stages"][:, 2].mean()), 4)},
                             "counts_": v["counts"],
                             "roofline": roofline_of(v["counts"], v["stages"], v["stage_views"], peak, peak_src,
                                                     traffic_of(args.workload, vmode, vtf + ("" if vtrav == "sort_last" else "/fused") +
                                                                ("/" + vsamp if vsamp != "manual" and vtf != "threshold" else "")))})
        g.set_transfer_function(tf, *tf_range(wl))
        g.set_sampler(sampler_id(vr, args.sampler))
        line["variants"] = variants

        def brief(v):
            r = v.get("roofline") or {}
            return {"frames_per_s": v.get("frames_per_s"), "gsamples_per_s": v.get("gsamples_per_s"), "raycast_ms": (v.get("stage_ms") or {}).get("raycast"),
                    "frac": r.get("frac"), "traffic": r.get("traffic"),
                    "traffic_over_algorithmic": round(r["traffic"] / r["algorithmic_bytes_per_launch"], 2) if r.get("traffic") and r.get("algorithmic_bytes_per_launch") else None}
        # the narrow copies in one place (they are variants above): NOT the headline, which keeps float32 texels
        nt = {}
        for v in variants:
            if v.get("frames_per_s") is None or v["traversal"] != "sort_last":
                continue
            if v["mode"] == "alpha" and v["sampler"].startswith("texture_half") and v["tf"] in ("ramp", "translucent"):
                nt["alpha_%s_float16_texels" % v["tf"]] = brief(v)
            if v["mode"] == "mip" and v["sampler"].startswith("texture_byte"):
                nt["mip_8bit_exact_filter"] = brief(v)
            if v["mode"] == "mip" and v["sampler"].startswith("manual"):
                nt["mip_hand_rolled"] = brief(v)
        if nt:
            nt["what"] = ("float16 copies of the float32 voxels for ALPHA sampling (inside north_star's 2e-3 with the float32 arrays' error to two "
                          "digits: DESIGN.md R22; tests/test_gpu_texture.py, tests/test_gpu_fullsize.py) and 8-bit arrays as an exact MIP filter "
                          "(frames bit-identical to the hand-rolled path: R23); the headline `value` uses float32 texels")
            line["narrow_texels"] = nt
        # the workloads the paper's cubes look like (faint sources: PAPER.md:19, :206) beside the opaque ramp: the same
        # fraction (algorithmic bytes of the ray-cast kernel over its time, of the measured HBM peak) for every variant
        line["roofline_variants"] = [{"mode": args.mode, "tf": args.tf, "traversal": args.traversal, "sampler": args.sampler,
                                      "frac": line.get("roofline_hbm", line["roofline"])["frac"],
                                      "lines_frac": line.get("roofline_hbm", line["roofline"]).get("lines_frac"),
                                      "frames_per_s": line["value"]}] + [
            {"mode": v["mode"], "tf": v["tf"], "traversal": v["traversal"], "sampler": v["sampler"], "frac": v["roofline"]["frac"],
             "lines_frac": v["roofline"].get("lines_frac"), "frames_per_s": v["frames_per_s"]} for v in variants if "roofline" in v]
        if args.sortlast_parts > 1 and args.mode == "alpha":
            line["sortlast"] = sortlast_report(vr, g, wl, cube, tf, args.sortlast_parts, order, K, Wm)
        # LAST (irreversible): the texture arm on THIS cube even where a second copy of the bricks does not fit - the bricks
        # become 3-D arrays one by one and their float32 cells go back to the device; the same frames again. Sample sets are
        # the hand-rolled path's, so the counting passes above supply the algorithmic bytes.
        if getattr(g, "releasable", False):
            transl = [v for v in variants if v["tf"] == "translucent" and v["traversal"] == "sort_last" and "counts_" in v]
            try:
                t0 = time.perf_counter()
                freed = g.release_store()
                rel = {"what": "vr_volume_release_store: float32 store handed back brick by brick, ALPHA frames through 3-D CUDA "
                               "arrays only (8-bit filter weights: inside 2e-3 on these tables, tests/test_gpu_texture.py)",
                       "freed_gb": round(freed / 1e9, 2), "convert_s": round(time.perf_counter() - t0, 2)}
                for vtf, cnts in (("ramp", m["counts"] if args.tf == "ramp" and args.mode == "alpha" else None),
                                  ("translucent", transl[0]["counts_"] if transl else None)):
                    g.set_transfer_function(pick_tf(wl, vtf), *tf_range(wl))
                    main = promote and vtf == args.tf and cnts is not None
                    cl = ClockSampler(local_rank) if main else None
                    if cl:
                        cl.start()
                    ms_r, la_r, st_r, sv_r = timed_device(g, wl, 0, order, K, Wm, out, dist)
                    rel[vtf] = {"frames_per_s": round(K / (ms_r * 1e-3), 3), "raycast_ms": round(float(st_r[:, 1].mean()), 4)}
                    if cnts is not None:
                        rel[vtf]["roofline"] = roofline_of(cnts, st_r, sv_r, peak, peak_src, traffic_of(args.workload, "alpha", vtf + "/texture"))
                    if main:  # the headline: this arm is the faster one on this cube (profiles/r2_raycast_c3_ramp_tex.md)
                        e2e_r = timed_e2e(g, wl, 0, order, K, Wm, host_bufs, dist, True)
                        e2e_sync_r = timed_e2e(g, wl, 0, order, K, Wm, host_bufs, dist, False)
                        keep = ("value", "ms_per_step", "gsamples_per_s", "gpu_launches", "e2e", "clocks", "stage_ms", "frame_ms", "roofline")
                        hand = {k: line[k] for k in keep if k in line}
                        hand["e2e"] = {k: line["e2e"][k] for k in ("value", "synchronous_value")}
                        hand["sampler"] = "manual: hand-rolled float32 tri-linear from the 4x4x2 micro-tiled store (the same frames, before the store was handed back)"
                        line["hand_rolled"] = hand
                        frame_r = st_r.sum(axis=1)
                        line.update({"value": round(K / (ms_r * 1e-3), 3), "ms_per_step": round(ms_r / K, 4),
                                     "gsamples_per_s": round(m["samples"] / (ms_r * 1e-3) / 1e9, 3), "gpu_launches": int(la_r),
                                     "clocks": cl.stop(),
                                     "stage_ms": {"setup": round(float(st_r[:, 0].mean()), 4), "raycast": round(float(st_r[:, 1].mean()), 4),
                                                  "composite": round(float(st_r[:, 2].mean()), 4)},
                                     "frame_ms": {"p50": round(float(np.percentile(frame_r, 50)), 4), "p75": round(float(np.percentile(frame_r, 75)), 4),
                                                  "min": round(float(frame_r.min()), 4), "max": round(float(frame_r.max()), 4), "views": int(len(st_r))},
                                     "roofline": rel[vtf]["roofline"]})
                        line["e2e"] = dict(line["e2e"], value=round(K / (e2e_r * 1e-3), 3), synchronous_value=round(K / (e2e_sync_r * 1e-3), 3))
                        line["sampler"] = ("auto -> texture: 3-D CUDA arrays behind texture objects after vr_volume_release_store (the faster arm on "
                                                     "this cube: profiles/r2_raycast_c3_ramp_tex.md against r2_raycast_c3_ramp.md); `hand_rolled` holds "
                                                     "the same measurements of the hand-rolled sampler")
                        rel["headline"] = True
                line["texture_released"] = rel
                line["roofline_variants"] += [{"mode": "alpha", "tf": vtf, "traversal": "sort_last", "sampler": "texture (released store)",
                                               "frac": rel[vtf]["roofline"]["frac"], "lines_frac": rel[vtf]["roofline"].get("lines_frac"),
                                               "frames_per_s": rel[vtf]["frames_per_s"]}
                                              for vtf in ("ramp", "translucent") if "roofline" in rel.get(vtf, {})]
            except vr.VrError as e:
                line["texture_released"] = {"unavailable": str(e)}
        for v in variants:
            v.pop("counts_", None)

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        g.close()
        torch.cuda.empty_cache()
        line["cpu_baseline"] = cpu_baseline(wl, tf, mode_id)
        for k in ("value", "msamples_per_s"):
            line["cpu_baseline"][k] = round(line["cpu_baseline"][k], 6)
    elif rank == 0:
        line["cpu_baseline"] = None
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
