#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 spectral-cube ray caster.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload config1|config0|config2|config4|stream] [--layout tex|linear]

Metric (BASELINE.json): Gsamples/s (and frames/s) at 1920x1080 per cube size,
with the fraction of the bounding roofline.  Default workload = BASELINE.json
configs[1]: 512x512x1024 float32 cube (1 GiB; noise + 200 sources, seed 1),
perspective 1920x1080, 8 orbit views, step 0.5 voxel, emission-absorption and
MIP.  One "step" = one pass of the hot path over that batch = 16 frames
(8 views x {EA, MIP}).  Inputs are synthetic (vr_inputs), generated on the GPU.

Prints ONE JSON line (rank 0).  `value` is device-resident throughput, `e2e` the
same metric through the C ABI with HOST buffers (cube upload from pinned host
memory + frames copied back to pinned host memory inside the timed region).
N > 1 (torchrun): the path does not shard ("replicas only"):
every rank renders its own replica of the workload; value = total samples / max time.
"""
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

EA, MIP = 0, 1
LAYOUTS = {"linear": 0, "tex": 1}      # vr_layout

# Algorithmic work per sample, from the numerical contract:
# mandatory fp32/int lane-operations of S4-S8 (EA) and S4-S6+S9 (MIP).
LANE_OPS_PER_SAMPLE = {EA: 80, MIP: 55}
LANES_PER_SM = 128

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed ncu captures
NCU_TRAFFIC = {("config1", "tex", "raycast_kernel"): 1.0977e9}

WORKLOADS = {
    "config0": dict(config=0, W=256, H=256, step=0.5, views="config0", lut="A"),
    "config1": dict(config=1, W=1920, H=1080, step=0.5, views="orbit8", lut="A"),
    "config2": dict(config=2, W=1920, H=1080, step=1.0, views="orbit8", lut="A"),
    "config4": dict(config=4, W=7680, H=4320, step=0.25, views="orbit1", lut="S"),
}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self.index), "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

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
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(np.max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def get_views(vi, kind, dims):
    if kind == "config0":
        return vi.config0_views()
    if kind == "orbit1":
        return vi.orbit_views(dims, 8)[1:2]
    return vi.orbit_views(dims, 8)


def get_lut(vi, kind):
    return vi.lut_a() if kind == "A" else vi.lut_s()


def max_over_ranks(values, world, device):
    """Multi-GPU numbers are the max over ranks of device-timed values (replicas only: no data-path collective)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def resident_roofline(workload, layout, kernel_name, nvox, W, H, n_sm, pk, mip_ms, ea_ms, mip_samples, ea_samples):
    """The `roofline` object of a resident-cube bench line (pure arithmetic; tests/test_bench_cpu.py)."""
    alu_peak = n_sm * LANES_PER_SM * pk["sm_max_mhz"] * 1e6 / 1e12          # T lane-ops/s
    # dominant kernel: the MIP ray caster (no early termination, every sample evaluated)
    achieved = mip_samples * LANE_OPS_PER_SAMPLE[MIP] / (mip_ms * 1e-3) / 1e12
    hbm_bytes = nvox * 4 + H * W * 16             # every voxel once + the image
    alu = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "Tlane-op/s", "frac": achieved / alu_peak,
           "peak_source": f"{n_sm} SMs x {LANES_PER_SM} fp32 lanes x {pk['sm_max_mhz']:.0f} MHz (DESIGN.md Sec. 6)",
           "lane_ops_per_sample": LANE_OPS_PER_SAMPLE[MIP]}
    hbm = {"bound": "hbm", "achieved": hbm_bytes / (mip_ms * 1e-3) / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
           "frac": hbm_bytes / (mip_ms * 1e-3) / 1e9 / pk["hbm_gbs"], "algorithmic_bytes_per_launch": hbm_bytes,
           "peak_source": pk["source"]}
    # the binding roofline is the one with the longer ideal time for this workload
    t_alu = mip_samples * LANE_OPS_PER_SAMPLE[MIP] / (alu_peak * 1e12)
    t_hbm = hbm_bytes / (pk["hbm_gbs"] * 1e9)
    binding, other = (hbm, alu) if t_hbm > t_alu else (alu, hbm)
    roofline = dict(binding)
    roofline.update({
        "kernel": f"{kernel_name}<MIP, layout={layout}>",
        "traffic": NCU_TRAFFIC.get((workload, layout, kernel_name)),
        "traffic_source": "profiles/r01b_tex_mip_views012.md (ncu --set full, dram read + write, mean of views 0-2)"
                          if (workload, layout, kernel_name) in NCU_TRAFFIC else None,
        "avg_launch_ms": mip_ms, "units_per_launch": mip_samples,
        "ideal_ms": {"alu": t_alu * 1e3, "hbm": t_hbm * 1e3},
        "ea": {"avg_launch_ms": ea_ms, "units_per_launch": ea_samples,
               "achieved": ea_samples * LANE_OPS_PER_SAMPLE[EA] / (ea_ms * 1e-3) / 1e12,
               "frac": ea_samples * LANE_OPS_PER_SAMPLE[EA] / (ea_ms * 1e-3) / 1e12 / alu_peak,
               "note": "EA frame against the ALU roofline (80 lane-ops per sample); early termination leaves most voxels untouched"},
        other["bound"]: other})
    return roofline


# ---------------------------------------------------------------------------------
def run_ours(args, rank, world, local_rank):
    import torch
    import paper_1001_2049_b200 as vr
    import vr_inputs as vi

    vr.lib()                                   # fail loudly if libvr.so is missing
    wl = WORKLOADS[args.workload]
    spec = vi.CONFIGS[wl["config"]]
    W, H, step = wl["W"], wl["H"], wl["step"]
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    lut, vmin, vmax = get_lut(vi, wl["lut"])
    views = get_views(vi, wl["views"], spec.dims)
    modes = [EA, MIP]
    frames_per_step = len(views) * len(modes)
    nvox = int(np.prod(spec.dims))

    # ---- inputs, resident in HBM before the timed region -------------------------
    Vd = vi.make_cube(spec, device=dev)
    vol = vr.Volume(spec.dims, device=local_rank, layout=LAYOUTS[args.layout])
    vol.set_option(vr.VR_OPT_KERNEL, args.kernel)
    if args.kernel == 2:
        vol.set_option(vr.VR_OPT_BEAM_STAGES, args.beam_stages)
        vol.set_option(vr.VR_OPT_BEAM_STAGE, args.beam_stage_bytes)
        vol.set_option(vr.VR_OPT_BEAM_BULK, args.beam_bulk)
    vol.upload(Vd)
    vol.set_transfer_function(lut, vmin, vmax)
    out = torch.empty((H, W, 4), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev)

    # ---- samples per step (untimed counting pass; deterministic) -------------------
    vol.set_option(vr.VR_OPT_COUNT, 1)
    samples = {EA: 0, MIP: 0}
    rays = 0
    for m in modes:
        for cam in views:
            vol.render(cam, W, H, step, m, out=out)
            st = vol.stats()
            samples[m] += st["samples"]
            rays += st["rays_hit"]
    vol.set_option(vr.VR_OPT_COUNT, 0)
    samples_per_step = samples[EA] + samples[MIP]
    kernel_name = {1: "raycast_kernel", 2: "raycast_beam_kernel"}[vol.stats()["kernel"]]
    beam_stage = vol.stats().get("beam_stage_bytes", 0) if kernel_name == "raycast_beam_kernel" else None

    def one_step(evs=None):
        q = 0
        for m in modes:
            for cam in views:
                if evs is not None:
                    evs[q][0].record(stream)
                vol.render(cam, W, H, step, m, out=out)
                if evs is not None:
                    evs[q][1].record(stream)
                q += 1

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        one_step()
    barrier()

    # ---- timed region: K steps, device timers on the launching stream ----------------
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.2)
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            for _ in range(frames_per_step)] for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for k in range(args.steps):
        one_step(evs[k])
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks([total_ms], world, dev)[0]
    ms_per_step = total_ms / args.steps
    launch_ms = {EA: [], MIP: []}
    for k in range(args.steps):
        q = 0
        for m in modes:
            for _ in views:
                launch_ms[m].append(evs[k][q][0].elapsed_time(evs[k][q][1]))
                q += 1

    # ---- e2e: the same step through the C ABI with HOST buffers ------------------------
    e2e = None
    if rank == 0 or world > 1:
        h_cube = torch.empty(Vd.shape, dtype=torch.float32, pin_memory=True)
        h_cube.copy_(Vd)
        h_imgs = torch.empty((frames_per_step, H, W, 4), dtype=torch.float32, pin_memory=True)
        torch.cuda.synchronize(dev)

        def e2e_step():
            vr.vr_volume_upload_bricks(vol.handle, [(0, 0, 0)], [spec.dims], [h_cube.data_ptr()], 0,
                                       stream.cuda_stream)
            vr.vr_set_transfer_function(vol.handle, lut, vmin, vmax)
            q = 0
            for m in modes:
                for cam in views:
                    vol.render_host(cam, W, H, step, m, out, h_imgs[q])
                    q += 1
            stream.synchronize()               # the frames are in host memory

        e2e_step()
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        barrier()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        e2e_s = max_over_ranks([e2e_s], world, dev)[0]
        e2e = {"value": samples_per_step * world / e2e_s / 1e9, "unit": "Gsamples/s",
               "h2d_bytes_per_step": nvox * 4 + lut.nbytes,
               "d2h_bytes_per_step": frames_per_step * H * W * 16,
               "ms_per_step": e2e_s * 1e3, "frames_per_s": frames_per_step * world / e2e_s,
               "timer": "host wall clock around upload + 16 x vr_render_host + stream sync"}
        del h_cube, h_imgs

    if rank != 0:
        return None

    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    roofline = resident_roofline(args.workload, args.layout, kernel_name, nvox, W, H, n_sm, peaks(),
                                 float(np.mean(launch_ms[MIP])), float(np.mean(launch_ms[EA])),
                                 samples[MIP] / len(views), samples[EA] / len(views))

    line = {
        "metric": "Gsamples/s", "value": samples_per_step * world / (ms_per_step * 1e-3) / 1e9,
        "unit": "Gsamples/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{wl['config']}] {spec.name}: {spec.dims[0]}x{spec.dims[1]}x{spec.dims[2]} f32, "
                               f"{W}x{H}, {len(views)} views x (EA+MIP), step {step}",
                   "layout": args.layout, "frames_per_step": frames_per_step, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (cube %.2f GiB vs 126 MB L2); no flush" % (nvox * 4 / 2 ** 30),
                   **({"kernel": "beam", "beam_stages": args.beam_stages, "beam_bulk": args.beam_bulk, "beam_stage_bytes_last_frame": beam_stage}
                      if beam_stage is not None else {})},
        "frames_per_s": frames_per_step * world / (ms_per_step * 1e-3),
        "samples_per_step": samples_per_step, "rays_hit_per_step": rays,
        # nominal = no early termination, no skipping: MIP evaluates every sample of every ray, so EA's nominal
        # count is MIP's ("report also nominal samples")
        "nominal_samples_per_step": 2 * samples[MIP],
        "gpu_launches": frames_per_step * args.steps,
        "e2e": e2e, "roofline": roofline, "clocks": clocks,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(Vd.cpu().numpy(), lut, vmin, vmax, views, W, H, step, budget_s=20.0)
    vol.close()
    return line


# ---------------------------------------------------------------------------------
def mem_available_bytes():
    for line in open("/proc/meminfo"):
        if line.startswith("MemAvailable:"):
            return int(line.split()[1]) * 1024
    return 0


def run_stream(args, rank, world, local_rank):
    """--workload stream: BASELINE configs[3], the out-of-core path.  512^3-cell bricks in pinned host
    memory stream through a small device pool on the copy stream, overlapped with per-brick ray casting;
    the running image carries (C, A) from brick to brick in view order (S12).  The 4096^3 cube (256 GiB)
    does not fit this box's host memory: the largest near-cubic brick grid that fits in --ooc-gb (default:
    55 % of MemAvailable) stands in for it, same bricks / seed / generator."""
    import torch
    import paper_1001_2049_b200 as vr
    import vr_inputs as vi

    vr.lib()
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    B, W, H, step = 512, 1920, 1080, 0.5
    budget = args.ooc_gb * 1e9 if args.ooc_gb > 0 else 0.55 * mem_available_bytes() / max(1, world)
    spec = vi.ooc_spec(budget, brick=B)
    lut, vmin, vmax = vi.lut_a()
    views = vi.orbit_views(spec.dims, 8)[: args.stream_views]
    modes = [EA, MIP]
    frames_per_step = len(views) * len(modes)

    t0 = time.perf_counter()
    params = vi.source_params(spec)
    boxes = vi.brick_boxes(spec.dims, B)
    store = []
    for origin, size in boxes:                       # generated brick by brick from the seed
        pb = vr.PinnedBrick((size[2], size[1], size[0]))
        blk = vi.make_box(spec, origin, size, device=dev, params=vi.sources_in_box(spec, params, origin, size))
        torch.from_numpy(pb.array).copy_(blk)
        del blk
        store.append(pb)
    gen_s = time.perf_counter() - t0
    store_bytes = sum(4 * int(np.prod(pb.shape)) for pb in store)

    # host-link peak on this box: one brick-sized pinned copy, best of 5
    probe = torch.empty(store[0].array.size, dtype=torch.float32, device=dev)
    src = torch.from_numpy(store[0].array).reshape(-1)
    link = 0.0
    for _ in range(5):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        vr.lib().vr_host_alloc      # (the copy below is a plain cudaMemcpyAsync through torch)
        probe.copy_(src, non_blocking=True)
        b.record()
        torch.cuda.synchronize(dev)
        link = max(link, probe.numel() * 4 / (a.elapsed_time(b) * 1e-3) / 1e9)
    del probe

    vol = vr.Volume(spec.dims, host_brick=B, n_slots=args.slots, device=local_rank, layout=LAYOUTS[args.layout])
    vol.vr_volume_upload_bricks([(o, pb) for (o, _), pb in zip(boxes, store)])
    vol.set_transfer_function(lut, vmin, vmax)
    out = torch.empty((H, W, 4), dtype=torch.float32, device=dev)
    h_img = torch.empty((H, W, 4), dtype=torch.float32, pin_memory=True)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    # samples per step: one counting pass (doubles as warm-up)
    vol.set_option(vr.VR_OPT_COUNT, 1)
    samples = {EA: 0, MIP: 0}
    for m in modes:
        for cam in views:
            vol.render(cam, W, H, step, m, out=out)
            samples[m] += vol.stats()["samples"]
    vol.set_option(vr.VR_OPT_COUNT, 0)
    for _ in range(max(0, args.warmup - 1)):
        for m in modes:
            for cam in views:
                vol.render(cam, W, H, step, m, out=out)
    barrier()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h2d = streamed = 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        for m in modes:
            for cam in views:
                vol.render(cam, W, H, step, m, out=out)
                st = vol.stats()
                h2d += st["h2d_bytes"]
                streamed += st["bricks_streamed"]
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None

    # e2e: the frame delivered to pinned host memory (the cube already lives on the host)
    barrier()
    t0 = time.perf_counter()
    for m in modes:
        for cam in views:
            vol.render_host(cam, W, H, step, m, out, h_img)
    stream.synchronize()
    e2e_s = time.perf_counter() - t0
    total_ms, e2e_s = max_over_ranks([total_ms, e2e_s], world, dev)
    n_slots = vol.stats()["n_slots"]
    vol.close()
    for pb in store:
        pb.close()
    if rank != 0:
        return None

    ms_per_step = total_ms / args.steps
    samples_per_step = samples[EA] + samples[MIP]
    n_frames = frames_per_step * args.steps
    h2d_per_frame = h2d / n_frames
    achieved = h2d / (total_ms * 1e-3) / 1e9
    return {
        "metric": "Gsamples/s", "value": samples_per_step * world / (ms_per_step * 1e-3) / 1e9, "unit": "Gsamples/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[3] out-of-core, scaled to this host: {spec.dims[0]}x{spec.dims[1]}x{spec.dims[2]} f32 "
                               f"({store_bytes / 2 ** 30:.1f} GiB pinned, {len(boxes)} bricks of {B}^3 cells; the 4096^3 cube needs 256 GiB), "
                               f"{W}x{H}, {len(views)} views x (EA+MIP), step {step}",
                   "layout": args.layout, "frames_per_step": frames_per_step, "device_slots": n_slots,
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "every brick crosses the host link every frame; nothing is cached between frames",
                   "generate_s": gen_s},
        "frames_per_s": frames_per_step * world / (ms_per_step * 1e-3),
        "samples_per_step": samples_per_step, "bricks_streamed_per_frame": streamed / n_frames,
        "gpu_launches": int(streamed + n_frames),
        "e2e": {"value": samples_per_step * world / e2e_s / 1e9, "unit": "Gsamples/s",
                "h2d_bytes_per_step": int(h2d_per_frame * frames_per_step), "d2h_bytes_per_step": frames_per_step * H * W * 16,
                "ms_per_step": e2e_s * 1e3, "timer": "host wall clock around vr_render_host x frames + stream sync"},
        "roofline": {"bound": "host_link", "kernel": "cudaMemcpyAsync H2D of bricks (copy stream) overlapped with raycast_kernel<BRICK>",
                     "achieved": achieved, "peak": link, "unit": "GB/s", "frac": achieved / link, "traffic": None,
                     "peak_source": "measured in this run: brick-sized pinned H2D copy, best of 5 (PCIe Gen5 x16, 63 GB/s nominal)",
                     "algorithmic_bytes_per_launch": h2d_per_frame, "avg_launch_ms": total_ms / n_frames},
        "clocks": clocks,
    }


# ---------------------------------------------------------------------------------
def cpu_baseline(V, lut, vmin, vmax, views, W, H, step, budget_s):
    """The oracle as it stands, on the host cores, on a bounded sample of the workload."""
    import oracle
    import vr_inputs as vi
    cores = os.cpu_count()
    ij = vi.tile_subset(W, H, n_tiles=64, tile=128, seed=0)      # about half the frame: 10-30 s on 16 cores
    t_total, s_total, n_calls = 0.0, 0, 0
    done = []
    for v, cam in enumerate(views):
        for mode in (EA, MIP):
            t0 = time.perf_counter()
            _, _, cnt = oracle.render_pixels(V, lut, vmin, vmax, cam, W, H, step, mode, ij, nthreads=0)
            t_total += time.perf_counter() - t0
            s_total += cnt["samples"]
            n_calls += 1
        done.append(v)
        if t_total > budget_s:
            break
    return {"value": s_total / t_total / 1e9, "unit": "Gsamples/s", "cores": cores, "kind": "oracle",
            "sample": f"sixty-four 128x128-pixel tiles ({len(ij)} rays) of views {done}, EA + MIP, "
                      f"{s_total} samples in {t_total:.1f} s",
            "seconds": t_total}


def run_reference(args, rank):
    """--impl reference: the CPU oracle, as it stands, on the same config and metric."""
    if rank != 0:
        return None
    import torch
    import oracle
    import vr_inputs as vi
    wl = WORKLOADS[args.workload]
    spec = vi.CONFIGS[wl["config"]]
    W, H, step = wl["W"], wl["H"], wl["step"]
    lut, vmin, vmax = get_lut(vi, wl["lut"])
    views = get_views(vi, wl["views"], spec.dims)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    V = vi.make_cube(spec, device=dev).cpu().numpy()
    ij = vi.tile_subset(W, H, n_tiles=16, tile=32, seed=0)
    cores = os.cpu_count()

    def one_step():
        s = 0
        for cam in views:
            for mode in (EA, MIP):
                _, _, cnt = oracle.render_pixels(V, lut, vmin, vmax, cam, W, H, step, mode, ij, nthreads=0)
                s += cnt["samples"]
        return s

    for _ in range(min(args.warmup, 1)):
        one_step()
    t0 = time.perf_counter()
    s = 0
    for _ in range(args.steps):
        s += one_step()
    dt = time.perf_counter() - t0
    value = s / dt / 1e9
    sample = (f"each step = sixteen 32x32-pixel tiles (16384 rays) of all {len(views)} views, EA + MIP "
              f"({s // args.steps} samples per step)")
    return {"impl": "reference", "metric": "Gsamples/s", "value": value, "unit": "Gsamples/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"BASELINE configs[{wl['config']}] {spec.name}: {spec.dims[0]}x{spec.dims[1]}x{spec.dims[2]} f32, "
                                   f"{W}x{H}, {len(views)} views x (EA+MIP), step {step}",
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": "Gsamples/s", "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": "Gsamples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config1", choices=sorted(WORKLOADS) + ["stream"])
    ap.add_argument("--ooc-gb", type=float, default=0.0, help="stream: pinned brick store budget (0 = 55%% of MemAvailable)")
    ap.add_argument("--slots", type=int, default=3, help="stream: device slots")
    ap.add_argument("--stream-views", type=int, default=2, help="stream: orbit views per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--layout", default=None, choices=sorted(LAYOUTS),
                    help="device layout; default tex for resident cubes, linear for --workload stream (a brick lands in a "
                         "linear slot at the full host-link rate, 55.5 of 55.6 GB/s measured; into a CUDA array at 32 GB/s)")
    ap.add_argument("--beam-stages", type=int, default=1, choices=[1, 2],
                    help="--kernel 2: VR_OPT_BEAM_STAGES (2 = the next slab's box is copied while this one is marched)")
    ap.add_argument("--beam-bulk", type=int, default=0, choices=[0, 1],
                    help="--kernel 2: VR_OPT_BEAM_BULK (1 = cp.async.bulk row copies counted on an mbarrier)")
    ap.add_argument("--beam-stage-bytes", type=int, default=0,
                    help="--kernel 2: VR_OPT_BEAM_STAGE (0 = chosen per frame from the camera)")
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 1, 2],
                    help="VR_OPT_KERNEL: 0 = automatic, 1 = direct kernel, 2 = beam kernel (linear layout)")
    args = ap.parse_args()
    if args.layout is None:
        args.layout = "linear" if args.workload == "stream" else "tex"

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        line = run_reference(args, rank)
        if line is not None:
            print(json.dumps(line), flush=True)
        return 0

    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    line = (run_stream if args.workload == "stream" else run_ours)(args, rank, world, local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
