#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 spectral-cube ray caster.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload all|config1|config0|config2|config4|stream] [--layout tex|linear]

Metric (BASELINE.json): Gsamples/s (and frames/s) at 1920x1080 PER CUBE SIZE, with the fraction of the bounding
roofline (HBM for the in-core cubes, the host link for the out-of-core one).  The default run (--workload all) therefore
renders three cubes in sequence and prints ONE JSON line (rank 0):

  configs[1]  512x512x1024 (1 GiB), 8 orbit views, step 0.5, EA + MIP       -- issue-bound (4 samples per voxel)
  configs[2]  2048^3 (32 GiB), 1920x1080, 8 orbit views, step 1.0, EA + MIP -- HBM-bound; the HEADLINE: `value`,
              `ms_per_step`, `roofline`, `e2e`, `cpu_baseline` are this cube's (the largest in-HBM 1080p cube)
  configs[3]  out-of-core: 512^3-cell bricks streamed from pinned host memory (the 4096^3 cube needs 256 GiB of
              host memory; the largest brick grid that fits this host stands in, said beside the number)

each with its own entry under `per_config` (value, ms_per_step, frames_per_s, roofline, e2e).  One "step" = one pass
of the hot path over one batch = all views x {EA, MIP} of that cube.  Inputs are synthetic (vr_inputs), generated on
the GPU.  `value` is device-resident throughput, `e2e` the same metric through the C ABI with HOST buffers (cube
upload from pinned host memory + frames copied back to pinned host memory inside the timed region).
N > 1 (torchrun): the path does not shard ("replicas only"): every rank renders its own replica of
the workload; value = total samples / max time.
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

# Algorithmic work per sample, from the numerical contract: mandatory fp32/int lane-operations of
# S4-S8 (EA) and S4-S6+S9 (MIP), and how many of them can share a packed instruction (Blackwell FFMA2 / FADD2 retire two
# independent binary32 operations per lane and clock): the ALU peak is restated for that share, so that no kernel --
# paired or not -- can pass 1.0 ("ALU peak").
LANE_OPS_PER_SAMPLE = {EA: 80, MIP: 55}
PAIRABLE_OPS_PER_SAMPLE = {EA: 30, MIP: 22}
LANES_PER_SM = 128
PCIE_NOMINAL_GBS = 63.0                 # PCIe Gen5 x16, one direction

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel come from the committed ncu
# captures (`ncu --set full` summaries under profiles/), parsed at run time; a (workload, layout, kernel) without a
# capture reports null
TRAFFIC_PROFILES = {("config1", "tex", "raycast_kernel"): "profiles/r01b_tex_mip_views012.md",
                    ("config1", "linear", "raycast_kernel"): "profiles/r01a_linear_mip_view0.md"}


def traffic_from_profile(workload, layout, kernel_name):
    """(bytes per launch or None, source text): dram read + write of the kernel's ncu capture, mean over its launches."""
    rel = TRAFFIC_PROFILES.get((workload, layout, kernel_name))
    if rel is None or not os.path.exists(os.path.join(ROOT, rel)):
        return None, "no ncu capture of this (workload, layout, kernel) is committed (GPU access closed since round 1)"
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot = {}
    for ln in open(os.path.join(ROOT, rel)):
        f = ln.split()
        if len(f) >= 3 and f[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and f[-1] in unit:
            try:
                vals = [float(x) for x in f[1:-1]]
            except ValueError:
                continue
            if len(vals) >= len(tot.get(f[0], [])):          # the table with most launches wins
                tot[f[0]] = [x * unit[f[-1]] for x in vals]
    if len(tot) != 2:
        return None, f"{rel}: no dram__bytes lines found"
    return (sum(tot["dram__bytes_read.sum"]) / len(tot["dram__bytes_read.sum"])
            + sum(tot["dram__bytes_write.sum"]) / len(tot["dram__bytes_write.sum"])), f"{rel} (ncu --set full, dram read + write, mean over the captured launches)"


# the out-of-core workload's shape and the CPU baseline's sample (module level so that the no-GPU dry run of
# tests/test_bench_dryrun.py can shrink them; nothing else changes them)
STREAM_SHAPE = dict(brick=512, W=1920, H=1080, budget=None)
CPU_BASELINE = dict(n_tiles=64, tile=128, budget_s=20.0)

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


def alu_peak_tops(n_sm, sm_max_mhz, mode):
    """Contract lane-operations per second the SMs can retire at most: one instruction per lane and clock, and the
    pairable operations of the contract two to an instruction."""
    ops, pair = LANE_OPS_PER_SAMPLE[mode], PAIRABLE_OPS_PER_SAMPLE[mode]
    return n_sm * LANES_PER_SM * sm_max_mhz * 1e6 / 1e12 * ops / (ops - pair / 2.0)


def resident_roofline(workload, layout, kernel_name, nvox, W, H, n_sm, pk, mip_ms, ea_ms, mip_samples, ea_samples):
    """The `roofline` object of a resident-cube bench line (pure arithmetic; tests/test_bench_cpu.py)."""
    alu_peak = alu_peak_tops(n_sm, pk["sm_max_mhz"], MIP)                   # T lane-ops/s
    # dominant kernel: the MIP ray caster (no early termination, every sample evaluated)
    achieved = mip_samples * LANE_OPS_PER_SAMPLE[MIP] / (mip_ms * 1e-3) / 1e12
    hbm_bytes = nvox * 4 + H * W * 16             # every voxel once + the image
    alu = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "Tlane-op/s", "frac": achieved / alu_peak,
           "peak_source": f"{n_sm} SMs x {LANES_PER_SM} fp32 lanes x {pk['sm_max_mhz']:.0f} MHz x "
                          f"{LANE_OPS_PER_SAMPLE[MIP]}/({LANE_OPS_PER_SAMPLE[MIP]} - {PAIRABLE_OPS_PER_SAMPLE[MIP]}/2) "
                          "(pairable operations two to an FFMA2 / FADD2; DESIGN.md Sec. 6)",
           "lane_ops_per_sample": LANE_OPS_PER_SAMPLE[MIP]}
    hbm = {"bound": "hbm", "achieved": hbm_bytes / (mip_ms * 1e-3) / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
           "frac": hbm_bytes / (mip_ms * 1e-3) / 1e9 / pk["hbm_gbs"], "algorithmic_bytes_per_launch": hbm_bytes,
           "peak_source": pk["source"]}
    # the binding roofline is the one with the longer ideal time for this workload
    t_alu = mip_samples * LANE_OPS_PER_SAMPLE[MIP] / (alu_peak * 1e12)
    t_hbm = hbm_bytes / (pk["hbm_gbs"] * 1e9)
    binding, other = (hbm, alu) if t_hbm > t_alu else (alu, hbm)
    traffic, traffic_source = traffic_from_profile(workload, layout, kernel_name)
    ea_peak = alu_peak_tops(n_sm, pk["sm_max_mhz"], EA)
    roofline = dict(binding)
    roofline.update({
        "kernel": f"{kernel_name}<MIP, layout={layout}>",
        "traffic": traffic, "traffic_source": traffic_source,
        "avg_launch_ms": mip_ms, "units_per_launch": mip_samples,
        "ideal_ms": {"alu": t_alu * 1e3, "hbm": t_hbm * 1e3},
        "ea": {"avg_launch_ms": ea_ms, "units_per_launch": ea_samples,
               "achieved": ea_samples * LANE_OPS_PER_SAMPLE[EA] / (ea_ms * 1e-3) / 1e12,
               "frac": ea_samples * LANE_OPS_PER_SAMPLE[EA] / (ea_ms * 1e-3) / 1e12 / ea_peak,
               "note": "EA frame against the ALU roofline (80 lane-ops per sample); early termination leaves most voxels untouched"},
        other["bound"]: other})
    return roofline


# ---------------------------------------------------------------------------------
def run_resident(args, wlname, rank, world, local_rank, with_cpu_baseline):
    """One resident-cube workload -> its bench line (rank 0) or None."""
    import torch
    import paper_1001_2049_b200 as vr
    import vr_inputs as vi

    vr.lib()                                   # fail loudly if libvr.so is missing
    wl = WORKLOADS[wlname]
    spec = vi.CONFIGS[wl["config"]]
    W, H, step = wl["W"], wl["H"], wl["step"]
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    lut, vmin, vmax = get_lut(vi, wl["lut"])
    views = get_views(vi, wl["views"], spec.dims)
    modes = [EA, MIP]
    frames_per_step = len(views) * len(modes)
    nvox = int(np.prod(spec.dims))
    layout = args.layout or "tex"

    # ---- inputs, resident in HBM before the timed region -------------------------
    Vd = vi.make_cube(spec, device=dev)
    vol = vr.Volume(spec.dims, device=local_rank, layout=LAYOUTS[layout])
    vol.set_option(vr.VR_OPT_KERNEL, args.kernel)
    if args.kernel == 2:
        vol.set_option(vr.VR_OPT_BEAM_STAGES, args.beam_stages)
        vol.set_option(vr.VR_OPT_BEAM_STAGE, args.beam_stage_bytes)
        vol.set_option(vr.VR_OPT_BEAM_BULK, args.beam_bulk)
    vol.upload(Vd)
    vol.set_transfer_function(lut, vmin, vmax)
    out = torch.empty((H, W, 4), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev)

    # ---- variant choice (untimed): vr_autotune times the direct kernel's variants on one MIP frame ----------
    tuned = None
    if args.kernel != 2:
        if args.pipeline >= 0:
            vol.set_option(vr.VR_OPT_PIPELINE, args.pipeline)
            vol.set_option(vr.VR_OPT_TILE_ORDER, max(args.tile_order, 0))
            vol.set_option(vr.VR_OPT_REUSE, max(args.reuse, 0))
        elif not args.no_autotune:
            tuned = vol.autotune(views[len(views) // 2], W, H, step, MIP, out=out)

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
    st = vol.stats()
    kernel_name = {1: "raycast_kernel", 2: "raycast_beam_kernel", 3: "raycast_pipe_kernel", 4: "raycast_reuse_kernel"}[st["kernel"]]
    beam_stage = st.get("beam_stage_bytes", 0) if kernel_name == "raycast_beam_kernel" else None

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

    # ---- the variants side by side (untimed region, rank 0): mean MIP frame of every (pipeline, tile order) --------
    variants = None
    if rank == 0 and args.kernel != 2 and not args.no_variants:
        variants = {}
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for order in (0, 1):
            for depth, reuse, name in ((1, 1, "pipeline1"), (2, 1, "pipeline2"), (4, 1, "pipeline4"), (1, 2, "reuse")):
                vol.set_option(vr.VR_OPT_PIPELINE, depth)
                vol.set_option(vr.VR_OPT_REUSE, reuse)
                vol.set_option(vr.VR_OPT_TILE_ORDER, order)
                vol.render(views[0], W, H, step, MIP, out=out)
                a.record(stream)
                for cam in views:
                    vol.render(cam, W, H, step, MIP, out=out)
                b.record(stream)
                torch.cuda.synchronize(dev)
                variants[f"{name}_tiles{order}"] = a.elapsed_time(b) / len(views)
        # back to the configuration that was timed
        if tuned is not None:
            vol.set_option(vr.VR_OPT_PIPELINE, tuned[0])
            vol.set_option(vr.VR_OPT_TILE_ORDER, tuned[1])
            vol.set_option(vr.VR_OPT_REUSE, tuned[2])
        elif args.pipeline >= 0:
            vol.set_option(vr.VR_OPT_PIPELINE, args.pipeline)
            vol.set_option(vr.VR_OPT_TILE_ORDER, max(args.tile_order, 0))
            vol.set_option(vr.VR_OPT_REUSE, max(args.reuse, 0))
        else:
            vol.set_option(vr.VR_OPT_PIPELINE, 0)
            vol.set_option(vr.VR_OPT_TILE_ORDER, 0)
            vol.set_option(vr.VR_OPT_REUSE, 0)

    # ---- A2: the min/max table of this cube, one pass over the voxels (rank 0, untimed region) -----------------------
    minmax_ms = None
    if rank == 0 and not args.no_variants:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(2):
            # an upload marks the table stale; a linear cube "uploaded" from its own storage is left where it is
            if layout == "linear":
                vr.vr_volume_upload_bricks(vol.handle, [(0, 0, 0)], [spec.dims], [vol.storage.data_ptr()], 1, stream.cuda_stream)
            else:
                vol.upload(Vd)
            torch.cuda.synchronize(dev)
            a.record(stream)
            vol.minmax()
            b.record(stream)
            torch.cuda.synchronize(dev)
            minmax_ms = a.elapsed_time(b) if minmax_ms is None else min(minmax_ms, a.elapsed_time(b))

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
        vol.close()
        return None

    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    pk = peaks()
    roofline = resident_roofline(wlname, layout, kernel_name, nvox, W, H, n_sm, pk,
                                 float(np.mean(launch_ms[MIP])), float(np.mean(launch_ms[EA])),
                                 samples[MIP] / len(views), samples[EA] / len(views))
    if variants is not None:
        roofline["variants_mip_ms"] = variants
    if minmax_ms is not None:
        roofline["minmax_kernel"] = {"ms": minmax_ms, "bytes": nvox * 4, "achieved_gbs": nvox * 4 / (minmax_ms * 1e-3) / 1e9,
                                     "frac_of_hbm": nvox * 4 / (minmax_ms * 1e-3) / 1e9 / pk["hbm_gbs"],
                                     "note": "A2: min/max table of the cube in one pass (kernel + 256 KB table read back), best of 2"}

    line = {
        "metric": "Gsamples/s", "value": samples_per_step * world / (ms_per_step * 1e-3) / 1e9,
        "unit": "Gsamples/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{wl['config']}] {spec.name}: {spec.dims[0]}x{spec.dims[1]}x{spec.dims[2]} f32, "
                               f"{W}x{H}, {len(views)} views x (EA+MIP), step {step}",
                   "layout": layout, "frames_per_step": frames_per_step, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (cube %.2f GiB vs 126 MB L2); no flush" % (nvox * 4 / 2 ** 30),
                   "kernel": kernel_name, "pipeline_depth": st["pipeline_depth"],
                   "autotuned": {"pipeline": tuned[0], "tile_order": tuned[1], "reuse": tuned[2]} if tuned else None,
                   **({"beam_stages": args.beam_stages, "beam_bulk": args.beam_bulk, "beam_stage_bytes_last_frame": beam_stage}
                      if beam_stage is not None else {})},
        "frames_per_s": frames_per_step * world / (ms_per_step * 1e-3),
        "samples_per_step": samples_per_step, "rays_hit_per_step": rays,
        # nominal = no early termination, no skipping: MIP evaluates every sample of every ray, so EA's nominal
        # count is MIP's ("report also nominal samples")
        "nominal_samples_per_step": 2 * samples[MIP],
        "gpu_launches": frames_per_step * args.steps,
        "e2e": e2e, "roofline": roofline, "clocks": clocks,
    }
    if with_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(Vd.cpu().numpy(), lut, vmin, vmax, views, W, H, step, budget_s=CPU_BASELINE["budget_s"])
    vol.close()
    del Vd, out
    torch.cuda.empty_cache()
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
    55 % of MemAvailable, at most 40 GB in the default run) stands in for it, same bricks / seed / generator
    (DESIGN.md Sec. 4).  Three regimes, same frames:
      link    every brick in the frustum crosses the host link every frame (3 slots, no culling, no cache): the clean
              host-link roofline measurement -- the line's `value` and `roofline`;
      culled  VR_OPT_STREAM_CULL: bricks no ray can still draw from stay on the host;
      cached  culling + the slot cache with a pool of 55 % of the bricks (the share of a 275 GB brick store that a
              150 GB pool holds), the views in orbit order."""
    import torch
    import paper_1001_2049_b200 as vr
    import vr_inputs as vi

    vr.lib()
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    B, W, H, step = STREAM_SHAPE["brick"], STREAM_SHAPE["W"], STREAM_SHAPE["H"], 0.5
    budget = args.ooc_gb * 1e9 if args.ooc_gb > 0 else 0.55 * mem_available_bytes() / max(1, world)
    if args.workload == "all" and args.ooc_gb <= 0:
        budget = min(budget, 40e9)
    if STREAM_SHAPE["budget"]:
        budget = STREAM_SHAPE["budget"]
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

    # host-link peak on this box: one brick-sized pinned copy, best of 5 (a plain cudaMemcpyAsync through torch)
    probe = torch.empty(store[0].array.size, dtype=torch.float32, device=dev)
    src = torch.from_numpy(store[0].array).reshape(-1)
    link = 0.0
    for _ in range(5):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        probe.copy_(src, non_blocking=True)
        b.record()
        torch.cuda.synchronize(dev)
        link = max(link, probe.numel() * 4 / (a.elapsed_time(b) * 1e-3) / 1e9)
    del probe

    layout = args.layout or "linear"
    out = torch.empty((H, W, 4), dtype=torch.float32, device=dev)
    h_img = torch.empty((H, W, 4), dtype=torch.float32, pin_memory=True)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    def open_volume(n_slots, cull, cache):
        vol = vr.Volume(spec.dims, host_brick=B, n_slots=n_slots, device=local_rank, layout=LAYOUTS[layout])
        vol.vr_volume_upload_bricks([(o, pb) for (o, _), pb in zip(boxes, store)])
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_STREAM_CULL, cull)
        vol.set_option(vr.VR_OPT_STREAM_CACHE, cache)
        return vol

    def timed_frames(vol, steps, warm):
        """Warm-up passes, `steps` timed passes over the frames (nothing but vr_render in the timed region), then one
        untimed pass that reads the per-frame statistics -> dict: ms (timed total) and per-PASS sums of h2d bytes,
        bricks streamed / cached / culled and the link-busy time."""
        def one_pass(stats_into=None):
            for m in modes:
                for cam in views:
                    vol.render(cam, W, H, step, m, out=out)
                    if stats_into is not None:
                        st = vol.stats()          # waits for the frame: its copy timings
                        stats_into["h2d"] += st["h2d_bytes"]; stats_into["streamed"] += st["bricks_streamed"]
                        stats_into["cached"] += st["bricks_cached"]
                        stats_into["culled"] += st["bricks_culled"] + st["bricks_empty"]
                        stats_into["h2d_ms"] += st["h2d_ms"]; stats_into["frame_ms"] += st["frame_ms"]
        for _ in range(warm):
            one_pass()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(steps):
            one_pass()
        e1.record(stream)
        barrier()
        acc = dict(h2d=0, streamed=0, cached=0, culled=0, h2d_ms=0.0, frame_ms=0.0)
        one_pass(acc)
        barrier()
        acc["ms"] = e0.elapsed_time(e1)
        return acc

    # ---- regime "link": the clean host-link roofline ---------------------------------------------------------------
    vol = open_volume(args.slots, 0, 0)
    vol.set_option(vr.VR_OPT_COUNT, 1)               # samples per step: one counting pass (doubles as warm-up)
    samples = {EA: 0, MIP: 0}
    for m in modes:
        for cam in views:
            vol.render(cam, W, H, step, m, out=out)
            samples[m] += vol.stats()["samples"]
    vol.set_option(vr.VR_OPT_COUNT, 0)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    acc = timed_frames(vol, args.steps, max(0, args.warmup - 1))
    clocks = sampler.stop() if rank == 0 else None
    total_ms = acc["ms"]

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

    # ---- regimes "culled" and "cached" (rank 0; same frames, bitwise the same pixels: tests/parity_cases.py) -----------
    regimes = {}
    if rank == 0 and not args.no_variants:
        try:
            vol = open_volume(args.slots, 1, 0)
            a = timed_frames(vol, 1, 2)              # warm-up frames also measure the bricks' value ranges
            vol.close()
            nfr = frames_per_step
            regimes["culled"] = {"ms_per_frame": a["ms"] / nfr, "frames_per_s": nfr / (a["ms"] * 1e-3),
                                 "bricks_streamed_per_frame": a["streamed"] / nfr, "bricks_culled_per_frame": a["culled"] / nfr,
                                 "h2d_gbs_while_copying": a["h2d"] / max(a["h2d_ms"], 1e-9) / 1e6,
                                 "link_busy_fraction_of_frame": a["h2d_ms"] / max(a["frame_ms"], 1e-9)}
            pool = max(3, int(0.55 * len(boxes)))
            free, _ = torch.cuda.mem_get_info()
            pool = max(3, min(pool, int(0.8 * free / (4 * (B + 1) ** 3))))
            vol = open_volume(pool, 1, 1)
            a = timed_frames(vol, 1, 2)
            vol.close()
            regimes["cached"] = {"slots": pool, "ms_per_frame": a["ms"] / nfr, "frames_per_s": nfr / (a["ms"] * 1e-3),
                                 "bricks_streamed_per_frame": a["streamed"] / nfr, "bricks_cached_per_frame": a["cached"] / nfr,
                                 "bricks_culled_per_frame": a["culled"] / nfr,
                                 "hit_rate": a["cached"] / max(1, a["cached"] + a["streamed"])}
        except Exception as ex:                        # the link line stands on its own
            regimes["error"] = repr(ex)
    for pb in store:
        pb.close()
    del out, h_img
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    ms_per_step = total_ms / args.steps
    samples_per_step = samples[EA] + samples[MIP]
    n_frames = frames_per_step * args.steps
    h2d_per_frame = acc["h2d"] / frames_per_step                    # (the statistics are those of one pass over the frames)
    achieved = acc["h2d"] * args.steps / (total_ms * 1e-3) / 1e9
    return {
        "metric": "Gsamples/s", "value": samples_per_step * world / (ms_per_step * 1e-3) / 1e9, "unit": "Gsamples/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[3] out-of-core, scaled to this host: {spec.dims[0]}x{spec.dims[1]}x{spec.dims[2]} f32 "
                               f"({store_bytes / 2 ** 30:.1f} GiB pinned, {len(boxes)} bricks of {B}^3 cells; the 4096^3 cube needs 256 GiB), "
                               f"{W}x{H}, {len(views)} views x (EA+MIP), step {step}",
                   "layout": layout, "frames_per_step": frames_per_step, "device_slots": n_slots,
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "every brick crosses the host link every frame; nothing is cached between frames",
                   "generate_s": gen_s},
        "frames_per_s": frames_per_step * world / (ms_per_step * 1e-3),
        "samples_per_step": samples_per_step, "bricks_streamed_per_frame": acc["streamed"] / frames_per_step,
        "gpu_launches": int(acc["streamed"] * args.steps + n_frames),
        "e2e": {"value": samples_per_step * world / e2e_s / 1e9, "unit": "Gsamples/s",
                "h2d_bytes_per_step": int(h2d_per_frame * frames_per_step), "d2h_bytes_per_step": frames_per_step * H * W * 16,
                "ms_per_step": e2e_s * 1e3, "timer": "host wall clock around vr_render_host x frames + stream sync"},
        "roofline": {"bound": "host_link", "kernel": "cudaMemcpyAsync H2D of bricks (copy stream) overlapped with raycast_kernel<BRICK>",
                     "achieved": achieved, "peak": link, "unit": "GB/s", "frac": achieved / link, "traffic": None,
                     "peak_source": "measured in this run: brick-sized pinned H2D copy, best of 5",
                     "frac_of_pcie_nominal": achieved / PCIE_NOMINAL_GBS,
                     "pcie_nominal_gbs": PCIE_NOMINAL_GBS,
                     "h2d_gbs_while_copying": acc["h2d"] / max(acc["h2d_ms"], 1e-9) / 1e6,
                     "link_busy_fraction_of_frame": acc["h2d_ms"] / max(acc["frame_ms"], 1e-9),
                     "algorithmic_bytes_per_launch": h2d_per_frame, "avg_launch_ms": total_ms / n_frames},
        "regimes": regimes,
        "clocks": clocks,
    }


# ---------------------------------------------------------------------------------
def cpu_baseline(V, lut, vmin, vmax, views, W, H, step, budget_s):
    """The oracle as it stands, on the host cores, on a bounded sample of the workload."""
    import oracle
    import vr_inputs as vi
    cores = os.cpu_count()
    ij = vi.tile_subset(W, H, n_tiles=CPU_BASELINE["n_tiles"], tile=CPU_BASELINE["tile"], seed=0)   # about half of a 1080p frame: 10-30 s on 16 cores
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
            "sample": f"{CPU_BASELINE['n_tiles']} tiles of {CPU_BASELINE['tile']}x{CPU_BASELINE['tile']} pixels ({len(ij)} rays) of views {done}, EA + MIP, "
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


HEADLINE_ORDER = ["config2", "config1", "stream"]       # the first of these that ran carries the top-level keys
SUB_KEYS = ["value", "unit", "ms_per_step", "frames_per_s", "samples_per_step", "nominal_samples_per_step", "config",
            "roofline", "e2e", "gpu_launches", "clocks", "regimes", "bricks_streamed_per_frame", "error"]


def assemble(lines, n_gpus, steps, warmup):
    """The one JSON line of the default run: the headline workload's keys at the top, every workload under per_config.
    lines: {name: bench line or {"error": ...}}."""
    head = next((n for n in HEADLINE_ORDER if n in lines and "error" not in lines[n]), None)
    per = {n: {k: ln[k] for k in SUB_KEYS if k in ln} for n, ln in lines.items()}
    if head is None:
        return {"metric": "Gsamples/s", "value": None, "unit": "Gsamples/s", "n_gpus": n_gpus, "steps": steps, "warmup": warmup,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "none completed"}, "per_config": per, "gpu_launches": 0}
    line = dict(lines[head])
    line["config"] = dict(line["config"])
    line["config"]["headline"] = (f"{head}: the largest in-HBM cube at 1920x1080 (HBM-bound); the other cube sizes of the metric are "
                                  "under per_config" if head == "config2" else f"{head} (configs[2] did not complete: see per_config)")
    line["per_config"] = per
    line["gpu_launches"] = sum(int(ln.get("gpu_launches", 0)) for ln in lines.values() if "error" not in ln)
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="all", choices=["all"] + sorted(WORKLOADS) + ["stream"],
                    help="all (default) = configs[1], configs[2] and the out-of-core stand-in in one line, headline configs[2]")
    ap.add_argument("--ooc-gb", type=float, default=0.0, help="stream: pinned brick store budget (0 = 55%% of MemAvailable; "
                                                              "at most 40 GB in the default run)")
    ap.add_argument("--slots", type=int, default=3, help="stream: device slots")
    ap.add_argument("--stream-views", type=int, default=2, help="stream: orbit views per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-autotune", action="store_true", help="keep VR_OPT_PIPELINE / VR_OPT_TILE_ORDER at their defaults")
    ap.add_argument("--no-variants", action="store_true", help="skip the untimed side measurements (variants, min/max, regimes)")
    ap.add_argument("--pipeline", type=int, default=-1, choices=[-1, 0, 1, 2, 4], help="VR_OPT_PIPELINE (-1 = vr_autotune)")
    ap.add_argument("--tile-order", type=int, default=-1, choices=[-1, 0, 1], help="VR_OPT_TILE_ORDER (with --pipeline)")
    ap.add_argument("--reuse", type=int, default=-1, choices=[-1, 0, 1, 2], help="VR_OPT_REUSE (with --pipeline)")
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

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world and not (args.impl == "reference" and world == 1):
        # one process per GPU: N > 1 is launched by torchrun (python -m torch.distributed.run --nproc-per-node N bench.py --gpus N)
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}; launch {args.gpus} ranks with "
                         "python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 bench.py --gpus N\n")
        return 2

    if args.impl == "reference":
        if args.workload == "all":
            args.workload = "config2"        # the headline workload of the default run
        line = run_reference(args, rank)
        if line is not None:
            print(json.dumps(line), flush=True)
        return 0

    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        backend = os.environ.get("VR_BENCH_DIST_BACKEND", "nccl")      # (the no-GPU dry run of the tests uses gloo)
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        else:
            dist.init_process_group(backend)
    if args.workload == "all":
        lines = {}
        for name in ("config1", "config2", "stream"):
            try:
                if name == "stream":
                    ln = run_stream(args, rank, world, local_rank)
                else:
                    ln = run_resident(args, name, rank, world, local_rank,
                                      with_cpu_baseline=(name == "config2" and not args.no_cpu_baseline))
            except Exception as ex:              # one cube failing must not take the others' numbers with it
                import traceback
                sys.stderr.write(f"bench.py: workload {name} failed:\n{traceback.format_exc()}\n")
                ln = {"error": repr(ex)}
                try:
                    import torch
                    torch.cuda.empty_cache()
                except Exception:
                    pass
            if ln is not None:
                lines[name] = ln
        line = assemble(lines, world, args.steps, args.warmup) if rank == 0 else None
    elif args.workload == "stream":
        line = run_stream(args, rank, world, local_rank)
    else:
        line = run_resident(args, args.workload, rank, world, local_rank, with_cpu_baseline=not args.no_cpu_baseline)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
