#!/usr/bin/env python
"""bench.py — frame throughput of the deferred hair pipeline on the north-star workload.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

A "step" is one frame = one pass of the whole hot path (LOD -> scan -> generate -> clear + raster
-> shade -> filter) over BASELINE.json configs[3]: the five-groom scene, 483 000 strands,
3840x2160, 1 spp, per-groom LOD lambda {4.0, 5.5, 2.0, 2.8, 3.0} (synthetic, seeded).
`value` = segments rasterised per second (whole job); `ms_per_step` = frame ms.
N > 1 = N independent replicas of the same frame ("replicas only": north_star excludes sharding).

Prints ONE JSON line. `--impl reference` times the CPU oracle instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Gsegments/s at 4K, 483k strands (frame ms = ms_per_step)"
UNIT = "Gsegments/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_counters():
    """Per-stage counters of one production frame from the committed `ncu --set full` capture (dram bytes, warp
    instructions, lts throughput, issue-active; profiles/r3_ncu_stage_counters.csv written by
    `python -m paper_2607_04230_b200.ncu_summary`) — never typed in here. The file carries the sha256 of csrc/ at capture
    time; `fresh` says whether the sources bench.py runs on still have it (a kernel edit makes the capture stale)."""
    from paper_2607_04230_b200 import ncu_summary
    p = os.path.join(ROOT, "profiles", "r3_ncu_stage_counters.csv")
    if not os.path.exists(p):
        return {}, {"source": None, "fresh": None}
    stages, sha = ncu_summary.read_stage_csv(p)
    now = ncu_summary.source_hash()
    return stages, {"source": "profiles/r3_ncu_stage_counters.csv (see r3_ncu_stage_counters.md)", "captured_src_sha256": sha,
                    "current_src_sha256": now, "fresh": sha == now,
                    "label": "fresh" if sha == now else "stale: csrc/ changed since the capture"}


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(index), "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL,
                                      text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def scene_for(args):
    from paper_2607_04230_b200 import synth
    return synth.config(args.config, scale=args.scale, res_scale=args.res_scale)


# ------------------------------------------------------------------------------- oracle legs
def oracle_sample(config: int, scale: float, res_scale: float):
    """One oracle frame (all of O1-O7) on a bounded sample; returns (seconds, segments, description)."""
    import oracle
    from paper_2607_04230_b200 import synth
    sc = synth.config(config, scale=scale, res_scale=res_scale)
    f = oracle.Frame(sc["grooms"])
    stage_s = {}

    def timed(name, fn, *a):
        t = time.perf_counter()
        r = fn(*a)
        stage_s[name] = time.perf_counter() - t
        return r

    t0 = time.perf_counter()
    timed("O1_lod_scan", f.lod, sc["camera"], sc["lam"])
    timed("O2_generate", f.generate)
    cnt = timed("O4_raster_resolve", f.raster, sc["camera"], sc["params"])
    timed("O6_shade", f.shade, sc["camera"], sc["params"])
    timed("O7_filter", f.filter, sc["camera"], sc["params"])
    dt = time.perf_counter() - t0
    oracle_sample.last_stage_seconds = stage_s
    n_seg = int(f.n_vertices - f.n_strands)
    desc = (f"config {config} with strand counts x{scale} ({synth.n_strands(sc)} strands, {f.n_strands} after LOD, "
            f"{n_seg} segments) at {sc['camera']['width']}x{sc['camera']['height']}, one full frame O1-O7")
    return dt, n_seg, desc, cnt


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, single-threaded, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    # a bounded sample of the metric's workload at its own resolution: 2 % of every groom's strands at 4K (about 3 s per
    # step on the GPU box's host), fewer strands when many steps are asked for so that the run ends within minutes
    n_runs = max(args.steps + args.warmup, 1)
    scale, res_scale = (0.02 if n_runs <= 40 else max(0.02 * 40.0 / n_runs, 0.002)), 1.0
    for _ in range(args.warmup):
        oracle_sample(args.config, scale, res_scale)
    t, seg, desc = 0.0, 0, ""
    for _ in range(args.steps):
        dt, n_seg, desc, _ = oracle_sample(args.config, scale, res_scale)
        t += dt
        seg += n_seg
    val = seg / t / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64/f32",
            "data": "synthetic", "config": {"workload": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                             "stage_seconds_last_step": getattr(oracle_sample, "last_stage_seconds", None),
                             "cpu_model": cpu_model(), "host_cores_available": os.cpu_count()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------- CUDA arm
def run_cuda(args):
    import numpy as np
    import torch
    from paper_2607_04230_b200 import binding, replicas, synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"

    sc = scene_for(args)
    cam, lam = sc["camera"], sc["lam"]
    W, H = cam["width"], cam["height"]
    h = binding.Hair(local_rank)
    for g in sc["grooms"]:
        h.mesh_upload(g)
    gb, rgb = h.alloc_outputs(W, H)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- algorithmic counts of the frame (untimed, instrumented kernels)
    h.set_render_params(sc["params"], flags=binding.FLAG_COUNTERS)
    h.render(cam, lam, gb, rgb)
    cnt = h.stats()
    # unique vertices the shading gathers touch (neighbouring pixels share them): v_{j-1} .. v_{j+2} of every centre word
    G0 = gb[..., 0].reshape(-1)
    G0 = G0[(G0 & 0xFFFFFFFFFF) != 0xFFFFFFFFFF]
    sid_j = (G0 >> 9) & 0x7FFFFFFF  # sid << 7 | j
    n_unique_vertices = int(torch.unique(torch.cat([sid_j - 1, sid_j, sid_j + 1, sid_j + 2])).numel())
    del G0, sid_j

    # ---- device-resident timing: K frames, one event pair, stage events inside the library
    h.set_render_params(sc["params"], flags=binding.FLAG_STAGE_TIMING)
    for _ in range(max(args.warmup, 3)):
        h.render(cam, lam, gb, rgb)
    h.stats()  # drain the warm-up stage timings
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        h.render(cam, lam, gb, rgb)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    st = h.stats()  # stage means over the timed frames
    ms_total = replicas.max_over_ranks(ms_total, dist, dev)
    ms_step = ms_total / args.steps
    n_seg = cnt["n_segments"]
    assert replicas.same_on_all_ranks(n_seg, dist, dev), "replicas rendered different frames"
    value = replicas.job_rate(n_seg, world, ms_step) / 1e9

    # ---- the same frames under camera motion (untimed for `value`): the depth ranges of the two-pass split and the
    # choice of passes are then one frame stale; a slow orbit + dolly, ~10 px of image motion per frame
    k_mov = max(8, min(args.steps, 64))
    for i in range(3):
        h.render(synth.moving_camera(cam, i), lam, gb, rgb)
    h.stats()
    barrier()
    e0.record()
    for i in range(k_mov):
        h.render(synth.moving_camera(cam, 3 + i), lam, gb, rgb)
    e1.record()
    barrier()
    ms_moving = e0.elapsed_time(e1) / k_mov
    st_mov = h.stats()

    # ---- two frames in flight: a second context on a second stream renders every other frame, so
    # frame i's shade + filter (FMA / XU-bound, L2 idle) can share the SMs with frame i+1's LOD / generate / raster
    # (L2-latency-bound, FMA pipe idle). Each context owns its scratch, so nothing is shared but the SMs; the frames are
    # the serial frame bit for bit (checked). Throughput only: a single frame's latency is ms_per_step or worse.
    h.set_render_params(sc["params"], flags=0)
    s1 = torch.cuda.current_stream()
    s2 = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(s2):
        h_b = binding.Hair(local_rank, stream=s2)
        for g in sc["grooms"]:
            h_b.mesh_upload(g)
        gb_b, rgb_b = h_b.alloc_outputs(W, H)
        h_b.set_render_params(sc["params"], flags=0)
    for _ in range(3):
        h.render(cam, lam, gb, rgb)
        h_b.render(cam, lam, gb_b, rgb_b)
    barrier()
    k_pipe = max(8, min(args.steps, 100)) // 2 * 2
    e_b = torch.cuda.Event()
    e0.record(s1)
    s2.wait_event(e0)
    for i in range(k_pipe // 2):
        h.render(cam, lam, gb, rgb)
        h_b.render(cam, lam, gb_b, rgb_b)
    e_b.record(s2)
    s1.wait_event(e_b)
    e1.record(s1)
    barrier()
    ms_pipelined = e0.elapsed_time(e1) / k_pipe
    pipelined_same = bool(torch.equal(gb, gb_b) and torch.equal(rgb, rgb_b))
    # the serial frame with the same flags (no stage events), for the comparison
    e0.record(s1)
    for _ in range(k_pipe):
        h.render(cam, lam, gb, rgb)
    e1.record(s1)
    barrier()
    ms_serial_noevents = e0.elapsed_time(e1) / k_pipe
    h_b.close()
    del gb_b, rgb_b

    # ---- end to end through the C ABI with HOST buffers: cage upload (pinned) + render + D2H of out_rgb, per step.
    # Headline: RGBA16F host output (HAIR_FLAG_RGB16F, written by the filter itself: 66 MB per 4K frame); the fp32 host
    # output (133 MB, PCIe-bound) is timed beside it.
    pinned = [(torch.from_numpy(np.ascontiguousarray(g["pos"])).pin_memory(),
               None if g["ao"] is None else torch.from_numpy(np.ascontiguousarray(g["ao"])).pin_memory())
              for g in sc["grooms"]]
    h2d = sum(p.numel() * 4 + (0 if a is None else a.numel() * 4) for p, a in pinned)

    def e2e_leg(dtype, flags, k_steps, with_gbuffer=False):
        h.set_render_params(sc["params"], flags=flags)
        hosts = [torch.empty((H, W, 4), dtype=dtype).pin_memory() for _ in range(2)]
        hosts_gb = [torch.empty((H, W, 2), dtype=torch.int64).pin_memory() for _ in range(2)] if with_gbuffer else [None, None]

        def step(i):
            # every step: this step's cages host -> device, the frame, this step's results device -> host. The copies
            # of step i run on the library's copy stream while step i+1 renders (hair_render_to_host_async).
            for gi, (p, a) in enumerate(pinned):
                h.mesh_update(gi, p, a)
            h.render_to_host_async(cam, lam, hosts[i % 2], hosts_gb[i % 2])

        for i in range(4):
            step(i)
        h.host_wait(-1)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        for i in range(k_steps):
            step(i)
        h.host_wait(-1)  # the last result is in host memory
        e1.record()
        barrier()
        ms = max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0)) / k_steps
        # the unpipelined call, for reference: one frame, copies inside the call
        t0 = time.perf_counter()
        for _ in range(5):
            for gi, (p, a) in enumerate(pinned):
                h.mesh_update(gi, p, a)
            h.render_to_host(cam, lam, hosts[0], hosts_gb[0])
        ms_sync = 1e3 * (time.perf_counter() - t0) / 5
        return ms, ms_sync, hosts[0].numel() * hosts[0].element_size() + (hosts_gb[0].numel() * 8 if with_gbuffer else 0)

    # Headline e2e: out_rgb as float32, the format hair_render declares (133 MB per 4K frame, PCIe-bound) — the number
    # comparable from round to round. Beside it: the RGBA16F output option (66 MB) and float32 + the G-buffer (265 MB).
    k_e2e = max(4, min(args.steps, 40))
    ms_e2e, ms_e2e_sync, d2h = e2e_leg(torch.float32, 0, k_e2e)
    ms_e2e16, ms_e2e16_sync, d2h16 = e2e_leg(torch.float16, binding.FLAG_RGB16F, k_e2e)
    ms_e2e_gb, ms_e2e_gb_sync, d2h_gb = e2e_leg(torch.float32, 0, max(4, k_e2e // 2), with_gbuffer=True)
    ms_e2e = replicas.max_over_ranks(ms_e2e, dist, dev)
    e2e_val = replicas.job_rate(n_seg, world, ms_e2e) / 1e9
    h.set_render_params(sc["params"], flags=0)

    # ---- the paper's sequential per-groom compositing, same scene, untimed leg
    for _ in range(3):
        h.render_sequential(cam, lam, None, None, gb, rgb)
    barrier()
    e0.record()
    for _ in range(10):
        h.render_sequential(cam, lam, None, None, gb, rgb)
    e1.record()
    barrier()
    ms_seq = e0.elapsed_time(e1) / 10

    # ---- SURVEY 8f NEXT-4 (last part): deep-opacity shadows, same scene, untimed leg: the maps of the
    # three lights at 1024^2 from the full grooms (483 k strands, LOD off), then frames shaded with HAIR_FLAG_SHADOWS
    lcams = synth.light_cameras(sc, 1024)
    h.shadow_build(lcams, 1e-4, 0.03)  # warm (allocations)
    barrier()
    e0.record()
    h.shadow_build(lcams, 1e-4, 0.03)
    e1.record()
    barrier()
    ms_dom_build = e0.elapsed_time(e1)
    h.set_render_params(sc["params"], flags=binding.FLAG_SHADOWS | binding.FLAG_STAGE_TIMING)
    for _ in range(3):
        h.render(cam, lam, gb, rgb)
    h.stats()
    barrier()
    e0.record()
    for _ in range(20):
        h.render(cam, lam, gb, rgb)
    e1.record()
    barrier()
    ms_dom_frame = e0.elapsed_time(e1) / 20
    st_dom = h.stats()
    h.shadow_clear()
    h.set_render_params(sc["params"], flags=0)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- rooflines: algorithmic work per frame / measured stage time, every peak measured in this run
    hbm_peak, hbm_src = peaks()
    words = torch.empty(W * H * 2, dtype=torch.int64, device=dev)
    n_ops = 1 << 28
    atom = {}
    for mode, name in ((0, "unique"), (1, "random"), (2, "hot1024")):
        h.atomic_microbench(mode, words, 1 << 24, 1024)  # warm
        ms = min(h.atomic_microbench(mode, words, n_ops, 1024) for _ in range(3))
        atom[name] = n_ops / (ms * 1e-3) / 1e9
    del words
    # 16-byte ld.global.cg of word pairs over the frame's own G-buffer, in the raster's access shapes (G pair loads / s)
    l2 = {}
    for mode, name in ((0, "row"), (1, "column"), (2, "random"), (5, "column_pairs")):
        h.l2_load_microbench(mode, gb, W, 32)  # warm
        l2[name] = max(n / (ms * 1e-3) / 1e9 for n, ms in (h.l2_load_microbench(mode, gb, W, 512) for _ in range(3)))
    n_px = W * H
    n_cons, n_cen, n_cons_y = cnt["n_atomics_cons"], cnt["n_atomics_center"], cnt["n_atomics_cons_ymajor"]
    n_at = n_cen + n_cons
    stages = {
        "generate": {"bound": "hbm", "ms": st["ms_generate"], "bytes": 16 * cnt["n_vertices"],
                     "note": "the G-buffer clear (16 B/px) runs beside LOD / scan / generate on the library's second stream "
                             "and is not in these bytes"},
        "raster": {"bound": "l2_load", "ms": st["ms_raster"], "pair_loads": n_cons, "hits": n_at,
                   "bytes": 16 * cnt["n_vertices"] + 8 * n_at},
        "shade": {"bound": "hbm", "ms": st["ms_shade"], "bytes": 16 * n_px + (16 + 64) * cnt["n_pixels_center"],
                  "bytes_unique_vertices": 16 * n_px + 16 * cnt["n_pixels_center"] + 16 * n_unique_vertices
                                           + 8 * cnt["n_strands_lod"]},
        "filter": {"bound": "hbm (nominal; ALU/issue in practice)", "ms": st["ms_filter"],
                   "bytes": 32 * n_px + 16 * cnt["n_pixels_center"]},
    }
    for k, s in stages.items():
        if s["ms"] > 0:
            s["GBps"] = s["bytes"] / (s["ms"] * 1e-3) / 1e9
            s["frac_hbm"] = s["GBps"] / hbm_peak
    sh = stages["shade"]
    sh["GBps_unique_vertices"] = sh["bytes_unique_vertices"] / (sh["ms"] * 1e-3) / 1e9
    sh["frac_hbm_unique_vertices"] = sh["GBps_unique_vertices"] / hbm_peak
    stages["lod_scan"] = {"bound": "latency", "ms": st["ms_lod"]}
    stages["clear"] = {"bound": "hbm", "ms": None, "bytes": 16 * n_px,
                       "note": "overlapped: runs on the library's second stream beside lod_scan + generate (not bracketed)"}
    # The raster (dominant): every pixel that passes the conservative predicate needs the existing word pair before
    # anything is known about its depth (read-before-atomic) = one 16-byte L2 load, the method's own
    # minimum. Lower bound of the time = x-major loads at the measured row rate + y-major loads at the column rate.
    ras = stages["raster"]
    l2_y = max(l2["column"], l2["column_pairs"])  # a y-major task requests the two minor-axis neighbours of a row together
    t_min_ms = ((n_cons - n_cons_y) / l2["row"] + n_cons_y / l2_y) / 1e9 * 1e3
    ras["Gpair_loads_per_s"] = n_cons / (ras["ms"] * 1e-3) / 1e9
    ras["Ghits_per_s"] = n_at / (ras["ms"] * 1e-3) / 1e9
    ras["frac_l2_load"] = t_min_ms / ras["ms"]
    ras["frac_l2_atomic_random"] = ras["Ghits_per_s"] / atom["random"]
    ncu, ncu_meta = ncu_counters()
    dom = max(("generate", "raster", "shade", "filter"), key=lambda k: stages[k]["ms"])
    d = stages[dom]
    sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
    n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    issue_peak = n_sm * 4 * sm_mhz * 1e6 / 1e9  # G warp instructions / s: one per scheduler (4 per SM) per clock
    for k in ("generate", "raster", "shade", "filter"):
        if k in ncu and stages[k]["ms"] > 0:
            stages[k]["warp_inst_ncu"] = ncu[k].get("warp_inst")
            stages[k]["frac_issue"] = ncu[k]["warp_inst"] / (stages[k]["ms"] * 1e-3) / 1e9 / issue_peak
            stages[k]["dram_bytes_ncu"] = ncu[k].get("dram_bytes")
            stages[k]["ncu_lts_throughput_pct"] = ncu[k].get("lts_throughput_pct")
            stages[k]["ncu_issue_active_pct"] = ncu[k].get("issue_active_pct")
    if dom == "raster":
        t_min_plain_ms = ((n_cons - n_cons_y) / l2["row"] + n_cons_y / l2["column"]) / 1e9 * 1e3
        views = {
            "survey_8d_l2_atomic": {
                "frac": ras["frac_l2_atomic_random"], "binds": False, "hits_per_s_G": ras["Ghits_per_s"],
                "peak_random_RED_G_per_s": atom["random"], "frac_of_coalesced_RED": ras["Ghits_per_s"] / atom["unique"],
                "note": "SURVEY 8(d) as written: predicate-true hits (n_atomics_cons + n_atomics_center) / time over the "
                        "measured random RED.MIN.64 rate. Far above 1: read-before-atomic sends only n_atomics_issued of "
                        "the hits to L2 as atomics, so this ceiling does not bind this design"},
            "issued_atomics": {"frac": cnt["n_atomics_issued"] / (ras["ms"] * 1e-3) / 1e9 / atom["random"],
                               "issued_Gatom_per_s": cnt["n_atomics_issued"] / (ras["ms"] * 1e-3) / 1e9, "binds": False},
            "l2_pair_load_model": {
                "frac_column_pairs": ras["frac_l2_load"], "frac_plain_column": t_min_plain_ms / ras["ms"], "binds": False,
                "note": "builder-defined: one 16-byte ld.global.cg per conservative-predicate-true pixel, x-major at the "
                        "measured row rate, y-major at the column rate; the two y-major denominators (plain column walk / "
                        "the two minor-axis neighbours requested together) bracket it. ncu's lts__throughput of the two "
                        "passes (below) says L2 is near half of its ceiling: not the binding resource either",
                "rates_G_pair_loads_per_s": l2},
            "ncu_capture": {"lts_throughput_pct": ncu.get("raster", {}).get("lts_throughput_pct"),
                            "issue_active_pct": ncu.get("raster", {}).get("issue_active_pct"),
                            "order": "near pass / k_hiz / far pass"},
        }
        wi = ncu.get("raster", {}).get("warp_inst")
        roofline = {"kernel": "k_raster", "bound": "alu",
                    "bound_detail": "warp-instruction issue slots, latency-limited: the pixel loop's integer / fp32 / LSU "
                                    "instructions, not bytes and not atomics (DESIGN.md 7.5)",
                    "achieved": None if wi is None else wi / (ras["ms"] * 1e-3) / 1e9, "peak": issue_peak,
                    "unit": "Gwarp-inst/s", "frac": ras.get("frac_issue"),
                    "peak_source": f"{n_sm} SMs x 4 schedulers x 1 warp instruction per clock x {sm_mhz:.0f} MHz (the SM clock "
                                   "sampled during the timed region; unit counts from B300_MICROARCH.md / B200_PROFILING.md)",
                    "algorithmic": f"{wi} warp instructions per frame (smsp__inst_executed.sum of near pass + k_hiz + far pass, "
                                   f"from the committed ncu capture: {ncu_meta.get('label')}) / stages.raster.ms measured in this "
                                   f"run; the frame draws {n_cons} conservative + {n_cen} centre predicate-true hits",
                    "traffic": ncu.get("raster", {}).get("dram_bytes"),
                    "covers": "the raster stage: k_raster (near pass) + k_hiz + k_raster (far pass); time = stages.raster.ms",
                    "views": views}
    else:
        roofline = {"kernel": "k_" + dom, "bound": "hbm", "achieved": d["GBps"], "peak": hbm_peak, "unit": "GB/s",
                    "frac": d["frac_hbm"], "traffic": ncu.get(dom, {}).get("dram_bytes"), "peak_source": hbm_src,
                    "algorithmic": f"{d['bytes']} bytes per frame"}
    roofline["traffic_source"] = ncu_meta
    # the three fractions north_star asks for, as it states them
    north_star = {
        "raster_vs_l2": {"frac_l2_load": ras["frac_l2_load"], "frac_l2_atomic_random": ras["frac_l2_atomic_random"]},
        "generate_vs_hbm": {"GBps": stages["generate"].get("GBps"), "frac": stages["generate"].get("frac_hbm")},
        "shade_vs_hbm": {"GBps": sh.get("GBps"), "frac": sh.get("frac_hbm"),
                         "frac_unique_vertices": sh["frac_hbm_unique_vertices"],
                         "note": "frac is on SURVEY 8(d)'s UPPER-BOUND bytes (64 B of gathers per centre hit); on the bytes "
                                 "actually touched (unique vertices) it is frac_unique_vertices: quote both"},
    }

    # ---- the oracle timed beside it on this box's host cores (bounded sample of the same workload)
    cpu_baseline = None
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        dt, seg, desc, _ = oracle_sample(args.config, args.cpu_scale, 1.0 if args.res_scale == 1.0 else args.res_scale)
        cpu_baseline = {"value": seg / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                        "seconds": dt, "stage_seconds": oracle_sample.last_stage_seconds, "cpu_model": cpu_model(),
                        "host_cores_available": os.cpu_count()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{args.config - 1}] '{sc['name']}': {synth.n_strands(sc)} strands, "
                               f"{len(sc['grooms'])} grooms, {W}x{H}, 1 spp, lod_lambda {list(lam)}",
                   "strands_after_lod": cnt["n_strands_lod"], "vertices": cnt["n_vertices"], "segments": n_seg,
                   "l2": "no flush: per-frame working set (G-buffer 16 B/px + colour + out_rgb + vertices = "
                         f"{(48 * n_px + 16 * cnt['n_vertices']) / 1e6:.0f} MB) exceeds the 126 MB L2",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "frame_ms": ms_step, "strands_per_s": world * cnt["n_strands_lod"] / (ms_step * 1e-3),
        "segments_per_s": world * n_seg / (ms_step * 1e-3),
        "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": ms_e2e, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step_unpipelined": ms_e2e_sync,
                "out_rgb_format": "float32 [h][w][4]", "out_gbuffer_copied": False,
                "what": "per step: hair_mesh_update of every cage (pinned host) + hair_render_to_host_async (out_rgb as "
                        "float32 to pinned host, 2 frames in flight), hair_host_wait after the last; wall clock over the "
                        "steps. out_gbuffer, hair_render's other result, STAYS ON THE DEVICE in this figure (host_gbuffer = "
                        "NULL); with it copied too see float32_and_gbuffer_host_output. PCIe-bound: the device frame is "
                        "ms_per_step of the top level",
                "rgb16f_host_output": {"ms_per_step": ms_e2e16, "ms_per_step_unpipelined": ms_e2e16_sync,
                                       "d2h_bytes_per_step": d2h16, "Gsegments_per_s": n_seg * world / (ms_e2e16 * 1e-3) / 1e9,
                                       "what": "HAIR_FLAG_RGB16F: the filter writes RGBA16F (|error| < 2e-3 for |v| < 4); "
                                               "rounds 1-2 reported this leg as e2e.value"},
                "float32_and_gbuffer_host_output": {"ms_per_step": ms_e2e_gb, "ms_per_step_unpipelined": ms_e2e_gb_sync,
                                                    "d2h_bytes_per_step": d2h_gb}},
        "gpu_launches": st["gpu_launches"] * args.steps,
        "roofline": roofline, "north_star_fractions": north_star, "stages": stages, "l2_atomic_peaks_Gatom_per_s": atom,
        "l2_pair_load_peaks_Gloads_per_s": l2,
        "hbm_peak_GBps": hbm_peak, "hbm_peak_source": hbm_src,
        "counts": {k: cnt[k] for k in ("n_bundles", "n_bundles_culled", "n_strands_total", "n_strands_lod", "n_vertices",
                                       "n_segments", "n_segments_drawn", "n_segments_live", "n_atomics_center", "n_atomics_cons",
                                       "n_atomics_cons_ymajor", "n_atomics_issued", "n_pixels_center", "n_pixels_cons")},
        "raster_passes": {"two_pass": st["two_pass"], "n_segments_hiz_culled": st["n_segments_hiz_culled"],
                          "what": "production frames: bundles in the front 60 % of their groom's depth range first, 16x16-tile "
                                  "hi-Z (k_hiz), then the rest; a segment behind every tile of its bounding box is dropped "
                                  "before any pixel work (same G-buffer bit for bit; DESIGN.md 7.3)"},
        "shadows": {"build_ms": ms_dom_build, "lights": len(lcams), "res": 1024, "ms_per_step": ms_dom_frame,
                    "ms_shade": st_dom["ms_shade"],
                    "what": "hair_shadow_build: deep opacity maps of the point lights from the full grooms (LOD off); then the "
                            "bench frame with HAIR_FLAG_SHADOWS (PAPER.md:192, Eq. 7 lookup with the frame's beta per groom)"},
        "moving_camera": {"ms_per_step": ms_moving, "frames": k_mov, "ms_raster": st_mov["ms_raster"],
                          "ms_filter": st_mov["ms_filter"], "n_segments_hiz_culled_last_frame": st_mov["n_segments_hiz_culled"],
                          "what": "synth.moving_camera: yaw +-0.04 rad, sideways swing and dolly, a new camera every frame"},
        "pipelined": {"ms_per_frame": ms_pipelined, "frames": k_pipe, "ms_per_frame_serial_same_flags": ms_serial_noevents,
                      "bit_identical_to_serial": pipelined_same,
                      "what": "two contexts on two streams render alternate frames (two frames in flight, each context "
                              "with its own scratch): throughput over back-to-back frames; single-frame latency is not "
                              "better than ms_per_step"},
        "sequential_per_groom": {"ms_per_step": ms_seq, "what": "hair_render_sequential: one LOD..filter pass per groom, "
                                 "depth kept, blended over the target (PAPER.md:208-210); the headline frame resolves "
                                 "all grooms in one G-buffer instead (DESIGN.md R15)"},
        "cpu_baseline": cpu_baseline, "clocks": clocks,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based); 4 = the metric's workload")
    ap.add_argument("--scale", type=float, default=1.0, help="strand-count multiplier (1.0 = as named)")
    ap.add_argument("--res-scale", type=float, default=1.0, dest="res_scale")
    ap.add_argument("--cpu-scale", type=float, default=0.1, dest="cpu_scale",
                    help="strand-count multiplier of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
