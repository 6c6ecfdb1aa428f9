#!/usr/bin/env python
"""bench.py - headline benchmark of the OSOG forward-render hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

One "step" = one pass of the whole hot path (H1-H7: prepare, bounding box + count, scan, CSR fill + per-tile cull, ordered tile
composition with the fused field write-out) over one seeded synthetic batch = one osog_render_field call.
Default workload: BASELINE.json configs[3] (the paper-scale headline: 40,000 mixed particles, 2048 x 2048,
NA 0.65, 10 degree oblique ramp).  Prints ONE JSON line (see DESIGN.md section 10 for every key).

--impl reference times the float64 CPU oracle (oracle/) on the host cores, on a bounded sample of the same
workload; it is a deliberately plain program, a reported baseline and not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particles/s (hot path osog_render_field, 40k particles on 2048^2)"
# identical in both arms' `config` (the driver compares them): how cache state is handled between timed steps
TIMING_NOTE = "GPU arm: L2 flushed between timed steps (256 MB memset); CPU arm: every step recomputes its whole sample"
UNIT = "particles/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ALU roofline: the composition is bound by instruction issue, not by HBM.
ALU_INSTR_PER_ELLIPSOID_PAIR = 13      # ~12 fp32 instructions + 1 MUFU per true covered pair
ALU_INSTR_PER_PRISM_PAIR = 40          # 12 plane values + min / max + accumulate per true covered pair
ALU_INSTR_PER_PIXEL = 30               # sincospi + complex multiply + store per output pixel
N_SM, SMSP_PER_SM, LANES = 148, 4, 32  # B200: one warp instruction per clock and SM sub-partition (nominal issue rate)


def _roofline_inputs():
    """Tracked measurement inputs of the roofline (profiles/r2_roofline_inputs.json): the FFMA issue rate measured by
    paper_2606_21381_b200/issue_rates on this pool's B200 (profiles/r2_issue_rates.md) and the DRAM traffic of the
    dominant kernel from its last ncu --set full capture (profiles/r2_compose_ncu.md), each with command, date and commit."""
    try:
        with open(os.path.join(ROOT, "profiles", "r2_roofline_inputs.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def _sm_clock_ghz():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"]) * 1e-3, "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        return 1.965, "fallback 1965 MHz"


def _covered_pairs(name):
    """True covered (particle, pixel) pairs of a workload, from tests/golden/covered_pairs.txt (written by the oracle
    through tests/golden/make_covered_pairs.py; a stored workload statistic, no oracle code runs here)."""
    try:
        with open(os.path.join(ROOT, "tests", "golden", "covered_pairs.txt")) as f:
            for ln in f:
                p = ln.split()
                if len(p) == 3 and p[0] == name:
                    return int(p[1]), int(p[2])
    except OSError:
        pass
    return None


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self._stop = threading.Event()
        self._th = threading.Thread(target=self._run, daemon=True)

    def _sample(self):
        try:
            out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
            parts = [x.strip() for x in out.strip().split(",")]
            if len(parts) >= 6:
                self.rows.append(parts)
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self._sample()
            self._stop.wait(0.1)

    def __enter__(self):
        self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._th.join(timeout=6)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({n for r in self.rows for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def _sample_rows(scene, rows):
    """Oracle OPD of `rows` consecutive pixel rows from the middle of frame 0 (a bounded sample of the workload)."""
    from oracle import oracle as o
    fs = scene.frame_start
    cols = {k: v[int(fs[0]):int(fs[1])] for k, v in scene.cols.items()}
    # a strip is its own frame whose pixel rows are shifted: move the particles instead of the window
    i0 = (scene.H - rows) // 2
    shifted = dict(cols)
    shifted["cy"] = (cols["cy"].astype(np.float64) - i0 * scene.pitch_um).astype(np.float32)
    return o.render_opd_frame(shifted, 0, cols["kind"].shape[0], rows, scene.W, scene.pitch_um, scene.n_medium)


def cpu_baseline(scene, budget_s=12.0):
    """Time the oracle as it stands on the host cores on a strip of frame 0; scale particles/s by area."""
    cores = len(os.sched_getaffinity(0))
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    rows = min(scene.H, 64)
    t0 = time.perf_counter()
    _sample_rows(scene, rows)                       # warm-up (also builds / loads the oracle library)
    dt = time.perf_counter() - t0
    rows = int(min(scene.H, max(16, rows * budget_s / max(dt, 1e-3) * 0.5)))
    t0 = time.perf_counter()
    _sample_rows(scene, rows)
    dt = time.perf_counter() - t0
    n0 = int(scene.frame_start[1] - scene.frame_start[0])
    frac = rows / scene.H                            # fraction of one frame's pixels (and of its particle work)
    pps = n0 * frac / dt
    return {"value": pps, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"OPD of {rows} of {scene.H} pixel rows of frame 0 ({n0} particles), float64, bcircle mode, "
                      f"{dt:.2f} s; particles/s = particles x row fraction / time"}, dt


def run_reference(args):
    from workloads import make_config, CONFIG_NAMES
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    scene = make_config(args.config)
    vals = []
    budget = min(4.0, 150.0 / max(1, args.steps + args.warmup))   # whole run stays within a few minutes
    for _ in range(args.warmup):
        cpu_baseline(scene, budget_s=budget)
    last = None
    for _ in range(args.steps):
        last, _dt = cpu_baseline(scene, budget_s=budget)
        vals.append(last["value"])
    v = float(np.mean(vals))
    n0 = int(scene.frame_start[1] - scene.frame_start[0])
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": n0 / v * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": CONFIG_NAMES[args.config], "N": scene.N, "H": scene.H, "W": scene.W, "B": scene.B,
                       "l2": TIMING_NOTE},
            "cpu_baseline": dict(last, value=v),
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def max_over_ranks(values, device=None):
    """MAX over ranks of a list of floats (timings): the slowest rank defines the job time.  Works on any
    initialised torch.distributed backend (nccl on the GPU box, gloo in the CPU test); identity for one process."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_value(units_per_rank_step, steps, world, t_max):
    """Replicas only: every rank processes the same number of units; value = all ranks' units / slowest rank's time."""
    return world * units_per_rank_step * steps / t_max


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_21381_b200 as og
    from workloads import make_config, CONFIG_NAMES

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # replicas only: every rank renders its own seeded copy of the workload, no collective
    scene = make_config(args.config)
    H, W, B, N = scene.H, scene.W, scene.B, scene.N
    ctx = og.Context(H, W, N, max_frames=B, device=dev, check=False)   # enqueue-only calls; status checked after the loops
    P = og.Particles.from_scene(scene, device=dev)
    opt = og.optics_from_scene(scene)
    field = torch.empty((B, H, W, 2), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)       # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream(dev)
    # ---- device-resident timing: K steps, each bracketed by CUDA events on the launching stream, L2 flushed between
    for _ in range(args.warmup):
        flush.zero_()
        ctx.render_field(P, opt, out=field)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for k in range(args.steps):
            flush.zero_()
            ev[k][0].record(stream)
            ctx.render_field(P, opt, out=field)
            ev[k][1].record(stream)
        barrier()
        t_wall = time.perf_counter() - t_wall0
        # keep the GPU busy a little longer so that the sampler sees clocks under load
        t_end = time.perf_counter() + 0.6
        while time.perf_counter() < t_end:
            ctx.render_field(P, opt, out=field)
        torch.cuda.synchronize()
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    t_steps = float(ms.sum()) * 1e-3
    r, bits, pairs = ctx.status()
    assert r == 0, f"osog_status {r}"

    # ---- end-to-end: host (pinned) particle arrays -> device, render, device -> host read of the result
    names = ("cx", "cy", "qw", "qx", "qy", "qz", "d0", "d1", "d2", "n_p")
    host = {k: torch.from_numpy(scene.cols[k]).pin_memory() for k in names}
    host["kind"] = torch.from_numpy(scene.cols["kind"]).pin_memory()
    devbuf = {k: torch.empty_like(v, device=dev) for k, v in host.items()}
    P2 = og.Particles(devbuf, scene.frame_start if B > 1 else None, device=dev)
    host_out = torch.empty((B, H, W, 2), dtype=torch.float32).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in host.values())
    d2h = host_out.numel() * host_out.element_size()

    # Two output buffers and a copy stream: the device->host read of step k overlaps the upload + render of step k + 1
    # (every step still uploads its own inputs and reads its own result back; nothing is skipped or reused).
    copy_stream = torch.cuda.Stream(device=dev)
    fields2 = [field, torch.empty_like(field)]
    host_outs = [host_out, torch.empty((B, H, W, 2), dtype=torch.float32).pin_memory()]
    rendered = [torch.cuda.Event() for _ in range(2)]
    copied = [torch.cuda.Event() for _ in range(2)]

    def e2e_step(k):
        s = k & 1
        for name, v in host.items():
            P2.t[name].copy_(v, non_blocking=True)
        if k >= 2:
            stream.wait_event(copied[s])                 # field[s] was read back two steps ago
        ctx.render_field(P2, opt, out=fields2[s])
        rendered[s].record(stream)
        with torch.cuda.stream(copy_stream):
            copy_stream.wait_event(rendered[s])
            host_outs[s].copy_(fields2[s], non_blocking=True)
            copied[s].record(copy_stream)

    for k in range(2 * max(1, args.warmup // 2)):
        e2e_step(k)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(args.steps):
        e2e_step(k + 2)
    stream.wait_stream(copy_stream)                      # the last read-backs are inside the timed region
    e1.record(stream)
    barrier()
    t_e2e = e0.elapsed_time(e1) * 1e-3

    # ---- dominant kernel (k_compose_tile) timed alone for the roofline, + the separately timed library stage
    lib = og.lib()
    inten = torch.empty((B, H, W), dtype=torch.float32, device=dev)
    ctx.render_intensity(P, opt, out=inten)
    ctx.field_to_intensity(opt, torch.view_as_complex(field), out=inten)    # (first out-of-place transform: plan warm-up)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.field_to_intensity(opt, torch.view_as_complex(field), out=inten)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_optics = e0.elapsed_time(e1) / 5
    # ---- DIC library stage (Eq. 5): shear + 4 cuFFTs + element-wise kernels, timed alone
    dic = og.make_dic(2, 0, 0.5)
    ctx.field_to_dic(opt, dic, torch.view_as_complex(field), out=inten)      # first call allocates the second batch
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.field_to_dic(opt, dic, torch.view_as_complex(field), out=inten)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_dic = e0.elapsed_time(e1) / 5
    ctx.render_opd(P, opt, out=inten)                  # (first use of this instantiation: module load outside the timed loop)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.render_opd(P, opt, out=inten)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_opd = e0.elapsed_time(e1) / 5

    # ---- G-buffer extras: depth + instance-id maps, binning included
    ctx.render_gbuffer(P, opt)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.render_gbuffer(P, opt)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_gbuffer = e0.elapsed_time(e1) / 5
    ctx.render_height(P, opt)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.render_height(P, opt)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_height = e0.elapsed_time(e1) / 5
    # ---- first backward step: dL/dn_p for an upstream dL/dOPD, preparation kernel included
    gopd = torch.ones((B, H, W), dtype=torch.float32, device=dev)
    ctx.backward_np(P, opt, gopd)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.backward_np(P, opt, gopd)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_backward = e0.elapsed_time(e1) / 5
    ctx.backward_centre(P, opt, gopd)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.backward_centre(P, opt, gopd)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_backward_c = e0.elapsed_time(e1) / 5
    ctx.backward_params(P, opt, gopd)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.backward_params(P, opt, gopd)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_backward_p = e0.elapsed_time(e1) / 5
    ctx.backward_particles(P, opt, gopd)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.backward_particles(P, opt, gopd)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_backward_all = e0.elapsed_time(e1) / 5
    ctx.backward_intensity(P, opt, gopd)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(5):
        ctx.backward_intensity(P, opt, gopd)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_backward_i = e0.elapsed_time(e1) / 5

    # ---- measured alternative (paper-style global atomicAdd scatter), OPD only, for the record
    e0.record(stream)
    for _ in range(3):
        ctx.render_opd_atomic(P, opt, out=inten)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_atomic = e0.elapsed_time(e1) / 3
    ctx.render_opd_smem_atomic(P, opt, out=inten)
    e0.record(stream)
    for _ in range(3):
        ctx.render_opd_smem_atomic(P, opt, out=inten)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_smem_atomic = e0.elapsed_time(e1) / 3

    # ---- the dominant kernel alone (k_compose_tile on the binning of the last call), CUDA events on its stream
    ctx.render_field(P, opt, out=field)
    for _ in range(3):
        ctx.recompose_field(field)
    torch.cuda.synchronize()
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
    for a_, b_ in kev:
        flush.zero_()
        a_.record(stream)
        ctx.recompose_field(field)
        b_.record(stream)
    torch.cuda.synchronize()
    ms_compose = float(np.mean([a_.elapsed_time(b_) for a_, b_ in kev]))

    t_steps, t_e2e = max_over_ranks([t_steps, t_e2e], dev)
    peak, peak_src = _peaks()
    # library stage (L1-L3): bytes this design has to move on a power-of-two frame: field read, the kept
    # columns written / read / written / read, intensity written; other frames (cuFFT path): SURVEY 8(d)'s 92 bytes per pixel
    pow2 = all(v >= 64 and v <= 4096 and (v & (v - 1)) == 0 for v in (H, W))
    if pow2:
        rx = max(int(np.floor(float(scene.NA[b]) * scene.pitch_um / float(scene.lambda_um[b]) * W)) + 1 for b in range(B))
        ncol = min(rx, W // 2 - 1) + min(rx, W // 2) + 1
        lib_bytes = 8 * B * H * W + 4 * 8 * B * ncol * H + 4 * B * H * W
    else:
        ncol, lib_bytes = W, 92 * B * H * W
    lib_gbs = lib_bytes / (ms_optics * 1e-3) / 1e9
    lib_roof = {"bound": "hbm", "achieved": lib_gbs, "peak": peak, "unit": "GB/s", "frac": lib_gbs / peak,
                "algorithmic_bytes": int(lib_bytes), "kept_columns": int(ncol), "stage_ms": ms_optics,
                "what": "osog_field_to_intensity: k_fo_rows_fwd, k_fo_cols, k_fo_rows_inv" if pow2 else "osog_field_to_intensity: cuFFT x 2, k_pupil, k_sensor",
                "note": "bytes of THIS design (pruned to the pupil's columns); SURVEY 8(d) counts 92 bytes per pixel for the unpruned stage"}
    alg_bytes = 48 * N + 8 * pairs + 8 * B * H * W      # SoA read + list write/read + complex64 write
    ms_step = t_steps / args.steps * 1e3
    step_gbs = alg_bytes / (ms_step * 1e-3) / 1e9
    k_bytes = 4 * pairs + 8 * B * H * W                 # k_compose_tile alone: list read + complex64 write
    achieved = k_bytes / (ms_compose * 1e-3) / 1e9
    rin = _roofline_inputs()
    cap = rin.get("k_compose_tile_dram", {})
    traffic = cap.get("bytes") if cap.get("workload") == CONFIG_NAMES[args.config] else None
    hbm = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "traffic": traffic, "traffic_note": ("dram read+write of one k_compose_tile launch, ncu --set full, captured "
           f"{cap.get('captured')} at commit {cap.get('commit')} ({cap.get('source')}); the field it writes mostly stays in "
           "the 126 MB L2 during the launch") if traffic is not None else "no tracked ncu capture for this workload",
           "peak_source": peak_src, "algorithmic_bytes": int(k_bytes), "kernel": "k_compose_tile",
           "kernel_ms": ms_compose, "frac_of_nominal_8TBs": achieved / 8000.0,
           "note": "BASELINE.json's '% of B200 HBM roofline'; the kernel is bound by instruction issue, see roofline"}
    cp = _covered_pairs(CONFIG_NAMES[args.config])
    if cp is not None:
        ghz, ghz_src = _sm_clock_ghz()
        ffma = rin.get("ffma_lanes_per_clk_per_sm", {})
        lanes_per_clk = float(ffma.get("value", SMSP_PER_SM * LANES))           # measured FFMA issue rate, else the nominal 128
        alu_peak = N_SM * lanes_per_clk * ghz * 1e-3                            # T lane-instructions / s
        alg_instr = (ALU_INSTR_PER_ELLIPSOID_PAIR * cp[0] + ALU_INSTR_PER_PRISM_PAIR * cp[1]
                     + ALU_INSTR_PER_PIXEL * B * H * W)
        alu_ach = alg_instr / (ms_compose * 1e-3) / 1e12
        roof = {"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "T lane-instructions/s",
                "frac": alu_ach / alu_peak, "traffic": hbm["traffic"], "kernel": "k_compose_tile",
                "kernel_ms": ms_compose, "algorithmic_instructions": int(alg_instr),
                "units": {"ellipsoid_pairs": cp[0], "prism_pairs": cp[1], "pixels": B * H * W,
                          "instr_per_unit": [ALU_INSTR_PER_ELLIPSOID_PAIR, ALU_INSTR_PER_PRISM_PAIR,
                                             ALU_INSTR_PER_PIXEL],
                          "source": "tests/golden/covered_pairs.txt (oracle count of pairs with positive thickness)"},
                "peak_source": (f"{N_SM} SMs x {lanes_per_clk:.1f} lane-instructions/clk/SM x {ghz:.3f} GHz ({ghz_src}); "
                                + (f"the rate is the MEASURED FFMA issue rate ({ffma.get('source')}, {ffma.get('captured')}), "
                                   f"{lanes_per_clk / (SMSP_PER_SM * LANES):.3f} of the nominal 128 = 4 sub-partitions x 32 lanes"
                                   if ffma else "NOMINAL 4 sub-partitions x 32 lanes (no tracked measurement found)")
                                + "; one warp instruction per clock and sub-partition is the ceiling of every pipe mix "
                                  "(DESIGN.md section 7)")}
    else:
        roof = hbm
    line = {
        "metric": METRIC, "value": whole_job_value(N, args.steps, world, t_steps), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32+f64", "data": "synthetic",
        "config": {"workload": CONFIG_NAMES[args.config], "N": N, "H": H, "W": W, "B": B, "l2": TIMING_NOTE},
        "extra": {"tile": og.osog_tile_size(), "pairs": int(pairs), "parallelism": "replicas only"},
        "frames_per_s": world * B * args.steps / t_steps,
        "ms_per_step_median": float(np.median(ms)), "ms_per_step_std": float(ms.std()),
        "e2e": {"value": world * N * args.steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h)},
        "gpu_launches": 3 * args.steps,
        "roofline": roof, "roofline_hbm": hbm,
        "roofline_step": {"achieved": step_gbs, "frac": step_gbs / peak, "algorithmic_bytes": int(alg_bytes),
                          "what": "whole hot path: k_prepare, k_sort_cull, k_compose_tile"},
        "roofline_library": lib_roof,
        "library_stage_ms": ms_optics, "dic_stage_ms": ms_dic, "gbuffer_ms": ms_gbuffer, "height_grad_lap_ms": ms_height, "backward_np_ms": ms_backward, "backward_centre_ms": ms_backward_c, "backward_params_ms": ms_backward_p, "backward_particles_ms": ms_backward_all, "backward_intensity_ms": ms_backward_i, "opd_only_ms": ms_opd, "atomic_alternative_opd_ms": ms_atomic, "smem_atomic_alternative_opd_ms": ms_smem_atomic,
        "paper_context": "PAPER.md:195: 40,000 particles < 50 ms on one A100 at 1024^2 (whole pipeline); context only",
        "clocks": clk.summary(),
    }
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"], _ = cpu_baseline(scene)
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
