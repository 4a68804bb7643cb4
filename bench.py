#!/usr/bin/env python
"""bench.py -- geodesic steps/s and images/s of the RAPTOR hot path on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W [--workload C2] [--impl reference]

A "step" is one pass of the whole hot path (camera, geodesic RHS, RK4 + step rule,
plasma sampler, fluid-frame quantities, emissivity/absorptivity/intensity update, image + flux reduction)
over one synthetic image.  N = 1 workload: C2 = BASELINE.json configs[2], the 1024^2-pixel configuration
the metric ("images/sec (1024^2 px)") is quoted on.  N > 1 (torchrun, one rank per GPU): rays are
independent, so every rank renders its own frame (weak scaling, no data-path collective); value = all
ranks' steps / max-over-ranks time.

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the definitions of every key.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "geodesic_steps_per_sec"
UNIT = "steps/s"

# FP64 peak of one B200 for "bound": "alu".  The denominator of roofline.frac is the MEASURED
# peak: the live DFMA probe raptor_fp64_peak (8 independent DFMA chains per thread on all SMs), run in this process
# right before the timed region.  The derived figure 148 SMs x 4 sub-partitions x 16 FP64 FMA lanes x 2 flop x
# 1.965 GHz (clocks.max.sm) is printed beside it as peak_nominal.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 4 * 16 * 2 * 1.965e9 / 1e12
# The numerator: executed FP64 instructions per accepted step of the SHIPPED kernel, measured by ncu and stored in
# profiles/fp64_inst_per_step.json together with the hash of the kernel sources (paper_1801_10452_b200/
# roofline_counts.py says how).  If the sources here hash differently the roofline is reported as null.
# paper's own numbers for its performance configuration (Table B.1 / PAPER.md:342, 666): context for PB1 only
PAPER_GEODESICS_PER_SEC = {"GTX 1080, OpenACC, single precision": 104900.0, "i7-6950X 10 cores, OpenMP, single precision": 10707.0}


LC_DT = 2.5      # workloads LC (32 frames per light curve) and C3B (8 spectra): camera-time spacing [M]


def build_scene(workload: str):
    from paper_1801_10452_b200 import scenes
    if workload == "C3B":
        # a batch of C3 spectra (256^2 x 32 frequencies each) traced by ONE launch: a single 256^2 frame is one wave of
        # 2,048 warps whose time is its longest ray's; batching is what fills the GPU
        from dataclasses import replace
        return replace(scenes.config("C3"), name="C3B")
    if workload == "LC":
        # slow-light light curve (Sect. 5): 256^2 pixels, the paper's four VLBI frequencies, 16 snapshots
        from dataclasses import replace
        s = scenes.config_C4(nx=256, n1=64, n2=48, n3=32, nt=16)
        return replace(s, name="LC", freq_hz=(22e9, 43e9, 86e9, 230e9))
    return scenes.config(workload)


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def oracle_sample(scene, row_stride, repeats=1):
    """Times the oracle, as it stands, on every row_stride-th image row of the workload (host cores)."""
    from oracle import oracle
    o = oracle.Oracle(scene, dtype="f32" if getattr(scene, "precision", 0) == 1 else "f64")
    t0 = time.perf_counter()
    steps = 0
    for _ in range(repeats):
        out = o.render(rows=(row_stride // 2, scene.ny), row_stride=row_stride)
        steps += out["steps"]
    dt = time.perf_counter() - t0
    return steps, dt


def omp_threads():
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def run_reference(args):
    """--impl reference: the CPU oracle (the only reference this tier has), bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene = build_scene(args.workload)
    # rows are the oracle's only parallel axis (OpenMP, schedule(dynamic, 1)): at least 2 rows per thread per step,
    # otherwise half the cores idle and the two oracle timings of one box (this arm, cpu_baseline) disagree
    rows_per_step = min(scene.ny, max(8, 2 * omp_threads()))
    stride = args.ref_row_stride or max(1, scene.ny // rows_per_step)
    for _ in range(args.warmup):
        oracle_sample(scene, max(stride, scene.ny // 2))
    tot_steps, tot_t = 0, 0.0
    for _ in range(args.steps):
        s, dt = oracle_sample(scene, stride)
        tot_steps += s
        tot_t += dt
    value = tot_steps / tot_t
    sample = (f"every {stride}th row of the {scene.nx}x{scene.ny} {args.workload} image per step "
              f"({len(range(stride // 2, scene.ny, stride))} rows on {omp_threads()} threads)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if scene.precision == 1 else "f64", "data": "synthetic",
            "config": {"workload": args.workload, "pixels": [scene.nx, scene.ny], "n_freq": scene.n_freq,
                       "note": "CPU oracle (oracle/raptor_oracle.c) as it stands, OpenMP over image rows"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": omp_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1801_10452_b200 import binding, parallel, roofline_counts

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()

    lc = args.workload in ("LC", "C3B")
    LC_FRAMES = {"LC": 32, "C3B": 8}.get(args.workload, 1)
    strong = args.scaling == "strong" and world > 1
    if strong and lc:
        raise SystemExit("--scaling strong shards one image by tiles; a light curve shards by frames")
    base_scene = build_scene(args.workload)
    # weak scaling (default): a movie, every rank renders its OWN frame (own camera time / own snapshot);
    # strong scaling: ONE image, every rank traces its interleaved tiles, one all-reduce(SUM) of the image per step
    scene = base_scene if strong else parallel.frame_of_rank(base_scene, rank)
    R = binding.Raptor(scene)
    if strong:
        R.set_shard(rank, world)
    image = torch.empty((scene.n_freq, scene.ny, scene.nx), dtype=torch.float64, device="cuda")
    flux = torch.empty((scene.n_freq,), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    sp = binding.C.c_void_p(stream.cuda_stream)
    l2_flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    lc_flux = torch.empty((LC_FRAMES, scene.n_freq), dtype=torch.float64, device="cuda") if lc else None
    lc_t0 = scene.t_cam - 0.5 * LC_FRAMES * LC_DT

    def render_call(img):
        binding.raptor_render(R.ctx, img.data_ptr(), None, None, sp)

    def flux_call(img):
        binding.raptor_flux(R.ctx, img.data_ptr(), flux.data_ptr(), sp)
        return flux

    def one_step(ev=None):
        # a1-a6 + image write (render kernel), a7 flux reduction (2 small kernels): 3 launches
        if ev:
            ev[0].record(stream)
        if lc:
            # one light curve: LC_FRAMES frames traced by one k_render launch + one flux reduction over all of them
            binding.raptor_light_curve(R.ctx, LC_FRAMES, lc_t0, LC_DT, lc_flux.data_ptr(), sp)
            if ev:
                ev[1].record(stream)
        elif strong:
            # the function the gloo test drives: zero, render this rank's tiles, all-reduce the image, flux
            def render_shard(img):
                render_call(img)
                if ev:
                    ev[1].record(stream)
            parallel.strong_step(render_shard, image, flux_call)
        else:
            render_call(image)
            if ev:
                ev[1].record(stream)
            flux_call(image)
        if ev:
            ev[2].record(stream)

    for _ in range(max(args.warmup, 3)):
        one_step()
    torch.cuda.synchronize()
    fp64_probe = binding.raptor_fp64_peak(1 << 16)[0]
    # issue rate of the FP64 pipe by operand form (raptor.h): cycles per warp instruction per sub-partition
    fp64_forms = None
    if rank == 0:
        names = ("dfma_1reg_imm", "dfma_3reg", "dfma_2reg", "dmul_2reg", "dadd_2reg")
        fp64_forms = {}
        for form, nm in enumerate(names):
            rate, clk = binding.raptor_fp64_probe(form)
            fp64_forms[nm] = 148 * 4 * clk / rate
    c_before = R.counters()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        l2_flush.zero_()                       # flush L2 between timed iterations (not timed)
        one_step(events[k])
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop() if rank == 0 else None
    step_ms = [e[0].elapsed_time(e[2]) for e in events]
    render_ms = [e[0].elapsed_time(e[1]) for e in events]
    c_after = R.counters()
    steps_done = c_after[0] - c_before[0]
    sampled_done = c_after[1] - c_before[1]
    total_ms = sum(step_ms)

    # ---- end to end through the C ABI with HOST buffers: grid upload (h2d), render, image + flux read back (d2h)
    h_image = torch.empty((scene.n_freq, scene.ny, scene.nx), dtype=torch.float64).pin_memory()
    h_flux = torch.empty((scene.n_freq,), dtype=torch.float64).pin_memory()
    h_grid = None
    if scene.grid is not None:
        g = np.ascontiguousarray(scene.grid, dtype=np.float32 if scene.grid_dtype == 1 else np.float64)
        h_grid = torch.from_numpy(g.reshape(-1).copy()).pin_memory()
    e2e_steps = max(2, min(args.steps, 5))
    h_lc = torch.empty((LC_FRAMES, scene.n_freq), dtype=torch.float64).pin_memory() if lc else None

    def e2e_step():
        # the upload is asynchronous on the caller's stream; raptor_render_host orders itself after it (raptor.h)
        if h_grid is not None:
            binding.raptor_upload_grid(R.ctx, h_grid.data_ptr(), h_grid.numel() * h_grid.element_size(), sp)
        if lc:
            binding.raptor_light_curve(R.ctx, LC_FRAMES, lc_t0, LC_DT, lc_flux.data_ptr(), sp)
            h_lc.copy_(lc_flux, non_blocking=True)
            torch.cuda.synchronize()
        elif strong:
            one_step()
            h_image.copy_(image, non_blocking=True)
            h_flux.copy_(flux, non_blocking=True)
            torch.cuda.synchronize()
        else:
            binding.raptor_render_host(R.ctx, h_image.data_ptr(), None, None, h_flux.data_ptr())

    e2e_step()
    barrier()
    c0 = R.counters()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    c1 = R.counters()

    # ---- aggregate over ranks (the helper the world-size-2 gloo test covers): max time, summed units
    total_ms_max, steps_all = parallel.aggregate(total_ms, float(steps_done), device="cuda")
    e2e_ms_max, e2e_units_all = parallel.aggregate(t_e2e * 1e3, float(c1[0] - c0[0]), device="cuda")
    render_ms_max, sampled_all = parallel.aggregate(sum(render_ms), float(sampled_done), device="cuda")

    if rank == 0:
        frames = LC_FRAMES if lc else 1
        images_per_step = frames * (1 if strong else world)
        value = steps_all / (total_ms_max * 1e-3)
        avg_render_ms = sum(render_ms) / len(render_ms)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": "strong" if strong else "weak",
            "vs_baseline": None, "dtype": "f32" if scene.precision == 1 else "f64", "data": "synthetic",
            "config": {"workload": args.workload, "pixels": [scene.nx, scene.ny], "n_freq": scene.n_freq,
                       "spin": scene.a, "incl_deg": scene.incl_deg, "plasma_model": scene.plasma_model,
                       "grid": [scene.nt, scene.n1, scene.n2, scene.n3], "l2": "flushed between timed iterations",
                       "integrator": ["RK4", "Verlet", "Verlet+corrector", "RK2 (midpoint)"][scene.integrator],
                       "step_policy": "A" if scene.step_policy == 0 else "B",
                       "step_rule": (f"h = min(clamp({scene.step_c} (r - r_H), {scene.step_min}, {scene.step_max}), "
                                     f"eps_polar r |sin theta|), eps_polar = {scene.eps_polar} (polar guard: DESIGN.md 3.2; "
                                     "BASELINE.json configs[0] states the clamp alone)") if scene.step_policy == 0
                                    else f"Eq. 21-24, eps = {scene.eps}, delta = {scene.delta}",
                       "eps_polar": scene.eps_polar if scene.step_policy == 0 else None,
                       "tau_cutoff": scene.tau_cutoff if math.isfinite(scene.tau_cutoff) else None,
                       "parallelism": ("single GPU" if world == 1 else
                                       f"one image, interleaved 8x4 tiles over {world} ranks + all-reduce(SUM) of the image" if strong
                                       else f"frames x{world}: every rank renders its own frame, no data-path collective")},
            "images_per_sec": images_per_step * args.steps / (total_ms_max * 1e-3),
            "steps_per_image": steps_all / (args.steps * images_per_step),
            "sampled_steps_per_image": sampled_all / (args.steps * images_per_step),
            "clocks": clocks,
            "e2e": {"value": e2e_units_all / (e2e_ms_max * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(h_grid.numel() * h_grid.element_size()) if h_grid is not None else 0,
                    "d2h_bytes_per_step": int(h_lc.numel() * 8) if lc else int(h_image.numel() * 8 + h_flux.numel() * 8),
                    "images_per_sec": images_per_step * e2e_steps / (e2e_ms_max * 1e-3)},
            "gpu_launches": 3 * args.steps,
            "frames_per_step": frames,
            "rays_per_sec": images_per_step * args.steps * scene.nx * scene.ny / (total_ms_max * 1e-3),
            "wall_s_timed_region": t_wall,
        }
        # ---- roofline of the dominant kernel (rank 0's launches): measured counts / measured peak
        counts, why = roofline_counts.load()
        row = counts.get(args.workload) if counts else None
        if row is None:
            line["roofline"] = None
            line["roofline_unavailable"] = why or f"no ncu counts for workload {args.workload} in profiles/fp64_inst_per_step.json"
        elif scene.precision == 1:
            # the single-precision kernel: FP32 FMA pipe, 128 lanes per SM; peak derived from unit counts and clocks
            flop_step = 2.0 * row["ffma"] + row["fmul"] + row["fadd"]
            steps_launch = steps_done / args.steps
            achieved = steps_launch * flop_step / (avg_render_ms * 1e-3) / 1e12
            peak32_nominal = 148 * 128 * 2 * 1.965e9 / 1e12
            peak32 = binding.raptor_fp32_peak(1 << 16)[0]               # measured here, after the timed region
            line["roofline"] = {
                "bound": "alu", "kernel": "k_render_f32", "achieved": achieved, "peak": peak32, "unit": "TFLOP/s",
                "frac": achieved / peak32,
                "peak_source": "measured: raptor_fp32_peak (independent FFMA chains on all SMs) in this process",
                "peak_nominal": peak32_nominal, "frac_of_nominal": achieved / peak32_nominal,
                "traffic": (row.get("dram_read_bytes", 0.0) + row.get("dram_write_bytes", 0.0)) if "dram_read_bytes" in row else None,
                "fp32_inst_per_step": {"ffma": row["ffma"], "fmul": row["fmul"], "fadd": row["fadd"]},
                "counts_source": "profiles/fp64_inst_per_step.json (ncu, source hash verified)",
                "kernel_ms": avg_render_ms, "kernel_share_of_step": avg_render_ms / (total_ms / args.steps),
                "algorithmic_flop_per_launch": steps_launch * flop_step}
        else:
            flop_step = 2.0 * row["dfma"] + row["dmul"] + row["dadd"]
            steps_launch = steps_done / args.steps
            achieved = steps_launch * flop_step / (avg_render_ms * 1e-3) / 1e12
            # the FP64 pipe issues one warp instruction per 2 cycles per sub-partition whether it is a DFMA, a DMUL/DADD or
            # a DSETP: share of those issue slots the kernel filled, and the flop ceiling its instruction mix allows
            slots = 148 * 4 * (clocks["sm_mhz"] or 1965.0) * 1e6 / 2.0 * avg_render_ms * 1e-3 if clocks else None
            pipe_frac = row["fp64_pipe_warp_inst"] * steps_launch / slots if slots and "fp64_pipe_warp_inst" in row else None
            n_arith = row["dfma"] + row["dmul"] + row["dadd"]
            line["roofline"] = {
                "bound": "alu", "kernel": "k_render", "achieved": achieved, "peak": fp64_probe, "unit": "TFLOP/s",
                "frac": achieved / fp64_probe,
                "peak_source": "measured: raptor_fp64_peak (independent DFMA chains on all SMs) in this process",
                "peak_nominal": FP64_PEAK_NOMINAL_TFLOPS, "frac_of_nominal": achieved / FP64_PEAK_NOMINAL_TFLOPS,
                "traffic": (row.get("dram_read_bytes", 0.0) + row.get("dram_write_bytes", 0.0)) if "dram_read_bytes" in row else None,
                "fp64_pipe_frac": pipe_frac, "mix_ceiling": flop_step / (2.0 * n_arith),
                "fp64_inst_per_step": {"dfma": row["dfma"], "dmul": row["dmul"], "dadd": row["dadd"],
                                       "pipe_warp_inst_x32": 32.0 * row.get("fp64_pipe_warp_inst", float("nan"))},
                "counts_source": "profiles/fp64_inst_per_step.json (ncu, source hash verified)",
                "kernel_ms": avg_render_ms, "kernel_share_of_step": avg_render_ms / (total_ms / args.steps),
                "algorithmic_flop_per_launch": steps_launch * flop_step,
                "fp64_issue_cycles_by_form": fp64_forms}
            of = row.get("operand_forms")
            if of and fp64_forms:
                # operand-aware bound: a DFMA with three different register sources issues every ~3.2
                # cycles, every other FP64 instruction every ~2.06 -- both measured live above
                slow = fp64_forms["dfma_3reg"]
                fast = (fp64_forms["dfma_2reg"] + fp64_forms["dmul_2reg"] + fp64_forms["dadd_2reg"]) / 3.0
                cyc = of["dfma_3reg"] * slow + (of["dfma_3reg_reuse_flagged"] + of["dfma_other"] + of["dmul"] + of["dadd"] + of["dsetp"]) * fast
                clk_hz = (clocks["sm_mhz"] or 1965.0) * 1e6
                bound_ms = (steps_launch / 32.0) * cyc / (148 * 4 * clk_hz) * 1e3
                line["roofline"]["operand_bound"] = {"cycles_per_warp_step": cyc, "ms": bound_ms, "frac": bound_ms / avg_render_ms,
                                                     "dfma_3reg_per_step": of["dfma_3reg"]}
        # ---- CPU baseline: the oracle on a bounded sample of the same workload (about 10-30 s of host work)
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            stride = max(1, scene.ny // max(8, 2 * omp_threads()))
            s_, dt = oracle_sample(scene, stride)
            if dt < 5.0:
                stride = max(1, stride // 4)
                s_, dt = oracle_sample(scene, stride)
            cpu = {"value": s_ / dt, "unit": UNIT, "cores": omp_threads(), "kind": "oracle",
                   "sample": f"every {stride}th row of the {scene.nx}x{scene.ny} {args.workload} image "
                             f"({s_} steps in {dt:.1f} s)"}
        line["cpu_baseline"] = cpu
        if args.workload in ("PB1", "PB1F32"):
            line["paper_geodesics_per_sec"] = PAPER_GEODESICS_PER_SEC      # other hardware, FP32: context only
        print(json.dumps(line))
    R.close()
    if world > 1:
        dist.destroy_process_group()

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=["C0", "C1", "C2", "C3", "C4", "PB1", "PB1F32", "LC", "C3B"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one frame per rank (default), strong = one image sharded by tiles + all-reduce")
    ap.add_argument("--ref-row-stride", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
