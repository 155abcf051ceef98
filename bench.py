#!/usr/bin/env python
"""Benchmark of the line-RT render hot path (BASELINE.json metric: ray.channel.step samples/s, fwd+bwd).

A *step* is one pass of the whole hot path over one synthetic disk: ray geometry + forward march with the L2 data
term fused into its epilogue (radt_render_loss) -> memory-free adjoint (SURVEY.md section 8(a) rows a-j).  The workload at N = 1 is BASELINE.json
`configs[1]` (256x128 (r,z) grid, 256x256 px, 64 channels, 256 steps per ray).  With N > 1 every rank renders
its own disk (independent problems, no data-path collective): weak scaling.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One JSON line is printed by rank 0.  `value` = nominal samples (rays x channels x steps, summed over ranks and
steps) / device time of the K steps (inputs resident in HBM; L2 flushed between steps outside the timed
events).  `e2e` = the same step through the HOST-buffer C-ABI entry point (copies inside the timed region).
`roofline` = the dominant kernel against the SFU issue peak measured in this run.
`cpu_baseline` = the fp64 oracle, as it stands, on this box's host cores, on a bounded ray sample.
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

METRIC = "ray*channel*step samples/s (fwd+bwd step)"
UNIT = "samples/s"


_SPH = {"npix": 256, "nchan": 64}       # config 6 image size and channel count (--sph-npix / --sph-nchan sweep them)


def _scenes(cfg):
    """Configs 1-5: BASELINE.json configs[0..4]; 6: stand-in for the paper's own timing benchmark."""
    from synth import make_config, sph_benchmark_scene
    s = sph_benchmark_scene(npix=_SPH["npix"], nchan=_SPH["nchan"]) if cfg == 6 else make_config(cfg)
    return s if isinstance(s, list) else [s]


def _workload_name(cfg):
    from synth import config_names
    return f"cfg6_sph512x96x256_img{_SPH['npix']}_c{_SPH['nchan']}_n256" if cfg == 6 else config_names()[cfg]


# ----------------------------------------------------------------------------------------------------
# clocks: sampled during the timed region through NVML
# ----------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    def __init__(self, index=0, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:      # noqa: BLE001  (NVML missing: report nulls)
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:      # noqa: BLE001
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands, on a bounded sample of the same workload
# ----------------------------------------------------------------------------------------------------
def oracle_sample_step(scene, stride, G=None):
    """One fwd+adjoint pass of the oracle over every `stride`-th ray of `scene`; returns (seconds, samples)."""
    from oracle import pyoracle as po
    nrays = scene.nrays
    idx = np.arange(0, nrays, stride, dtype=np.int64)
    t0 = time.perf_counter()
    cube = po.render(scene, rays=idx)
    g = cube * 1e-6 if G is None else G
    po.render_bwd(scene, g, rays=idx)
    dt = time.perf_counter() - t0
    return dt, len(idx) * len(scene.line.vchan) * scene.geom.nstep


def cpu_baseline(scene, budget_s=12.0):
    """The oracle as it stands on this box's host cores: whole fwd + adjoint passes over every 2nd ray of the scene,
    repeated until about `budget_s` seconds of wall time (>= 2 passes)."""
    from oracle import pyoracle as po
    oracle_sample_step(scene, 64)          # load the library, touch the pages
    stride, tot_t, tot_n, passes = 2, 0.0, 0, 0
    while passes < 2 or tot_t < budget_s:
        dt, n = oracle_sample_step(scene, stride)
        tot_t += dt
        tot_n += n
        passes += 1
    cores = po.num_threads()
    # the same oracle on ONE thread (every 16th ray): the per-core figure SURVEY.md section 8(d) asks for
    po.set_num_threads(1)
    dt1, n1 = oracle_sample_step(scene, 16)
    po.set_num_threads(cores)
    return {"value": tot_n / tot_t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{scene.name}: {passes} passes over every {stride}nd ray ({tot_n:.3g} samples), fp64 forward + adjoint, "
                      f"{tot_t:.1f} s wall",
            "value_1thread": n1 / dt1}


def run_reference(args):
    """--impl reference: the reference arm of this tier is the fp64 CPU oracle on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pyoracle as po
    scene = _scenes(args.config)[0]
    # size the per-step ray sample so that the whole run stays within ~2 minutes on this box
    oracle_sample_step(scene, 256)
    dt, _ = oracle_sample_step(scene, 64)
    t_full = dt * 64.0
    stride = int(min(max(np.ceil(t_full * (args.steps + args.warmup) / 120.0), 1), scene.nrays // 8))
    for _ in range(args.warmup):
        oracle_sample_step(scene, stride)
    tot_t, tot_n = 0.0, 0
    for _ in range(args.steps):
        dt, n = oracle_sample_step(scene, stride)
        tot_t += dt
        tot_n += n
    val = tot_n / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(args.config), "sample": f"every {stride}th ray per step"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": po.num_threads(), "kind": "oracle",
                             "sample": f"every {stride}th ray of {_workload_name(args.config)} per step, fwd + adjoint"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------
def time_kernel_group(fn, stream, torch, flush, reps):
    """Average device time of fn() over `reps` launches, CUDA events on `stream`, L2 flushed before each."""
    tot = 0.0
    for _ in range(reps):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        fn()
        e1.record(stream)
        e1.synchronize()
        tot += e0.elapsed_time(e1)
    return tot / reps


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_03623_b200 import Renderer, binding as B
    from synth import l2_target

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the render has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()
    B.radt_set_option(B.OPT_WIN_PATH, args.win_path)

    scenes = _scenes(args.config)
    R = Renderer(scenes, device=f"cuda:{local}")
    stream = torch.cuda.current_stream()
    nominal = sum(s.nominal_samples for s in scenes)

    # target cube of the L2 data term: seed-generated from a first render (an input, built before timing)
    R.render()
    torch.cuda.synchronize()
    cube0 = R.cube.cpu().numpy()
    tgt = np.empty_like(cube0)
    sig = 0.0
    for b in range(cube0.shape[0]):
        t, s = l2_target(cube0[b], 36230 + args.config + 97 * rank + b)
        tgt[b] = t
        sig = max(sig, s)
    R.set_target(tgt, sig)

    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=R.device)     # > 126 MB L2

    def flush():
        flush_buf.fill_(1)

    def step():
        R.fit_step(stream)

    launches_per_step = 0
    R.render_loss(stream); launches_per_step += B.radt_last_launch_count()
    R.render_bwd(stream=stream); launches_per_step += B.radt_last_launch_count()

    for _ in range(max(args.warmup, 3)):
        flush()
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    torch.cuda.synchronize()
    events = []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        step()
        e1.record(stream)
        events.append((e0, e1))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    ms_total = sum(a.elapsed_time(b) for a, b in events)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=R.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    loss = float(R.loss.cpu())
    ms_step = ms_total / args.steps
    value = world * nominal * args.steps / (ms_total * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- per-kernel device times (forward march, adjoint march) and work counters
    reps = max(5, min(args.steps, 30))
    t_fwd = time_kernel_group(lambda: R.render(stream), stream, torch, flush, reps)
    cnt = R.counters()
    t_fl = time_kernel_group(lambda: R.render_loss(stream), stream, torch, flush, reps)
    t_l2 = time_kernel_group(lambda: R.l2_loss_grad(stream), stream, torch, flush, reps)
    t_bwd = time_kernel_group(lambda: R.render_bwd(stream=stream), stream, torch, flush, reps)
    cnt_b = R.counters()
    # the exact shortcut of the paper's fit chain: no march of the steps without opacity
    B.radt_set_option(B.OPT_ZERO_DENS_GRAD, 0)
    t_bwd_fit = time_kernel_group(lambda: R.render_bwd(stream=stream), stream, torch, flush, reps)
    B.radt_set_option(B.OPT_ZERO_DENS_GRAD, 1)
    fwd_exec = cnt[1] * 32 // 2        # executed samples, 2 MUFU.EX2 lane-ops each
    bwd_exec = cnt_b[3] * 32 // 2      # 2-EX2 equivalents (zero-opacity adjoint samples need one EX2: counted as 1/2)

    # ---- physics pre-pass: T grid -> n_CO, v_phi and its adjoint, timed beside the step
    prepass = None
    if scenes[0].grid.kind == 0 and scenes[0].grid.mirror_z and len(scenes) <= 16:
        from types import SimpleNamespace
        disks = B.make_disks([SimpleNamespace(gm_star=2.0 * 1.32712440018e26, m_gas=2.37 * 1.66053906660e-24, sigma0=30.0,
                                              r_c=150.0, gamma=1.0, x_co=1e-4, t_freeze=19.0, n_dissoc=1e21, f_col=0.706)
                              for _ in scenes])
        pws = torch.empty(B.radt_disk_workspace_bytes(R.desc), dtype=torch.uint8, device=R.device)
        pd, pv, pg = torch.empty_like(R.temp), torch.empty_like(R.temp), torch.zeros_like(R.temp)
        t_pf = time_kernel_group(lambda: B.radt_disk_fields(disks, R.desc, R.temp, pd, pv, pws, stream), stream, torch, flush, reps)
        t_pb = time_kernel_group(lambda: B.radt_disk_fields_bwd(disks, R.desc, R.temp, R.g_dens, R.g_vel, pg, pws, stream),
                                 stream, torch, flush, reps)
        mlp = B.make_mlp(L=4)
        mp = torch.zeros(B.radt_mlp_num_params(mlp), dtype=torch.float32, device=R.device).uniform_(-0.1, 0.1)
        mg, mt = torch.empty_like(mp), torch.empty_like(R.temp[0])
        t_mf = time_kernel_group(lambda: B.radt_mlp_temperature(mlp, R.desc, mp, mt, stream), stream, torch, flush, reps)
        t_mb = time_kernel_group(lambda: B.radt_mlp_temperature_bwd(mlp, R.desc, mp, pg[0], mg, stream), stream, torch, flush, reps)
        prepass = {"fwd_ms": t_pf, "bwd_ms": t_pb, "mlp_fwd_ms": t_mf, "mlp_bwd_ms": t_mb,
                   "what": "radt_disk_fields(_bwd): T grid -> n_CO, v_phi; radt_mlp_temperature(_bwd): parameters -> T grid "
                           "(one grid); both outside the timed step, each figure includes the host-side enqueue"}

    # ---- roofline: SFU (MUFU.EX2) issue peak measured now, at the clock the GPU runs at
    mufu_peak, mufu_clk = B.radt_pipe_peak(0)
    ffma_peak, _ = B.radt_pipe_peak(1)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.txt")      # one JSON object: DRAM bytes per launch from the ncu capture
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath))
        except Exception:      # noqa: BLE001
            traffic = None

    def roof(kernel, t_ms, exec_samples, key, ops, peak, unit, why):
        """ALGORITHMIC lane-operations of the executed samples (per-sample figure x samples one
        launch executes) over the launch time, against the issue peak of the pipe that binds, measured in this run."""
        achieved = ops * exec_samples / (t_ms * 1e-3)
        return {"kernel": kernel, "bound": "alu", "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": unit,
                "frac": achieved / peak, "frac_nominal": ops * nominal / (t_ms * 1e-3) / peak,
                "frac_mufu": 2.0 * exec_samples / (t_ms * 1e-3) / mufu_peak,
                "ops_per_sample": ops, "executed_samples": exec_samples, "ms": t_ms,
                "peak_source": f"{why}, measured by radt_pipe_peak in this run at {mufu_clk:.0f} MHz "
                               "(MEASURED_PEAKS.json holds no SFU/FP32 issue figure)",
                "traffic": (traffic or {}).get(key)}

    # forward: 2 MUFU.EX2 + ~8 FP32 per sample -> the SFU pipe (16 lanes/clk/SM) binds before FP32 (128 lanes/clk/SM);
    # adjoint: 2 MUFU.EX2 + ~20 FP32 per sample -> 20/128 > 2/16: FP32 issue binds
    r_f = roof("k_march_fwd (includes the fused setup launch)", t_fwd, fwd_exec, "k_march_fwd", 2.0, mufu_peak,
               "T MUFU lane-op/s", "SFU issue peak (MUFU.EX2)")
    r_b = roof("k_march_bwd (includes setup and gradient unpack)", t_bwd, bwd_exec, "k_march_bwd", 20.0, ffma_peak,
               "T FP32 lane-op/s", "FP32 issue peak (FFMA)")
    dominant, other = (r_b, r_f) if t_bwd >= t_fwd else (r_f, r_b)

    # ---- e2e: the same step through the HOST-buffer C-ABI entry point, pinned host memory
    d = R.desc
    hf = [torch.from_numpy(h).pin_memory() for h in B.stack_fields(scenes)]
    ht = torch.from_numpy(np.ascontiguousarray(tgt, np.float32)).pin_memory()
    hg = [torch.empty_like(h).pin_memory() for h in hf]
    e2e_steps = max(3, min(args.steps, 50))
    for _ in range(max(args.warmup, 10)):      # the stream-ordered pool and the copy engines need a few calls to settle
        B.radt_fit_step_host(d, *[h.numpy() for h in hf], ht.numpy(), sig, None, *[g.numpy() for g in hg])
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.radt_fit_step_host(d, *[h.numpy() for h in hf], ht.numpy(), sig, None, *[g.numpy() for g in hg])
    torch.cuda.synchronize()
    e2e_t = (time.perf_counter() - t0) / e2e_steps
    h2d = sum(h.numel() * 4 for h in hf) + ht.numel() * 4
    d2h = sum(g.numel() * 4 for g in hg) + 8

    cpu = cpu_baseline(scenes[0]) if world == 1 and not args.no_cpu_baseline else None

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": _workload_name(args.config), "rays": int(sum(s.nrays for s in scenes)),
                   "channels": d.nchan, "steps_per_ray": d.nstep, "grid": list(d.grid_shape),
                   "nominal_samples_per_step": int(nominal), "parallelism": f"independent disks x{world}",
                   "l2": "flushed between timed steps (256 MiB fill outside the events)",
                   "kernels": "window (uniform channel lattice)" if args.win_path else "channel table"},
        "fwd_value": nominal / (t_fwd * 1e-3), "fwd_ms": t_fwd, "fwd_loss_fused_ms": t_fl, "l2_ms": t_l2, "bwd_ms": t_bwd,
        "bwd_ms_zero_dens_grad_off": t_bwd_fit,
        "executed_samples": {"fwd": int(fwd_exec), "bwd": int(bwd_exec), "fwd_active_ray_steps": int(cnt[0]),
                             "bwd_active_ray_steps": int(cnt_b[2]), "nominal": int(nominal)},
        "prepass": prepass,
        "roofline": dominant, "roofline_other": other,
        "pipe_peaks": {"mufu_lane_ops_per_s": mufu_peak, "ffma_lane_ops_per_s": ffma_peak, "sm_mhz": mufu_clk},
        "cpu_baseline": cpu,
        "e2e": {"value": nominal / e2e_t, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": 1e3 * e2e_t, "api": "radt_fit_step_host (pinned host buffers)"},
        "gpu_launches": int(launches_per_step * args.steps),
        "clocks": clocks, "loss": loss, "wall_s": t_wall,
        "context": "paper: ~10,000x vs RADMC-3D, ~100 ms per cube, A6000 vs Xeon Gold 6348 (PAPER.md:302-304); another machine and workload",
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=2, help="SURVEY.md config 1..5 (BASELINE.json configs[k-1]); 6 = spherical 512x96x256 grid at 256x256 px, the shape "
                         "of the paper's own timing benchmark")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--win-path", type=int, default=1, choices=[0, 1],
                    help="RADT_OPT_WIN_PATH: 1 = window kernels on uniform channel lattices (default), 0 = channel-table kernels")
    ap.add_argument("--sph-npix", type=int, default=256, help="config 6: image size (the paper sweeps it at 20 channels)")
    ap.add_argument("--sph-nchan", type=int, default=64, help="config 6: channels of 0.1 km/s (the paper sweeps them at 256 px)")
    args = ap.parse_args()
    _SPH.update(npix=args.sph_npix, nchan=args.sph_nchan)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
