#!/usr/bin/env python
"""Benchmark of the line-RT render hot path (BASELINE.json metric: ray.channel.step samples/s, fwd and fwd+bwd).

A *step* is one pass of the whole hot path over one synthetic workload: ray geometry + forward march with the chi^2 data
term fused into its epilogue (radt_render_loss, low-order words kept) -> memory-free adjoint reusing the forward's setup
(SURVEY.md section 8(a) rows a-j).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k | --configs 1,2,...] [--impl ours|reference]

ONE run measures every config (BASELINE.json configs[0..4] = 1..5, and 6 = the stand-in for the paper's own timing benchmark,
a 512 x 96 x 256 spherical grid) and rank 0 prints ONE JSON line of less than 3 KB.  Its `value`, `ms_per_step`,
`config.workload`, `roofline`, `e2e`, `cpu_baseline` are those of the HEADLINE workload: config 5 (16 x 512^2 px x 128 channels x
512 steps, 2.75e11 nominal samples), the largest single-GPU configuration; `per_config_ms` has one short row per config and
gpurun_out/bench_detail.json (named in `detail_file`) carries every measurement of every config, the pre-pass times and the
work counters.
With N > 1 every rank renders its own disks (independent problems, no data-path collective): weak scaling.  `--shard` instead
splits ONE job (config 5's 16 disks) over the ranks through shard.ShardedRender: whole items per rank
and one all-gather of the packed gradient cells per step (rows and an all-reduce when there are more ranks than items); strong
scaling, `value` = the job's samples / max-over-ranks time.

`value` = nominal samples (rays x channels x steps, summed over ranks and steps) / device time of the K steps (inputs resident
in HBM; L2 flushed between steps outside the timed events).  `e2e` = the same step through the HOST-buffer C-ABI entry point
radt_fit_step_host (pinned host buffers, copies inside the timed region); `e2e_render` = radt_render_host (cube D2H inside).
`roofline` = the dominant kernel against the issue peak measured in this run: `frac` counts EXECUTED
samples only; `speedup_from_skipping` = nominal / executed samples (an algorithmic saving, not pipe efficiency);
`executed_samples.fwd_in_window_over_executed` = the share of executed (channel, step) samples that lie inside their step's line
window, i.e. of the 32 lanes that can contribute (useful over executed work).
`cpu_baseline` = the fp64 oracle, as it stands, on this box's host cores, on a bounded ray sample of the headline workload.
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
HEADLINE = 5
ALL_CONFIGS = (1, 2, 3, 4, 5, 6)

_SPH = {"npix": 256, "nchan": 64}       # config 6 image size and channel count (--sph-npix / --sph-nchan sweep them)


def _scenes(cfg):
    """Configs 1-5: BASELINE.json configs[0..4]; 6: stand-in for the paper's own timing benchmark."""
    from synth import make_config, sph_benchmark_scene
    s = sph_benchmark_scene(npix=_SPH["npix"], nchan=_SPH["nchan"]) if cfg == 6 else make_config(cfg)
    return s if isinstance(s, list) else [s]


def _workload_name(cfg):
    from synth import config_names
    return f"cfg6_sph512x96x256_img{_SPH['npix']}_c{_SPH['nchan']}_n256" if cfg == 6 else config_names()[cfg]


def _config_dict(cfg, scenes, world):
    """The workload description: the same dict in both arms (ours and --impl reference)."""
    s0 = scenes[0]
    return {"workload": _workload_name(cfg), "rays": int(sum(s.nrays for s in scenes)), "channels": int(len(s0.line.vchan)),
            "steps_per_ray": int(s0.geom.nstep), "grid": [int(n) for n in s0.grid.n], "batch": len(scenes),
            "nominal_samples_per_step": int(sum(s.nominal_samples for s in scenes)),
            "parallelism": f"independent disks x{world}",
            "l2": "flushed between timed steps (256 MiB fill)"}


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
def _subset(scene, stride_xy):
    """Every `stride_xy`-th row and column of the image (SURVEY.md:328 allows this ray subset for the large configs)."""
    ny, nx = scene.geom.ny, scene.geom.nx
    iy, ix = np.arange(0, ny, stride_xy), np.arange(0, nx, stride_xy)
    return (iy[:, None] * nx + ix[None, :]).reshape(-1).astype(np.int64)


def oracle_pass(scene, idx):
    """One fwd + adjoint pass of the oracle over rays `idx` of `scene`; returns (seconds, samples)."""
    from oracle import pyoracle as po
    t0 = time.perf_counter()
    cube = po.render(scene, rays=idx)
    po.render_bwd(scene, cube * 1e-6, rays=idx)
    dt = time.perf_counter() - t0
    return dt, len(idx) * len(scene.line.vchan) * scene.geom.nstep


def _sample_stride(scenes, budget_s, npasses):
    """Row/column stride such that `npasses` oracle passes over the subset of ALL scenes take about budget_s."""
    probe = _subset(scenes[0], 32)
    oracle_pass(scenes[0], probe[:64])                      # load the library, touch the pages
    dt, n = oracle_pass(scenes[0], probe)
    rate = n / dt                                           # samples / s
    total = sum(s.nominal_samples for s in scenes)
    want = max(rate * budget_s / max(npasses, 1), 1.0)      # samples per pass
    return int(min(max(np.ceil(np.sqrt(total / want)), 1), 64))


def cpu_baseline(scenes, name, budget_s=12.0):
    """The oracle as it stands on this box's host cores: whole fwd + adjoint passes over a fixed ray subset of every batch
    item (every s-th row and column), repeated until about `budget_s` seconds of wall time (>= 2 passes)."""
    from oracle import pyoracle as po
    stride = _sample_stride(scenes, budget_s, 2)
    tot_t, tot_n, passes = 0.0, 0, 0
    while passes < 2 or tot_t < budget_s:
        for sc in scenes:
            dt, n = oracle_pass(sc, _subset(sc, stride))
            tot_t += dt
            tot_n += n
        passes += 1
    cores = po.num_threads()
    # the same oracle on ONE thread: the per-core figure SURVEY.md section 8(d) asks for
    po.set_num_threads(1)
    dt1, n1 = oracle_pass(scenes[0], _subset(scenes[0], max(4 * stride, 16)))
    po.set_num_threads(cores)
    return {"value": tot_n / tot_t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{name}: {passes} passes over every {stride}th row and column of all {len(scenes)} item(s) "
                      f"({tot_n:.3g} samples), fp64 forward + adjoint, {tot_t:.1f} s wall",
            "value_1thread": n1 / dt1}


def run_reference(args, configs):
    """--impl reference: the reference arm of this tier is the fp64 CPU oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import pyoracle as po
    cfg = configs[-1] if len(configs) == 1 else HEADLINE
    scenes = _scenes(cfg)
    # size the per-step ray sample so that the whole run stays within ~100 s on this box
    stride = _sample_stride(scenes, 100.0, args.steps + args.warmup)
    subsets = [_subset(sc, stride) for sc in scenes]

    def step():
        t, n = 0.0, 0
        for sc, idx in zip(scenes, subsets):
            dt, nn = oracle_pass(sc, idx)
            t += dt
            n += nn
        return t, n

    for _ in range(args.warmup):
        step()
    tot_t, tot_n = 0.0, 0
    for _ in range(args.steps):
        dt, n = step()
        tot_t += dt
        tot_n += n
    val = tot_n / tot_t
    sample = f"every {stride}th row and column of all {len(scenes)} item(s) of {_workload_name(cfg)} per step, fwd + adjoint"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _config_dict(cfg, scenes, 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": po.num_threads(), "kind": "oracle", "sample": sample},
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


def aggregate_ms(ms_total, ctx):
    """Time of the K steps as the MAX over ranks (device timing per rank; one all-reduce on the rank's own device)."""
    if ctx["world"] == 1:
        return ms_total
    torch, dist = ctx["torch"], ctx["dist"]
    t = torch.tensor([ms_total], dtype=torch.float64, device=ctx["reduce_device"])
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(nominal_per_rank, steps, ms_total_max, world):
    """Aggregate throughput over all ranks: every rank processes `nominal_per_rank` samples per step (weak scaling)."""
    return world * nominal_per_rank * steps / (ms_total_max * 1e-3)


def measure_config_dry(cfg, args, ctx, with_cpu):
    """--dry-run: no GPU work.  Every rank 'takes' (1 + rank) x 1 ms per step; exercises the rank / barrier / max-over-ranks /
    aggregation / rank-0-prints logic of the multi-rank bench on CPU (gloo), tests/test_shard_gloo.py."""
    world, rank = ctx["world"], ctx["rank"]
    nominal = {1: 3932160, 2: 1073741824, 3: 17179869184, 4: 8589934592, 5: 274877906944, 6: 1073741824}[cfg]
    if world > 1:
        ctx["dist"].barrier()
    ms_total = aggregate_ms(args.steps * 1.0 * (1 + rank), ctx)
    if world > 1:
        ctx["dist"].barrier()
    if rank != 0:
        return None
    res = {k: None for k in ("fwd_value", "fwd_ms", "fwd_loss_fused_ms", "l2_ms", "bwd_ms", "bwd_ms_own_setup",
                             "bwd_ms_zero_dens_grad_off", "step_ms_without_cube_lo", "executed_samples", "roofline",
                             "roofline_other", "e2e", "e2e_render", "launches_per_step", "clocks", "cpu_baseline", "loss",
                             "wall_s")}
    res.update(config={"workload": _workload_name(cfg), "nominal_samples_per_step": nominal, "parallelism": f"independent disks x{world}"},
               value=whole_job_value(nominal, args.steps, ms_total, world), unit=UNIT, steps=args.steps,
               warmup=max(args.warmup, 3), ms_per_step=ms_total / args.steps, gpu_launches=0)
    return res


class _DryEngine:
    """--dry-run --shard: stands in for shard.CudaEngine with zero tensors of the right shapes (no render, no oracle)."""

    def __init__(self, scenes):
        import torch
        self.torch, self.n = torch, len(scenes)
        self.cells = int(np.prod(scenes[0].grid.n))

    def set_target(self, target, sigma):
        pass

    def fit_step_packed(self):
        return self.torch.zeros((self.n, self.cells * 4)), self.torch.zeros(1, dtype=self.torch.float64)


def measure_config_shard(cfg, args, ctx, with_cpu):
    """--shard: ONE job (the config's whole batch) split over the ranks by shard.plan_units (batch items first, rows second;
    SURVEY.md section 8(e)): per step every rank runs forward + fused chi^2 + adjoint of its units and the ranks exchange the
    packed gradient cells with ONE collective (all-gather for whole items, all-reduce for split rows).  Strong scaling:
    `value` = the job's nominal samples / max-over-ranks device time."""
    from paper_2509_03623_b200.shard import ShardedRender
    torch, dist = ctx["torch"], ctx["dist"]
    world, rank, local = ctx["world"], ctx["rank"], ctx["local"]
    dry = args.dry_run
    if world > 1 or not dry:
        assert dist.is_initialized(), "--shard needs a process group (torch.distributed.run sets it up)"
    if dry:
        from synth import make_config
        scenes = make_config(cfg, npix=8) if cfg != 6 else _scenes(cfg)
        scenes = scenes if isinstance(scenes, list) else [scenes]
        nominal = {1: 3932160, 2: 1073741824, 3: 17179869184, 4: 8589934592, 5: 274877906944, 6: 1073741824}[cfg]
        sh = ShardedRender(scenes, _DryEngine)
    else:
        from paper_2509_03623_b200.shard import CudaEngine
        scenes = _scenes(cfg)
        nominal = sum(s.nominal_samples for s in scenes)
        sh = ShardedRender(scenes, lambda group: CudaEngine(group, f"cuda:{local}"))
        slabs = sh.render()
        gen = torch.Generator(device=f"cuda:{local}").manual_seed(36230 + cfg + 97 * rank)
        peak = max([float(v.amax()) for v in slabs.values()] or [1.0])
        sig = 0.015 * peak
        sh.set_targets({u: v * (1.0 + 0.05 * torch.randn(v.shape, generator=gen, device=v.device))
                        + sig * torch.randn(v.shape, generator=gen, device=v.device) for u, v in slabs.items()}, sig)
        del slabs
    warm = max(args.warmup, 3)
    for _ in range(warm if not dry else 1):
        sh.fit_step()
    n0 = sh.n_collectives
    if dry:
        if world > 1:
            dist.barrier()
        for _ in range(args.steps):
            sh.fit_step()
        ms_local, clocks = args.steps * 1.0 * (1 + rank), None
    else:
        stream = torch.cuda.current_stream()
        torch.cuda.synchronize()
        dist.barrier()
        sampler = ClockSampler(local)
        sampler.start()
        torch.cuda.synchronize()
        events = []
        for _ in range(args.steps):
            ctx["flush_buf"].fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            sh.fit_step()
            e1.record(stream)
            events.append((e0, e1))
        torch.cuda.synchronize()
        dist.barrier()
        clocks = sampler.stop()
        ms_local = sum(a.elapsed_time(b) for a, b in events)
    per_step = (sh.n_collectives - n0) / args.steps
    ms_total = aggregate_ms(ms_local, ctx)
    if world > 1:
        dist.barrier()
    if rank != 0:
        return None
    res = {k: None for k in ("fwd_value", "fwd_ms", "fwd_loss_fused_ms", "l2_ms", "bwd_ms", "bwd_ms_own_setup",
                             "bwd_ms_zero_dens_grad_off", "step_ms_without_cube_lo", "executed_samples", "roofline",
                             "roofline_other", "e2e", "e2e_render", "launches_per_step", "cpu_baseline", "loss", "wall_s")}
    res.update(config={"workload": _workload_name(cfg), "nominal_samples_per_step": int(nominal),
                       "parallelism": f"one job sharded over {world} rank(s): {len(sh.units)} unit(s) on rank 0, {sh.collective} of the packed gradient cells"},
               value=nominal * args.steps / (ms_total * 1e-3), unit=UNIT, steps=args.steps, warmup=warm,
               ms_per_step=ms_total / args.steps, clocks=clocks, scaling="strong",
               gpu_launches=0 if dry else int(5 * len(sh.groups) * args.steps),
               shard={"collective": sh.collective, "collectives_per_step": per_step, "units_per_rank": [len(us) for us in sh.plan]})
    return res


def _load_traffic():
    """DRAM bytes per launch from the committed ncu captures (profiles/traffic_r02.json, one entry per config and kernel);
    configs without a capture report null."""
    path = os.path.join(ROOT, "profiles", "traffic_r02.json")
    try:
        with open(path) as f:
            return json.load(f)
    except Exception:      # noqa: BLE001
        return {}


def measure_config(cfg, args, ctx, with_cpu):
    """All measurements of one config on this rank; rank 0 gets the full dict."""
    torch, dist, B, Renderer = ctx["torch"], ctx["dist"], ctx["B"], ctx["Renderer"]
    world, rank, local = ctx["world"], ctx["rank"], ctx["local"]
    scenes = _scenes(cfg)
    R = Renderer(scenes, device=f"cuda:{local}", options=dict(win_path=args.win_path))
    stream = torch.cuda.current_stream()
    nominal = sum(s.nominal_samples for s in scenes)
    d = R.desc

    # target cube of the L2 data term, D = I (1 + 0.05 xi) + sigma eta, sigma = 0.015 max I, built from a
    # first render before timing; drawn on the device (torch Philox, seeded) so that the 2 GB of config 5 take no host time
    R.render()
    gen = torch.Generator(device=R.device).manual_seed(36230 + cfg + 97 * rank)
    sig = 0.015 * float(R.cube.amax())
    tgt = torch.empty_like(R.cube)
    for b in range(R.cube.shape[0]):          # item by item: no second cube-sized temporary
        tgt[b] = R.cube[b] * (1.0 + 0.05 * torch.randn(R.cube[b].shape, generator=gen, device=R.device))
        tgt[b] += sig * torch.randn(R.cube[b].shape, generator=gen, device=R.device)
    R.set_target(tgt, sig)
    del tgt

    flush_buf = ctx["flush_buf"]

    def flush():
        flush_buf.fill_(1)

    def step():
        R.fit_step(stream)

    launches_per_step = 0
    R.render_loss(stream); launches_per_step += B.radt_last_launch_count()
    R.render_bwd(stream=stream, reuse_setup=True); launches_per_step += B.radt_last_launch_count()

    warm = max(args.warmup, 3)
    for _ in range(warm):
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
    ms_total = aggregate_ms(sum(a.elapsed_time(b) for a, b in events), ctx)
    loss = float(R.loss.cpu())
    ms_step = ms_total / args.steps
    value = whole_job_value(nominal, args.steps, ms_total, world)
    if rank != 0:
        return None

    # ---- per-kernel device times (forward march, adjoint march) and work counters
    reps = max(3, min(args.steps, 20 if nominal < 1e11 else 5))
    t_fwd = time_kernel_group(lambda: R.render(stream), stream, torch, flush, reps)
    cnt = R.counters()
    lanes = R.lane_counters()          # (samples inside their step's line window, samples executed) of that forward
    t_fl = time_kernel_group(lambda: R.render_loss(stream), stream, torch, flush, reps)
    t_l2 = time_kernel_group(lambda: R.l2_loss_grad(stream), stream, torch, flush, reps)
    R.render_loss(stream)
    t_bwd = time_kernel_group(lambda: R.render_bwd(stream=stream, reuse_setup=True), stream, torch, flush, reps)
    cnt_b = R.counters()
    t_bwd_own = time_kernel_group(lambda: R.render_bwd(stream=stream), stream, torch, flush, reps)
    # the exact shortcut of the paper's fit chain: no march of the steps without opacity
    R.set_options(zero_dens_grad=0)
    R.render_loss(stream)
    t_bwd_fit = time_kernel_group(lambda: R.render_bwd(stream=stream, reuse_setup=True), stream, torch, flush, reps)
    R.set_options(zero_dens_grad=1)
    # without the low-order words (cube_lo = NULL): what the compensation costs
    Rp = None
    t_plain = None
    if nominal < 1e11:
        Rp = Renderer(scenes, device=f"cuda:{local}", options=dict(win_path=args.win_path), compensated=False)
        Rp.set_target(R.target, sig)
        Rp.fit_step(stream)
        t_plain = time_kernel_group(lambda: Rp.fit_step(stream), stream, torch, flush, reps)
        del Rp
    fwd_exec = cnt[1] * 32 // 2        # executed samples, 2 MUFU.EX2 lane-ops each
    bwd_exec = cnt_b[3] * 32 // 2      # 2-EX2 equivalents (zero-opacity adjoint samples need one EX2: counted as 1/2)

    mufu_peak, ffma_peak, mufu_clk = ctx["mufu_peak"], ctx["ffma_peak"], ctx["mufu_clk"]
    traffic = ctx["traffic"].get(f"cfg{cfg}", {})

    def roof(kernel, t_ms, exec_samples, key, ops, peak, unit, why):
        """ALGORITHMIC lane-operations of the EXECUTED samples (per-sample figure x samples one launch
        executes) over the launch time, against the issue peak of the pipe that binds, measured in this run."""
        achieved = ops * exec_samples / (t_ms * 1e-3)
        return {"kernel": kernel, "bound": "alu", "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": unit,
                "frac": achieved / peak,
                "frac_mufu": 2.0 * exec_samples / (t_ms * 1e-3) / mufu_peak,
                "speedup_from_skipping": nominal / max(exec_samples, 1),
                "ops_per_sample": ops, "executed_samples": int(exec_samples), "ms": t_ms,
                "peak_source": f"{why}, radt_pipe_peak in this run at {mufu_clk:.0f} MHz",
                "traffic": traffic.get(key)}

    # forward: 2 MUFU.EX2 + ~8 FP32 per sample -> the SFU pipe (16 lanes/clk/SM) binds before FP32 (128 lanes/clk/SM);
    # adjoint: 2 MUFU.EX2 + ~20 FP32 per sample -> 20/128 > 2/16: FP32 issue binds
    r_f = roof("k_march_fwd (includes the fused setup launch)", t_fwd, fwd_exec, "k_march_fwd", 2.0, mufu_peak,
               "T MUFU lane-op/s", "SFU issue peak (MUFU.EX2)")
    r_b = roof("k_march_bwd (adjoint march + gradient unpack, setup reused from the forward)", t_bwd, bwd_exec, "k_march_bwd", 20.0,
               ffma_peak, "T FP32 lane-op/s", "FP32 issue peak (FFMA)")
    dominant, other = (r_b, r_f) if t_bwd >= t_fwd else (r_f, r_b)

    # ---- e2e: the same step through the HOST-buffer C-ABI entry points, pinned host memory
    hf = [torch.from_numpy(h).pin_memory() for h in B.stack_fields(scenes)]
    ht = torch.empty(R.target.shape, dtype=torch.float32, pin_memory=True)
    ht.copy_(R.target)
    hg = [torch.empty_like(h).pin_memory() for h in hf]
    hc = torch.empty(R.cube.shape, dtype=torch.float32, pin_memory=True)
    nvox = R.cube.numel()
    del R
    torch.cuda.empty_cache()
    big = nominal > 1e10
    e2e_steps = max(3, min(args.steps, 5 if big else 50))
    for _ in range(2 if big else max(args.warmup, 10)):      # the arena and the copy engines need a few calls to settle
        B.radt_fit_step_host(d, *[h.numpy() for h in hf], ht.numpy(), sig, None, *[g.numpy() for g in hg])
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.radt_fit_step_host(d, *[h.numpy() for h in hf], ht.numpy(), sig, None, *[g.numpy() for g in hg])
    torch.cuda.synchronize()
    e2e_t = (time.perf_counter() - t0) / e2e_steps
    h2d = sum(h.numel() * 4 for h in hf) + ht.numel() * 4
    d2h = sum(g.numel() * 4 for g in hg) + 8
    for _ in range(2):
        B.radt_render_host(d, *[h.numpy() for h in hf], hc.numpy())
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.radt_render_host(d, *[h.numpy() for h in hf], hc.numpy())
    e2e_r = (time.perf_counter() - t0) / e2e_steps
    del ht, hc

    cpu = cpu_baseline(scenes, _workload_name(cfg)) if with_cpu else None

    return {
        "config": _config_dict(cfg, scenes, world), "value": value, "unit": UNIT, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_step, "fwd_value": nominal / (t_fwd * 1e-3),
        "fwd_ms": t_fwd, "fwd_loss_fused_ms": t_fl, "l2_ms": t_l2, "bwd_ms": t_bwd, "bwd_ms_own_setup": t_bwd_own,
        "bwd_ms_zero_dens_grad_off": t_bwd_fit, "step_ms_without_cube_lo": t_plain,
        "executed_samples": {"fwd": int(fwd_exec), "bwd": int(bwd_exec), "fwd_active_ray_steps": int(cnt[0]),
                             "bwd_active_ray_steps": int(cnt_b[2]), "nominal": int(nominal),
                             "fwd_executed_over_nominal": fwd_exec / nominal,
                             "fwd_in_window": int(lanes[0]) if lanes[0] else None,
                             "fwd_in_window_over_executed": (lanes[0] / max(lanes[1], 1)) if lanes[0] else None},
        "roofline": dominant, "roofline_other": other,
        "e2e": {"value": nominal / e2e_t, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": 1e3 * e2e_t, "steps": e2e_steps, "api": "radt_fit_step_host (pinned host buffers)"},
        "e2e_render": {"value": nominal / e2e_r, "unit": "samples/s (forward only)", "h2d_bytes_per_step": int(sum(h.numel() * 4 for h in hf)),
                       "d2h_bytes_per_step": int(nvox * 4), "ms_per_step": 1e3 * e2e_r, "api": "radt_render_host (cube D2H inside)"},
        "gpu_launches": int(launches_per_step * args.steps), "launches_per_step": int(launches_per_step),
        "clocks": clocks, "loss": loss, "wall_s": t_wall, "cpu_baseline": cpu,
    }


def prepass_times(ctx, args):
    """Physics pre-pass and MLP field on the config-2 grid, timed beside the step."""
    from types import SimpleNamespace
    torch, B, Renderer = ctx["torch"], ctx["B"], ctx["Renderer"]
    scenes = _scenes(2)
    R = Renderer(scenes, device=f"cuda:{ctx['local']}")
    stream = torch.cuda.current_stream()
    R.render(); R.dl_dcube.fill_(1e-9); R.render_bwd()

    def flush():
        ctx["flush_buf"].fill_(1)
    reps = 10
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
    return {"grid": "config 2 (256 x 128)", "fwd_ms": t_pf, "bwd_ms": t_pb, "mlp_fwd_ms": t_mf, "mlp_bwd_ms": t_mb,
            "what": "radt_disk_fields(_bwd): T grid -> n_CO, v_phi; radt_mlp_temperature(_bwd): parameters -> T grid "
                    "(one grid); both outside the timed step, each figure includes the host-side enqueue"}


def _clean(x, sig=6):
    """JSON-safe copy: floats rounded to `sig` significant digits, NaN / Infinity -> null, numpy scalars -> Python."""
    if isinstance(x, dict):
        return {str(k): _clean(v, sig) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_clean(v, sig) for v in x]
    if isinstance(x, (bool, type(None), str)):
        return x
    if isinstance(x, (int, np.integer)):
        return int(x)
    if isinstance(x, (float, np.floating)):
        x = float(x)
        return float(f"{x:.{sig}g}") if np.isfinite(x) else None
    return str(x)


MAX_LINE_BYTES = 3000       # the driver reads the LAST stdout line; round 2's 20.5 KB line did not parse


def headline_line(H, results, configs, world, args, dry=False):
    """The ONE stdout line: the headline workload only, < MAX_LINE_BYTES.  Everything else (all six per-config dicts, pre-pass
    times, counters) goes to the detail file (write_detail)."""
    def roof(r):
        if not r:
            return None
        return {k: r[k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic", "ms", "executed_samples",
                                  "ops_per_sample", "peak_source") if k in r}

    def e2e(e):
        return {k: e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step")} if e else None

    def summary(r):         # one short row per config: [step ms, forward ms, adjoint ms, forward frac, adjoint frac, e2e step ms]
        rf, rb = r.get("roofline"), r.get("roofline_other")
        if rf and rb and rf["kernel"].startswith("k_march_bwd"):
            rf, rb = rb, rf
        return [r.get("ms_per_step"), r.get("fwd_ms"), r.get("bwd_ms"), rf and rf["frac"], rb and rb["frac"],
                r.get("e2e") and r["e2e"]["ms_per_step"]]

    cpu = H.get("cpu_baseline")
    if cpu:
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "value_1thread") if k in cpu}
    clocks = H.get("clocks")
    line = {
        "metric": METRIC, "value": H["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": H["warmup"],
        "ms_per_step": H["ms_per_step"], "higher_is_better": True, "scaling": H.get("scaling", "weak"), "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": H["config"],
        "roofline": roof(H.get("roofline")), "roofline_other": roof(H.get("roofline_other")),
        "cpu_baseline": cpu, "e2e": e2e(H.get("e2e")), "e2e_render": e2e(H.get("e2e_render")),
        "gpu_launches": H["gpu_launches"], "clocks": clocks,
        "fwd_ms": H.get("fwd_ms"), "bwd_ms": H.get("bwd_ms"),
        "per_config_ms": {"columns": "step,fwd,bwd,frac_fwd,frac_bwd,e2e_step",
                          **{f"cfg{c}": summary(results[c]) for c in configs}},
    }
    if H.get("shard"):
        line["shard"] = H["shard"]
    if dry:
        line["dry_run"] = True
    line = _clean(line)
    # belt and braces: never let an unforeseen long string push the line past the limit
    for drop in ("per_config_ms", "roofline_other", "e2e_render"):
        if len(json.dumps(line, separators=(",", ":"))) <= MAX_LINE_BYTES:
            break
        line.pop(drop, None)
    return line


def write_detail(detail, args):
    """Everything that is not the headline: one JSON file under gpurun_out/ (the folder that comes back from a GPU box; never
    read by anything committed).  Returns the path relative to the repository, or null if the folder cannot be written."""
    rel = os.path.join("gpurun_out", "bench_detail.json")
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, rel), "w") as f:
            json.dump(_clean(detail, 9), f, indent=1, allow_nan=False)
        return rel
    except OSError:
        return None


def run_ours(args, configs):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dry = args.dry_run
    if not dry and not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the render has no CPU fallback")
    ctx = {"torch": torch, "dist": dist, "world": world, "rank": rank, "local": local, "traffic": _load_traffic()}
    if dry:
        if world > 1:
            dist.init_process_group("gloo")
        ctx["reduce_device"] = "cpu"
        ctx["mufu_peak"] = ctx["ffma_peak"] = ctx["mufu_clk"] = None
        measure = measure_config_dry
        if args.shard and world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29517")
            dist.init_process_group("gloo", rank=0, world_size=1)
    else:
        from paper_2509_03623_b200 import Renderer, binding as B
        torch.cuda.set_device(local)
        if world > 1 or args.shard:
            # NCCL_DEBUG=INFO (if the launcher sets it) shows the ranks and NVLS; without --shard the only collectives of this
            # bench are the barriers around the timed region and the max-over-ranks of its duration
            if world == 1:
                os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
                os.environ.setdefault("MASTER_PORT", "29517")
            dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
        B.lib()
        ctx.update(B=B, Renderer=Renderer, reduce_device=f"cuda:{local}",
                   flush_buf=torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}"))     # > 126 MB L2
        # roofline denominators: issue peaks measured now, at the clock the GPU runs at
        ctx["mufu_peak"], ctx["mufu_clk"] = B.radt_pipe_peak(0)
        ctx["ffma_peak"], _ = B.radt_pipe_peak(1)
        measure = measure_config
    if args.shard:
        measure = measure_config_shard

    head = configs[0] if len(configs) == 1 else (HEADLINE if HEADLINE in configs else configs[-1])
    results = {}
    t_start = time.perf_counter()
    for cfg in configs:
        t0 = time.perf_counter()
        res = measure(cfg, args, ctx, with_cpu=(cfg == head and world == 1 and not args.no_cpu_baseline))
        if res is not None:
            res["bench_wall_s"] = time.perf_counter() - t0
            results[cfg] = res
        if not dry:
            torch.cuda.empty_cache()
    if rank != 0:
        if dist.is_initialized():
            dist.destroy_process_group()
        return
    prepass = prepass_times(ctx, args) if (world == 1 and not args.no_prepass and not dry and not args.shard) else None

    H = results[head]
    keep = ("config", "value", "ms_per_step", "steps", "fwd_value", "fwd_ms", "fwd_loss_fused_ms", "l2_ms", "bwd_ms",
            "bwd_ms_own_setup", "bwd_ms_zero_dens_grad_off", "step_ms_without_cube_lo", "executed_samples", "roofline",
            "roofline_other", "e2e", "e2e_render", "launches_per_step", "clocks", "bench_wall_s")
    detail = {
        "per_config": [{k: results[c].get(k) for k in keep} for c in configs], "prepass": prepass,
        "pipe_peaks": {"mufu_lane_ops_per_s": ctx["mufu_peak"], "ffma_lane_ops_per_s": ctx["ffma_peak"], "sm_mhz": ctx["mufu_clk"]},
        "executed_samples": H["executed_samples"], "loss": H["loss"], "wall_s": H["wall_s"],
        "kernels": "window (uniform channel lattice)" if args.win_path else "channel table",
        "bench_total_wall_s": time.perf_counter() - t_start,
        "peak_note": "MEASURED_PEAKS.json holds no SFU/FP32 issue figure: the roofline denominators are radt_pipe_peak's, measured in this run",
        "headline_rule": "largest single-GPU configuration of BASELINE.json (configs[4])",
        "context": "paper: ~10,000x vs RADMC-3D, ~100 ms per cube, A6000 vs Xeon Gold 6348 (PAPER.md:302-304); another machine and workload",
    }
    line = headline_line(H, results, configs, world, args, dry)
    if not dry:
        line["detail_file"] = write_detail(detail, args)
    print(json.dumps(line, allow_nan=False, separators=(",", ":")), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=None, help="measure ONE config (1..5 = BASELINE.json configs[k-1]; 6 = spherical "
                    "512x96x256 grid at 256x256 px, the shape of the paper's own timing benchmark); default: all, headline 5")
    ap.add_argument("--configs", type=str, default=None, help="comma-separated subset, e.g. 2,3,5")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-prepass", action="store_true")
    ap.add_argument("--shard", action="store_true", help="ONE job (the headline config's 16 disks) split over the ranks through "
                    "shard.ShardedRender: items first, rows second, one collective per step over the packed gradient cells; strong scaling "
                    "(default without it: every rank renders its own disks, weak scaling)")
    ap.add_argument("--dry-run", action="store_true", help="no GPU work: exercise the multi-rank timing / aggregation logic on CPU (gloo)")
    ap.add_argument("--win-path", type=int, default=1, choices=[0, 1],
                    help="radt_options.win_path: 1 = window kernels on uniform channel lattices (default), 0 = channel-table kernels")
    ap.add_argument("--sph-npix", type=int, default=256, help="config 6: image size (the paper sweeps it at 20 channels)")
    ap.add_argument("--sph-nchan", type=int, default=64, help="config 6: channels of 0.1 km/s (the paper sweeps them at 256 px)")
    args = ap.parse_args()
    _SPH.update(npix=args.sph_npix, nchan=args.sph_nchan)
    if args.config is not None:
        configs = [args.config]
    elif args.configs:
        configs = [int(c) for c in args.configs.split(",")]
    else:
        configs = [HEADLINE] if args.shard else list(ALL_CONFIGS)
    if args.impl == "reference":
        run_reference(args, configs)
    else:
        run_ours(args, configs)


if __name__ == "__main__":
    main()
