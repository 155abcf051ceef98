"""Neural-field fit on a synthetic disk, end to end on one GPU (Fig. 2):

    MLP parameters -> T(r, |z|) grid -> hydrostatic density, CO layer, rotation -> line-RT render -> chi^2
    and all adjoints back to the parameters, ADAM on the parameter vector (learning rate decaying polynomially, as in
    PAPER.md:221).

The "observed" cube is rendered from the config's own parametric temperature grid pushed through the same physics
pre-pass (no ALMA data are available offline), with 1.5 % noise.  Every step of the chain runs in this package's CUDA
kernels; torch supplies device memory and the optimiser's elementwise update only.

    python -m paper_2509_03623_b200.fit_demo --config 2 --steps 300
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time
from types import SimpleNamespace

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import numpy as np
    import torch
    from paper_2509_03623_b200 import Renderer, binding as B
    from synth import make_config

    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3])
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--lr", type=float, default=5e-4)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--full-dens-grad", action="store_true", help="keep RADT_OPT_ZERO_DENS_GRAD on (march the steps without opacity)")
    ap.add_argument("--no-graph", action="store_true", help="enqueue every step from Python instead of replaying one CUDA graph")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("fit_demo needs a CUDA device: there is no CPU fallback")

    sc = make_config(args.config)
    R = Renderer([sc])
    desc = R.desc
    disks = B.make_disks([SimpleNamespace(gm_star=2.0 * 1.32712440018e26, m_gas=2.37 * 1.66053906660e-24, sigma0=30.0,
                                          r_c=150.0, gamma=1.0, x_co=1e-4, t_freeze=19.0, n_dissoc=1e21, f_col=0.706)])
    pws = torch.empty(B.radt_disk_workspace_bytes(desc), dtype=torch.uint8, device=R.device)
    mlp = B.make_mlp(L=4)
    nparams = B.radt_mlp_num_params(mlp)
    # the pre-pass holds the CO mask fixed and discards dL/dn of masked cells: the render adjoint need not march the
    # steps that only feed those cells
    B.radt_set_option(B.OPT_ZERO_DENS_GRAD, 1 if args.full_dens_grad else 0)

    # observed cube: the config's temperature grid through the pre-pass and the render, plus noise
    t_true = R.temp.clone()
    B.radt_disk_fields(disks, desc, R.temp, R.dens, R.vel, pws)
    R.render()
    gen = torch.Generator(device=R.device).manual_seed(36230 + args.seed)
    sigma = 0.015 * float(R.cube.max())
    target = R.cube + sigma * torch.randn(R.cube.shape, generator=gen, device=R.device)
    R.set_target(target, sigma)

    # parameters: uniform +-1/sqrt(fan_in) like the usual linear-layer default
    g = torch.Generator(device="cpu").manual_seed(args.seed)
    D = 2 + 4 * 4
    parts = []
    for fan_in, fan_out in [(D, 64), (64, 64), (64, 64), (64, 64), (64, 1)]:
        k = fan_in ** -0.5
        parts += [(torch.rand(fan_out * fan_in, generator=g) * 2 - 1) * k, (torch.rand(fan_out, generator=g) * 2 - 1) * k]
    params = torch.cat(parts)
    params[-1] = -2.5          # output bias: start near 35 K (a start at the sigmoid's middle, 200 K, overshoots the CO
                               # freeze-out threshold on the way down and the hard mask of Eq. 9 then kills every gradient)
    params = params.to(R.device)
    assert params.numel() == nparams
    params.grad = torch.zeros_like(params)
    use_graph = not args.no_graph
    # the learning rate lives on the device so that the captured optimiser step follows the schedule
    lr_t = torch.tensor(args.lr, device=R.device)
    opt = torch.optim.Adam([params], lr=lr_t if use_graph else args.lr, capturable=use_graph)

    def lr_at(it):                      # polynomial decay to zero, power 2 ("polynomially decays")
        return args.lr * (1.0 - min(it, args.steps) / args.steps) ** 2

    def chain(stream=None):
        B.radt_mlp_temperature(mlp, desc, params, R.temp[0], stream)
        B.radt_disk_fields(disks, desc, R.temp, R.dens, R.vel, pws, stream)
        R.fit_step(stream)                                    # render + chi^2 + render adjoint
        B.radt_disk_fields_bwd(disks, desc, R.temp, R.g_dens, R.g_vel, R.g_temp, pws, stream)
        B.radt_mlp_temperature_bwd(mlp, desc, params, R.g_temp[0], params.grad, stream)
        opt.step()

    graph = None
    if use_graph:
        # every entry point is stream ordered and allocation free, so one fit step is one CUDA graph
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            snap = params.clone()
            for _ in range(3):
                chain(side)                                   # warm-up (also creates the optimiser state)
            params.copy_(snap)
            for st in opt.state.values():
                for v in st.values():
                    if torch.is_tensor(v):
                        v.zero_()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            chain(torch.cuda.current_stream())

    def step(it):
        if use_graph:
            lr_t.fill_(lr_at(it))
            graph.replay()
        else:
            for gp in opt.param_groups:
                gp["lr"] = lr_at(it)
            chain()

    losses = []
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for it in range(args.steps):
        step(it)
        if it % max(1, args.steps // 10) == 0 or it == args.steps - 1:
            losses.append((it, float(R.loss.cpu())))
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    co = (R.dens[0] > 0) & (t_true[0] > 19.0)
    rel = float(((R.temp[0][co] - t_true[0][co]).abs() / t_true[0][co]).median()) if bool(co.any()) else float("nan")
    print(json.dumps({"workload": sc.name, "steps": args.steps, "ms_per_fit_step": 1e3 * dt / args.steps,
                      "fit_steps_per_s": args.steps / dt, "loss": losses,
                      "median_rel_T_error_in_CO_layer": rel, "n_params": nparams,
                      "cuda_graph": use_graph,
                      "chain": "MLP -> pre-pass -> render -> chi^2 -> adjoints -> ADAM (torch elementwise update)"}))


if __name__ == "__main__":
    main()
