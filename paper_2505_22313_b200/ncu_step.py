"""One forward+adjoint step of a BASELINE.json configuration, bracketed by cudaProfilerStart/Stop, for
`ncu --profile-from-start off ...` (measurement aid; the timed numbers come from bench.py, never from a
run under the profiler).

  python -m paper_2505_22313_b200.ncu_step --config C5 [--ny NY --nx NX] [--labels gpurun_out/labels_C5.json] [key=value ...]

Runs two untimed warm-up steps (the second with per-launch profiling on, to learn the pass label of
every launch), then exactly one step inside the profiler range, and writes the labels in launch order
as JSON, so that ncu_summary.py can name every captured kernel after the pass it ran.  key=value
arguments are dop_tuning fields (xdigits / ydigits as comma lists)."""
from __future__ import annotations

import argparse
import json

import torch

from . import dop, synth


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="C5", choices=sorted(synth.CONFIGS))
    ap.add_argument("--labels", default=None)
    ap.add_argument("--ny", type=int, default=0, help="same recipe and optics on a smaller grid (0 = the configuration's own)")
    ap.add_argument("--nx", type=int, default=0)
    ap.add_argument("tuning", nargs="*")
    args = ap.parse_args()
    tun = {}
    for a in args.tuning:
        k, v = a.split("=")
        tun[k] = tuple(int(x) for x in v.split(",")) if k in ("xdigits", "ydigits") else int(v)
    cfg = synth.CONFIGS[args.config]
    if args.ny or args.nx:
        cfg = cfg.scaled(args.ny or cfg.ny, args.nx or cfg.nx)
    dev = "cuda:0"
    flags = dop.DOP_WRITE_INTENSITY if cfg.write_intensity else 0
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, cfg.sigma_px, flags, dev,
                    tuning=dop.make_tuning(**tun) if tun else None)
    h, T = synth.make_height(cfg, dev), synth.make_target(cfg, dev)
    grad = torch.empty_like(h)
    inten = torch.empty((len(cfg.lambdas), cfg.ny, cfg.nx), dtype=torch.float32, device=dev) if flags else None
    loss = torch.zeros(1, dtype=torch.float64, device=dev)

    def step():
        plan.fwd(h, T, inten, loss)
        plan.adj(h, None, grad)

    step()
    dop.dop_plan_set_profiling(plan.handle, True)
    step()
    torch.cuda.synchronize()
    labels = [name for name, _, _ in dop.dop_plan_get_pass_times(plan.handle)]
    dop.dop_plan_set_profiling(plan.handle, False)
    torch.cuda.cudart().cudaProfilerStart()
    step()
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStop()
    if args.labels:
        with open(args.labels, "w") as f:
            json.dump({"config": args.config, "points_per_plane": cfg.ny * cfg.nx, "labels": labels,
                       "describe": plan.describe()}, f)
    print(f"{args.config}: {len(labels)} launches, loss {loss.item():.9g}")
    plan.close()


if __name__ == "__main__":
    main()
