#!/usr/bin/env python
"""bench.py -- forward+adjoint ASM throughput on B200 (BASELINE.json metric), with the kernel
roofline and the fp64 CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1..C5] [--impl reference] [--tuning key=value ...]

A step = one pass of the whole hot path (dop_propagate_fwd + dop_propagate_adj, every
wavelength) over one batch of seeded synthetic input.  BASELINE.json's metric names no
configuration and north_star sets its bar "on the largest grid that fits one GPU", so the default
workload is the largest of C5, C4, C3, C2, C1 whose buffers fit the device's free memory (C5:
98304 x 65536, 120 GiB on a 180 GB B200); --config selects any other.  N > 1 = N independent
replicas, one per GPU ("replicas only"): no data-path collective, weak scaling; without
a torchrun environment --gpus N re-launches itself under torch.distributed.run.

Prints ONE JSON line (rank 0).  `value` = Gpoints/s with inputs resident in HBM; `e2e` = the same
metric with host buffers (pinned) and host<->device copies inside the timed region; `roofline` =
achieved algorithmic HBM GB/s of the dominant kernel from per-launch CUDA events; `cpu_baseline`
= the oracle (oracle/, as it stands) on this box's host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "ASM forward+adjoint Gpoints/s (complex64)"
UNIT = "Gpoints/s"


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): bounded sample of the same workload
# ------------------------------------------------------------------------------------------------
def oracle_sample(cfg_name: str):
    """(cfg, sample ny, nx, description): one wavelength on a crop the oracle finishes in ~10-30 s."""
    from paper_2505_22313_b200 import synth
    cfg = synth.CONFIGS[cfg_name]
    ny, nx = min(cfg.ny, 3072), min(cfg.nx, 4096)
    if cfg.ny == cfg.nx:
        ny = nx = min(cfg.ny, 4096 if cfg.sigma_px == 0 else 3072)
    lam = cfg.lambdas[len(cfg.lambdas) // 2]
    desc = (f"{cfg.name} recipe, top-left {ny}x{nx} crop of the seeded inputs, 1 of {len(cfg.lambdas)} "
            f"wavelength(s) ({lam * 1e9:.0f} nm), fwd+adj in fp64")
    return cfg, ny, nx, lam, desc


def time_oracle(cfg_name: str, steps: int = 1):
    """Times oracle forward()+adjoint() as they stand; returns (Gpoints/s, cores, sample text, s/step)."""
    import numpy as np
    import torch
    from oracle import asm_oracle as O
    from paper_2505_22313_b200 import synth
    cfg, ny, nx, lam, desc = oracle_sample(cfg_name)
    small = cfg.scaled(ny, nx)
    h = synth.make_height(small, "cpu").numpy()
    T = synth.make_target(small, "cpu").numpy()
    n_refr = cfg.n_refr[len(cfg.lambdas) // 2]
    times = []
    for _ in range(max(1, steps)):
        t0 = time.perf_counter()
        O.forward(h, cfg.pitch, [lam], [n_refr], cfg.z, target=T, sigma_px=cfg.sigma_px, keep_field=False)
        O.adjoint(h, cfg.pitch, [lam], [n_refr], cfg.z, target=T, sigma_px=cfg.sigma_px)
        times.append(time.perf_counter() - t0)
    dt = statistics.median(times)
    return ny * nx / dt / 1e9, O.num_threads(), desc, dt


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(cfg_name: str, pass_name: str):
    """(DRAM bytes per launch, note) of the dominant pass: dram__bytes_read.sum + dram__bytes_write.sum
    from the committed `ncu --set full` capture of one step (profiles/r02_ncu_<config>.csv, written by
    paper_2505_22313_b200/ncu_summary.py).  The capture records the hash of the kernel sources it was
    taken with; a capture of other sources is refused (traffic = null) rather than quoted."""
    import csv
    from paper_2505_22313_b200 import build as dop_build
    path = os.path.join(ROOT, "profiles", f"r02_ncu_{cfg_name}.csv")
    try:
        with open(path) as f:
            stamp = f.readline().strip()
            if not stamp.startswith("# source_stamp="):
                return None, f"{os.path.basename(path)}: no source stamp"
            if stamp.split("=", 1)[1] != dop_build.source_stamp():
                return None, f"{os.path.basename(path)} was captured with other kernel sources (stale): refused"
            rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#"))]
        vals = [float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]) for r in rows
                if r["pass"].split(":", 1)[-1] == pass_name]
        if vals:
            return sum(vals) / len(vals), f"{os.path.basename(path)}, {len(vals)} launch(es) of one step"
        return None, f"{os.path.basename(path)}: pass not in the capture"
    except FileNotFoundError:
        return None, "no committed ncu capture for this config"
    except Exception as e:  # a malformed file must not take the bench down
        return None, f"{os.path.basename(path)}: {type(e).__name__}"


def device_bytes_needed(cfg) -> int:
    """Device memory of one replica: fields + (pre-filter plane) + h, T, grad (+ I) + slack."""
    n = cfg.ny * cfg.nx
    planes = 3 + (len(cfg.lambdas) if cfg.write_intensity else 0) + (1 if cfg.sigma_px > 0 else 0)
    return n * 8 * len(cfg.lambdas) + n * 4 * planes + (2 << 30)


def pick_default_config(free_bytes: int) -> str:
    from paper_2505_22313_b200 import synth
    for name in ("C5", "C4", "C3", "C2", "C1"):
        if device_bytes_needed(synth.CONFIGS[name]) <= free_bytes:
            return name
    return "C1"


def max_over_ranks(ms: float, dist, device) -> float:
    """Multi-rank timing rule: every rank times its own replica on its device; the step time is the
    MAX over ranks (all_reduce on `device`: a cuda device under nccl, 'cpu' under gloo in tests)."""
    if dist is None:
        return ms
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(points_per_replica: int, world: int, ms_per_step: float) -> float:
    """Whole-job Gpoints/s of `world` independent replicas (weak scaling, no data-path collective)."""
    return world * points_per_replica / (ms_per_step * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2505_22313_b200 import synth
    cfg = synth.CONFIGS[args.config]
    for _ in range(min(args.warmup, 1)):
        time_oracle(args.config, 1)
    gps, cores, desc, dt = time_oracle(args.config, max(1, min(args.steps, 3)))
    line = {
        "impl": "reference", "metric": METRIC, "value": gps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": max(1, min(args.steps, 3)), "warmup": min(args.warmup, 1), "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": desc},
        "cpu_baseline": {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": gps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_name(cfg) -> str:
    lam = "/".join(f"{l * 1e9:.0f}" for l in cfg.lambdas)
    s = (f"{cfg.name}: ASM forward+adjoint {cfg.ny}x{cfg.nx}, pitch {cfg.pitch * 1e6:g} um, lambda {lam} nm, "
         f"z {cfg.z * 1e3:g} mm, L2 loss")
    if cfg.sigma_px > 0:
        s += f", Gaussian pre-filter sigma {cfg.sigma_px:g} px"
    if cfg.write_intensity:
        s += ", intensity output"
    return s


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default=None, choices=["C1", "C2", "C3", "C4", "C5"],
                    help="default: the largest configuration that fits the device (C5 on a 180 GB B200)")
    ap.add_argument("--impl", default="dop", choices=["dop", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="do not replay launch-bound configs as a CUDA graph")
    ap.add_argument("--tuning", nargs="*", default=[], metavar="KEY=VALUE",
                    help="dop_tuning fields for A/B measurements (include/dop.h), e.g. no_tma=1 cluster_force=1 ydigits=256,384")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    # --gpus N must be what runs: under torchrun WORLD_SIZE has to agree; a bare `bench.py --gpus N`
    # (N > 1) re-launches itself as N ranks, one per GPU
    env_world = os.environ.get("WORLD_SIZE")
    if env_world is None and args.gpus > 1:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                  "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if env_world is not None and int(env_world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={env_world}; launch one rank per GPU")
    if args.impl == "reference":
        if args.config is None:  # a bounded sample of the workload the dop arm picks on this box
            args.config = "C5"
            try:
                import torch
                if torch.cuda.is_available():
                    args.config = pick_default_config(torch.cuda.mem_get_info(0)[0])
            except Exception:
                pass
        run_reference(args)
        return

    import torch
    from paper_2505_22313_b200 import dop, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if args.config is None:
        args.config = pick_default_config(torch.cuda.mem_get_info(dev)[0])
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = synth.CONFIGS[args.config]
    warmup = max(args.warmup, 3)
    steps = max(args.steps, 1)
    flags = dop.DOP_WRITE_INTENSITY if cfg.write_intensity else 0
    tun = {}
    for kv in args.tuning:
        k, v = kv.split("=")
        tun[k] = tuple(int(x) for x in v.split(",")) if k in ("xdigits", "ydigits") else int(v)
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, cfg.sigma_px,
                    flags, device=str(dev), tuning=dop.make_tuning(**tun) if tun else None)
    h = synth.make_height(cfg, dev)
    T = synth.make_target(cfg, dev)
    grad = torch.empty_like(h)
    inten = torch.empty((len(cfg.lambdas), cfg.ny, cfg.nx), dtype=torch.float32, device=dev) if flags else None
    loss = torch.zeros(1, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    points = cfg.points

    def raw_step():
        plan.fwd(h, T, inten, loss)
        plan.adj(h, None, grad)

    step = raw_step

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    # Launch-bound case (the field fits L2: C1, ten ~10 us kernels): replay the step as one CUDA
    # graph, which is how a caller would run a launch-bound loop; the library calls only enqueue
    # kernels on the current stream, so they capture as they are.
    use_graph = points * 8 <= (64 << 20) and not args.no_graph
    if use_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            raw_step()
        step = graph.replay
        for _ in range(3):
            step()
        barrier()

    # ---- timed region: K steps, inputs resident in HBM, CUDA events on the launching stream
    # nvidia-smi samples every 100 ms, so the same steps also run (untimed, back to back, no sync in
    # between) for >= 250 ms before and after the K timed ones: the clock record then describes this
    # load even when the timed region itself is shorter than the sampling period.
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    step()
    e1.record(stream)
    barrier()
    n_lead = max(1, min(4000, int(250.0 / max(e0.elapsed_time(e1), 1e-3)) + 1))
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        t_wait = time.time()
        while not sampler.rows and time.time() - t_wait < 5.0:   # nvidia-smi can take a second to start
            time.sleep(0.05)
    barrier()
    for _ in range(n_lead):
        step()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    for _ in range(n_lead):
        step()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None:
        clocks["sampling"] = f"100 ms period over {n_lead} + {steps} timed + {n_lead} back-to-back steps"
    ms = max_over_ranks(ms, dist, dev)
    ms_per_step = ms / steps
    value = aggregate_value(points, world, ms_per_step)
    loss_value = float(loss.item())

    # ---- per-launch CUDA events (same stream, same steps): the roofline of the dominant kernel
    dop.dop_plan_set_profiling(plan.handle, True)
    acc = {}
    order = []
    prof_steps = min(steps, 10)
    for _ in range(prof_steps):
        raw_step()
        torch.cuda.synchronize()
        for name, t_ms, bpp in dop.dop_plan_get_pass_times(plan.handle):
            key = name.split(":", 1)[1] if ":" in name else name  # merge fwd/adj launches of the same kernel+digit
            if key not in acc:
                acc[key] = [0.0, 0, bpp, 0.0]
                order.append(key)
            acc[key][0] += t_ms
            acc[key][1] += 1
            acc[key][3] += bpp
    dop.dop_plan_set_profiling(plan.handle, False)
    peak, peak_src = measured_peak_gbs()
    npts_plane = cfg.ny * cfg.nx
    passes = []
    for key in order:
        tot, cnt, _, bsum = acc[key]
        avg_ms = tot / cnt
        gbs = (bsum / cnt) * npts_plane / (avg_ms * 1e-3) / 1e9 if avg_ms > 0 else 0.0
        passes.append({"pass": key, "launches_per_step": cnt / prof_steps, "avg_ms": round(avg_ms, 4),
                       "bytes_per_point": bsum / cnt, "GBps": round(gbs, 1), "frac": round(gbs / peak, 4),
                       "share": 0.0})
    total_prof = sum(acc[k][0] for k in order)
    for p_, key in zip(passes, order):
        p_["share"] = round(acc[key][0] / total_prof, 4)
    dom = max(passes, key=lambda p_: p_["share"])
    step_bytes = sum(acc[k][3] for k in order) / prof_steps * npts_plane
    traffic, traffic_note = ncu_traffic(args.config, dom["pass"])
    roofline = {
        "bound": "hbm", "kernel": dom["pass"], "achieved": dom["GBps"], "peak": peak, "unit": "GB/s",
        "frac": round(dom["GBps"] / peak, 4), "traffic": traffic, "traffic_source": traffic_note,
        "peak_source": peak_src, "bytes_per_launch": dom["bytes_per_point"] * npts_plane,
        "avg_launch_ms": dom["avg_ms"], "share_of_step": dom["share"],
        "whole_step": {"algorithmic_bytes_per_point": step_bytes / points,
                       "GBps": round(step_bytes / (ms_per_step * 1e-3) / 1e9, 1),
                       "frac": round(step_bytes / (ms_per_step * 1e-3) / 1e9 / peak, 4),
                       "fused_minimum_bytes_per_point": 80 + (4 if cfg.write_intensity else 0) + (36 if cfg.sigma_px > 0 else 0),
                       },
        "passes": passes,
    }

    # ---- e2e: host (pinned) buffers, H2D of h and T and D2H of grad + loss inside the timed region
    e2e = None
    if not args.no_e2e:
        h_host = h.cpu().pin_memory()
        T_host = T.cpu().pin_memory()
        g_host = torch.empty_like(h_host).pin_memory()
        l_host = torch.zeros(1, dtype=torch.float64).pin_memory()
        i_host = torch.empty(inten.shape, dtype=torch.float32).pin_memory() if inten is not None else None
        e2e_steps = max(1, min(steps, 5))
        # Second set of device buffers -> the copies of step k+1 / k-1 overlap the kernels of step k
        # (three streams, events; every step still moves its own inputs in and its own results out).
        extra = (3 * h.numel() + (inten.numel() if inten is not None else 0)) * 4
        # (not worth its event traffic on the latency-bound C1: 0.46 against 0.33 ms per step)
        pipelined = extra >= (64 << 20) and torch.cuda.mem_get_info(dev)[0] > extra + (2 << 30)
        if pipelined:
            bufs = [(h, T, inten, loss, grad),
                    (torch.empty_like(h), torch.empty_like(T), torch.empty_like(inten) if inten is not None else None,
                     torch.zeros_like(loss), torch.empty_like(grad))]
            s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
            ev_in = [torch.cuda.Event() for _ in range(2)]
            ev_comp = [torch.cuda.Event() for _ in range(2)]
            ev_out = [torch.cuda.Event() for _ in range(2)]
            for e in ev_comp + ev_out:
                e.record(stream)

            def e2e_step(k):
                hh, TT, ii, ll, gg = bufs[k % 2]
                with torch.cuda.stream(s_in):
                    s_in.wait_event(ev_comp[k % 2])      # the kernels that last read these inputs are done
                    hh.copy_(h_host, non_blocking=True)
                    TT.copy_(T_host, non_blocking=True)
                    ev_in[k % 2].record(s_in)
                stream.wait_event(ev_in[k % 2])
                stream.wait_event(ev_out[k % 2])         # the previous results of this slot have left
                plan.fwd(hh, TT, ii, ll)
                plan.adj(hh, None, gg)
                ev_comp[k % 2].record(stream)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_comp[k % 2])
                    g_host.copy_(gg, non_blocking=True)
                    l_host.copy_(ll, non_blocking=True)
                    if i_host is not None:
                        i_host.copy_(ii, non_blocking=True)
                    ev_out[k % 2].record(s_out)

            def e2e_join():
                for e in ev_out:
                    stream.wait_event(e)
        else:
            def e2e_step(k):
                h.copy_(h_host, non_blocking=True)
                T.copy_(T_host, non_blocking=True)
                step()
                g_host.copy_(grad, non_blocking=True)
                l_host.copy_(loss, non_blocking=True)
                if i_host is not None:
                    i_host.copy_(inten, non_blocking=True)

            def e2e_join():
                pass

        e2e_step(0)
        e2e_step(1)
        e2e_join()
        barrier()
        e0.record(stream)
        for k in range(e2e_steps):
            e2e_step(k)
        e2e_join()
        e1.record(stream)
        barrier()
        ms2 = e0.elapsed_time(e1)
        ms2 = max_over_ranks(ms2, dist, dev)
        h2d = h_host.numel() * 4 + T_host.numel() * 4
        d2h = g_host.numel() * 4 + 8 + (i_host.numel() * 4 if i_host is not None else 0)
        e2e = {"value": aggregate_value(points, world, ms2 / e2e_steps), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "ms_per_step": ms2 / e2e_steps,
               "overlap": "copies of neighbouring steps overlap the kernels (2 buffer sets, 3 streams)" if pipelined
               else "serial (small problem, or no memory for a second buffer set)"}
        del h_host, T_host, g_host, i_host

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        gps, cores, desc, dt = time_oracle(args.config, 1)
        cpu = {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
               "seconds": round(dt, 2)}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "c64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "points_per_step": points, "parallelism": f"replicas x{world}", "cuda_graph": bool(use_graph),
                       "tuning": {k: (list(v) if isinstance(v, tuple) else v) for k, v in tun.items()},
                       "l2": "working set (>= 1.5 GiB) larger than the 126 MB L2; no flush between steps"
                       if points * 8 > 4 * 126e6 else "working set fits L2 (latency-bound config)",
                       "loss": loss_value},
            "clocks": clocks, "e2e": e2e, "gpu_launches": plan.launches * steps, "roofline": roofline,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    plan.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
