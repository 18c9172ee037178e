"""N > 1 host logic of bench.py on CPU: world_size-2 gloo ("replicas only").

The path does not shard: every rank runs an independent replica, the step time is the max over
ranks and the value is the whole-job aggregate.  No GPU and no CUDA call here."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    my_ms = 10.0 + 5.0 * rank  # rank 1 is the slow replica
    ms = bench.max_over_ranks(my_ms, dist, "cpu")
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "value": bench.aggregate_value(1_000_000, world, ms)}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_weak_scaling_aggregate(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(2)]
    assert res[0] == res[1]
    assert res[0]["ms"] == 15.0  # the max, not the mean, not rank 0's
    assert abs(res[0]["value"] - 2 * 1_000_000 / 15e-3 / 1e9) < 1e-12


def test_single_rank_passthrough():
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.aggregate_value(2_000_000_000, 1, 1000.0) == 2.0


def test_reference_arm_runs_on_rank0_only():
    """--impl reference under torchrun: ranks != 0 exit 0 without work and print nothing."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpus_flag_must_agree_with_the_launch():
    """bench.py --gpus N under a launcher whose WORLD_SIZE differs fails instead of silently running N = 1."""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], env=env, capture_output=True,
                       text=True, timeout=120)
    assert r.returncode != 0 and "WORLD_SIZE=1" in (r.stderr + r.stdout)


def test_default_workload_is_the_largest_that_fits():
    import bench
    assert bench.pick_default_config(int(178e9)) == "C5"      # 120 GiB + slack on a 180 GB B200
    assert bench.pick_default_config(int(120e9)) == "C4"      # 96 GiB with the intensity plane
    assert bench.pick_default_config(int(40e9)) == "C3"
    assert bench.pick_default_config(int(3e9)) == "C1"


def test_stale_ncu_capture_is_refused(tmp_path, monkeypatch):
    """roofline.traffic comes from a committed capture only if it was taken with the current kernel sources."""
    import bench
    from paper_2505_22313_b200 import build as dop_build
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    body = "pass,kernel,time_us,dram_bytes_read,dram_bytes_write\nfwd:y0:y-fwd,k,1,100,50\nadj:y0:y-fwd,k,1,102,52\n"
    (prof / "r02_ncu_C9.csv").write_text("# source_stamp=deadbeef\n# note\n" + body)
    val, note = bench.ncu_traffic("C9", "y0:y-fwd")
    assert val is None and "stale" in note
    (prof / "r02_ncu_C9.csv").write_text(f"# source_stamp={dop_build.source_stamp()}\n# note\n" + body)
    val, note = bench.ncu_traffic("C9", "y0:y-fwd")
    assert val == 152.0 and "2 launch" in note
    assert bench.ncu_traffic("C8", "y0:y-fwd")[0] is None
