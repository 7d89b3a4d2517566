"""bench.py's N > 1 host logic on CPU (gloo, world_size 2): replicas only - no data-path collective; the job's time is
the max over ranks, its work the sum over ranks; the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r measured (10 + 5r) ms and (7 + r) ms, and processed 1000 (r + 1) and 10 (r + 1) segments
        t, s = bench.reduce_over_ranks([10.0 + 5.0 * rank, 7.0 + rank], [1000.0 * (rank + 1), 10.0 * (rank + 1)], "cpu", world)
        torch.save({"t": t, "s": s, "v": bench.job_throughput(s[0], t[0])}, os.path.join(out, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_max_time_and_summed_work_over_two_ranks(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        d = torch.load(os.path.join(tmp_path, f"r{r}.pt"))
        assert d["t"] == [15.0, 8.0]                      # max over ranks
        assert d["s"] == [3000.0, 30.0]                   # sum over ranks
        assert d["v"] == 3000.0 / 15.0e-3                 # whole-job segments per second


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    t, s = bench.reduce_over_ranks([3.0], [5.0], "cpu", 1)
    assert t == [3.0] and s == [5.0]
    assert bench.job_throughput(5.0, 0.0) == 0.0


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "config1"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["metric"] == "ray_cell_segments_per_s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] == d["e2e"]["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["config"]["workload"] == "config1" and d["value"] > 0


def test_gpus_flag_starts_its_own_ranks_without_torchrun():
    """`python bench.py --gpus 2` with no torchrun environment (how the driver calls it at N = 1) must start two ranks
    itself: one JSON line from rank 0 with n_gpus = 2, and rank 1 was really there"""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "config1"], capture_output=True, text=True, cwd=ROOT, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert "rank 1 of 2" in r.stderr


def test_bench_defaults_to_the_largest_single_gpu_configuration():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.DEFAULT_CONFIG == "config5_N512_S1024"
    names = [n for n, _, _ in bench.PER_CONFIG]
    assert names[:4] == ["config1", "config2", "config3", "config4"] and all(n.startswith("config5_N") for n in names[4:])
    # a committed ncu capture is only used for the workload, flags and csrc build it was taken on
    cap, why = bench.ncu_capture("config5_N512_S1024", 1.0, {"geom_corr": 0})
    assert cap is None and "different number of segments" in why or "no committed" in why or "another build" in why
    cap, why = bench.ncu_capture("config4", 1.0, {"geom_corr": 2})
    assert cap is None


def test_cuda_arm_refuses_to_run_without_a_device():
    if torch.cuda.is_available():
        return
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0", "--config", "config1"],
                       capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
