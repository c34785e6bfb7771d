"""world_size-2 gloo test (CPU) of bench.py's multi-rank host logic: replicas only, max-over-ranks timing, whole-job
aggregate, and the reference arm running on rank 0 alone."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_step, t_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 3.0 - rank], dist, "cpu")
    val = bench.aggregate_value(world, 1000.0, t_step)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"t_step": t_step, "t_e2e": t_e2e, "value": val}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = json.load(open(tmp_path / "r0.json"))
    r1 = json.load(open(tmp_path / "r1.json"))
    assert r0 == r1
    assert r0["t_step"] == 15.0 and r0["t_e2e"] == 3.0           # MAX over ranks
    assert abs(r0["value"] - 2 * 1000.0 / 15e-3) < 1e-6          # sum of per-rank units / slowest rank


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], None, "cpu") == [1.5, 2.5]
    assert bench.aggregate_value(1, 10.0, 1000.0) == 10.0


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=300)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "cMAC/s"


def _nyq_worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import numpy as np
    from paper_2107_09879_b200 import nyquist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    plans = [(np.array([i]), np.array([i, i + 1])) for i in range(5)]
    mine = nyquist.partition_plans(plans, rank, world)
    # a stand-in for the per-window field (the solver needs a GPU): window i contributes (i + 1) at every detector point
    E_local = np.zeros((4, 3), dtype=complex)
    for sidx, _ in mine:
        E_local += (sidx[0] + 1) * (1.0 + 0.5j)
    E = nyquist.sum_fields(E_local, dist)
    np.save(os.path.join(out_dir, f"E{rank}.npy"), E)
    with open(os.path.join(out_dir, f"n{rank}.txt"), "w") as f:
        f.write(str(len(mine)))
    dist.barrier()
    dist.destroy_process_group()


def test_nyquist_windows_split_over_ranks_and_field_sum_gloo(tmp_path):
    """The strategy's only communication: windows are dealt to the ranks, the detector fields are summed once."""
    import numpy as np
    port = 31500 + os.getpid() % 2000
    mp.spawn(_nyq_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    E0, E1 = np.load(tmp_path / "E0.npy"), np.load(tmp_path / "E1.npy")
    assert np.array_equal(E0, E1) and np.allclose(E0, 15 * (1.0 + 0.5j))        # 1 + 2 + 3 + 4 + 5
    assert int(open(tmp_path / "n0.txt").read()) == 3 and int(open(tmp_path / "n1.txt").read()) == 2
