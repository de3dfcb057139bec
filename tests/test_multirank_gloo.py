"""N > 1 path of bench.py on the CPU: two gloo ranks.  The path shards by time frame with no
data-path collective: every rank takes its own seeded frame, the job
time is the max over ranks and the work the sum.  Checked here: the reduction, that the ranks'
frames differ and are reproducible, and that the reference arm prints on rank 0 only."""
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import SEED_BASE, make_frame
    fr = make_frame(1, seed=bench.rank_seed(SEED_BASE, 1, rank))
    ms_local = 10.0 + 5.0 * rank           # rank 1 is the slow one
    ms, units = bench.aggregate_over_ranks(ms_local, fr.n_digits, torch.device("cpu"), world)
    with open(os.path.join(out_dir, "r%d.json" % rank), "w") as f:
        json.dump({"ms": ms, "units": units, "n": fr.n_digits, "checksum": fr.meta["checksum"]}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / ("r%d.json" % i))) for i in range(2)]
    assert r[0]["ms"] == r[1]["ms"] == 15.0                      # max over ranks
    assert r[0]["units"] == r[1]["units"] == r[0]["n"] + r[1]["n"]  # sum over ranks
    assert r[0]["checksum"] != r[1]["checksum"]                  # each rank has its own frame
    sys.path.insert(0, ROOT)
    import bench
    from workloads import SEED_BASE, make_frame
    assert make_frame(1, seed=bench.rank_seed(SEED_BASE, 1, 1)).meta["checksum"] == r[1]["checksum"]


def test_reference_arm_rank0_only():
    """--impl reference under torchrun: rank 0 alone runs and prints, the other ranks exit 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", CUDA_VISIBLE_DEVICES="")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "digits/s"
