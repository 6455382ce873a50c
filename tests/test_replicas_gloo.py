"""N > 1 host logic ("replicas only") on CPU: world_size-2 gloo process group.
The path has no data-path collective; what is covered is the measurement protocol (max over ranks,
whole-job aggregate) and the rank handling of the reference arm."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2309_11273_b200 import replicas
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 2.0 + 3.0 * rank                      # rank 1 is the slow one
    ms = replicas.max_over_ranks(ms_local)
    val = replicas.whole_job_throughput(1000, 10, ms, world)
    dist.barrier()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"rank": replicas.rank_info()[0], "world": replicas.rank_info()[2], "ms": ms, "value": val}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate(tmp_path):
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(2, 29731, out), nprocs=2, join=True)
    res = [json.load(open(f"{out}.{r}")) for r in range(2)]
    for r, d in enumerate(res):
        assert d["rank"] == r and d["world"] == 2
        assert d["ms"] == 5.0                                   # max over ranks, on both ranks
        assert d["value"] == 2 * 1000 * 10 / 5.0e-3             # whole job: both replicas' units / slowest rank's time
    # single process: identity
    sys.path.insert(0, ROOT)
    from paper_2309_11273_b200 import replicas
    assert replicas.max_over_ranks(1.25) == 1.25
    assert replicas.whole_job_throughput(100, 2, 4.0, 1) == 100 * 2 / 4.0e-3


def test_reference_arm_nonzero_rank_is_silent():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""
