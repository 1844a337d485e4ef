"""world_size-2 checks of the N > 1 path on CPU (gloo): the timing reduction takes the slowest rank,
throughput is the whole-job aggregate, and the reference arm prints from rank 0 only."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_2606_01751_b200 import dist_util as du
    r, w = du.init("gloo")
    du.barrier()
    ms = du.max_over_ranks(10.0 + 5.0 * rank)          # rank 1 is slower
    q.put((r, w, ms, du.job_throughput(1000.0, ms, w)))
    du.barrier()


def test_max_over_ranks_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29641, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [x[0] for x in res] == [0, 1] and all(x[1] == 2 for x in res)
    assert all(x[2] == 15.0 for x in res)                           # max over ranks
    assert all(abs(x[3] - 2 * 1000.0 / 15e-3) < 1e-6 for x in res)  # whole-job aggregate


def test_reference_arm_rank0_only():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29642", WORLD_SIZE="2", LOCAL_RANK="0")
    outs = []
    for rank in (0, 1):
        env["RANK"] = str(rank)
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                            "--steps", "1", "--warmup", "0", "--gpus", "2", "--no-cpu-measured"],
                           env=env, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["estimated"] is True and 0 < line["config"]["sample_fraction_of_step"] <= 1.0
    assert outs[1] == ""
