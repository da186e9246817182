"""N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").

Checks the rank plumbing only -- barrier, max-over-ranks time, whole-job rate -- and that `bench.py --impl reference`
lets rank 0 alone print its line while the other ranks exit 0 without work.  No GPU, no data-path collective."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_1012_1900_b200.replicas import Replicas

    r = Replicas(backend="gloo")
    r.barrier()
    seconds = 0.010 * (rank + 1)            # rank 1 is the slow one
    units = 1000.0 + rank                   # each replica counts its own evaluated voxels
    out = (r.rank, r.world, r.max_over_ranks(seconds), r.sum_over_ranks(units), r.job_rate(units, seconds))
    r.barrier()
    r.close()
    q.put(out)


def test_two_replicas_take_the_max_time_and_sum_the_units():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    for _, world, tmax, usum, rate in res:
        assert world == 2
        assert abs(tmax - 0.020) < 1e-12
        assert usum == 2001.0
        assert abs(rate - 2001.0 / 0.020) < 1e-6


def test_single_process_needs_no_group():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1012_1900_b200.replicas import Replicas\n"
            "import torch.distributed as d\n"
            "r = Replicas(); r.barrier()\n"
            "assert r.world == 1 and not d.is_initialized()\n"
            "assert r.max_over_ranks(3.5) == 3.5 and r.job_rate(7.0, 2.0) == 3.5\n" % ROOT)
    subprocess.run([sys.executable, "-c", code], check=True, env=env, timeout=120)


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus",
           "2", "--steps", "2", "--warmup", "1", "--case", "cfg2_small"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(ln) for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    ln = lines[0]
    assert ln["impl"] == "reference" and ln["n_gpus"] == 2 and ln["value"] > 0
    assert ln["cpu_baseline"]["kind"] == "oracle" and ln["e2e"]["h2d_bytes_per_step"] == 0
