"""The N > 1 harness of bench.py on CPU (gloo, world_size 2, 127.0.0.1): MRCQR does not shard (DESIGN.md section 8:
replicas only), so the only multi-process logic is the timing rule -- barrier, then the MAX over ranks of the
per-rank device time -- and the rule that the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
assert bench.max_over_ranks(3.5) == 3.5                 # before init: single process, no collective
dist.init_process_group("gloo")
dist.barrier()
mine = 1.25 if rank == 0 else 7.5                        # rank 1 is the slow replica
got = bench.max_over_ranks(mine)
again = bench.max_over_ranks(10.0 - mine)                # now rank 0 is the slow one
dist.barrier()
dist.destroy_process_group()
print(json.dumps({"rank": rank, "got": got, "again": again}))
""" % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(code, world, extra_env=None):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_max_over_ranks_gloo_world2():
    outs = _spawn(WORKER, 2)
    res = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    assert [d["rank"] for d in res] == [0, 1]
    for d in res:                                          # every rank sees the slowest replica's time
        assert d["got"] == 7.5 and d["again"] == 8.75


def test_reference_arm_runs_on_rank0_only():
    # under torchrun (N > 1) rank 0 alone times the oracle; the other ranks exit 0 without work or output
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, cwd=ROOT, capture_output=True, text=True, timeout=240)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_product_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        return
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"],
                       cwd=ROOT, capture_output=True, text=True, timeout=240)
    assert p.returncode != 0 and "no CPU fallback" in (p.stderr + p.stdout)
