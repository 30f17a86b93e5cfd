"""-m "not gpu": the N > 1 plumbing of bench.py on CPU (gloo, world_size 2, 127.0.0.1): max-over-ranks timing,
whole-job throughput of independent replicas, and the reference arm printing on rank 0 only."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"],
                        rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank = dist.get_rank()
ms = [10.0 + 5.0 * rank, 3.0 - rank]           # rank 1 is slower on the first, faster on the second
out = bench.max_over_ranks(ms, device="cpu")
dist.barrier()
if rank == 0:
    print(json.dumps({"max": out, "value": bench.job_throughput(2, 1000, 4, out[0])}))
dist.destroy_process_group()
""" % ROOT


def _spawn(code, port, extra_args=()):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code, *extra_args], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    return [o[0] for o in outs]


def test_max_over_ranks_and_replica_throughput_gloo():
    outs = _spawn(WORKER, 29611)
    assert outs[1].strip() == ""                       # only rank 0 prints
    d = json.loads(outs[0].strip().splitlines()[-1])
    assert d["max"] == [15.0, 3.0]
    assert d["value"] == 2 * 1000 * 4 / 15e-3


def test_reference_arm_prints_on_rank0_only():
    code = "import sys; sys.path.insert(0, %r); sys.argv=['bench.py','--impl','reference','--config','c0','--steps','1','--warmup','0','--gpus','2']; import bench; bench.main()" % ROOT
    outs = _spawn(code, 29612)
    assert outs[1].strip() == ""
    d = json.loads(outs[0].strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["n_gpus"] == 2
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
