"""N>1 host logic of bench.py on CPU: world_size 2, gloo (replicas only, no data-path collective).

Covers the rendezvous from the torchrun environment, the whole-job aggregation (sum of clusters over ranks / max of the
per-rank step time) and the reference arm under two ranks (rank 0 prints the line, rank 1 exits 0 without work).
"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch
import bench
rank, world, local, dist = bench.init_dist(2)
assert world == 2 and dist is not None and dist.get_backend() == "gloo"
# rank r pretends to have tracked (r+1)*1000 clusters in (r+1)*2 ms
value, ms, n_total = bench.aggregate(dist, torch.device("cpu"), (rank + 1) * 1000, (rank + 1) * 2.0)
print(json.dumps({{"rank": rank, "value": value, "ms": ms, "n_total": n_total}}), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(argv_of_rank, timeout=300):
    port = str(_free_port())
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port, CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen(argv_of_rank(r), env=env, cwd=ROOT, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=timeout)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_aggregate_sum_of_clusters_over_max_time_world2_gloo():
    outs = _spawn(lambda r: [sys.executable, "-c", _WORKER.format(root=ROOT)])
    for o in outs:
        d = json.loads(o.strip().splitlines()[-1])
        assert d["n_total"] == 3000
        assert abs(d["ms"] - 4.0) < 1e-12                  # the slowest rank's time
        assert abs(d["value"] - 3000 / 4.0e-3) < 1e-6       # whole-job clusters/s


def test_reference_arm_world2_rank0_prints_rank1_silent():
    outs = _spawn(lambda r: [sys.executable, "bench.py", "--impl", "reference", "--gpus", "2", "--config", "1",
                             "--steps", "1", "--warmup", "0"])
    line = json.loads(outs[0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert outs[1].strip() == ""
