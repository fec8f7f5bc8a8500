"""The N > 1 path on CPU (gloo, world_size 2): the path shards by independent batches with no data-path collective
(replicas only), so what there is to check is the host logic of bench.py -- every rank draws its own
seeded batch, the timing reduction is a MAX over ranks, and the reference arm prints one line from rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = bench.make_workload("config3", rank, n_models=8, n_epochs=10)
    digest = torch.tensor([float(wl.s.sum()), float(wl.zeta.sum())], dtype=torch.float64)
    got = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(got, digest)
    ms = bench.max_over_ranks([10.0 + rank, 5.0 - rank], torch.device("cpu"), world)
    q.put((rank, [g.tolist() for g in got], ms, wl.n_sources))
    dist.destroy_process_group()


def test_rank_batches_differ_and_timing_is_max_over_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, digests, ms, n in out:
        assert n == 80
        assert digests[0] != digests[1]                 # different seeds -> different batches
        assert ms == [11.0, 5.0]                        # MAX over ranks, element-wise
    assert out[0][1] == out[1][1]                       # both ranks saw the same pair of digests


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--steps", "1", "--warmup", "1", "--cpu-sample", "300"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and np.isfinite(d["ms_per_step"])
