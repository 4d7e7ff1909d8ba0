"""N>1 logic of bench.py on CPU: two gloo ranks, each with its own scene seed, agree on max-over-ranks step times."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_29794_b200 import replicas, scenes


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w, r, _ = replicas.world()
    scene = scenes.make_scene(1, seed=replicas.rank_seed(r))
    ms = [10.0 + 5.0 * rank, 20.0 - 3.0 * rank]              # rank 0: (10, 20), rank 1: (15, 17)
    mx = replicas.max_over_ranks(ms)
    dist.barrier()
    q.put((rank, w, mx, float(scene["means"].sum())))
    dist.destroy_process_group()


def test_two_ranks_max_times_and_distinct_scenes():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps: p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60); assert p.exitcode == 0
    assert [o[1] for o in out] == [2, 2]
    assert out[0][2] == out[1][2] == [15.0, 20.0]            # max over ranks, identical on both
    assert out[0][3] != out[1][3]                            # different seeds -> different scenes
    assert replicas.aggregate_throughput(100.0, 20.0, 2) == 2 * 100.0 / 0.020


def test_single_process_is_identity():
    assert replicas.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert replicas.world()[0] >= 1


def test_bench_spawns_its_own_ranks_when_not_under_torchrun():
    """`python bench.py --gpus 2` outside torchrun must start two ranks itself (the driver's torchrun command line) and print ONE line
    with n_gpus = 2.  --impl selftest runs the rank plumbing on CPU with gloo (no kernel, no measurement)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "selftest"], capture_output=True, text=True,
                         timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(ln) for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["max_over_ranks"] == [11.0, 5.0]
    # one process: no spawn, n_gpus = 1
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "selftest"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0 and json.loads(out.stdout.strip().splitlines()[-1])["n_gpus"] == 1
