"""N > 1 host logic (replicas only) on CPU: world_size 2, gloo backend, 127.0.0.1 rendezvous."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1008_0135_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    views = [replicas.view_of(k, rank, world, 36) for k in range(36)]
    local_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    dist.barrier()
    worst = replicas.max_over_ranks(local_ms, dist)
    gathered = [None] * world
    dist.all_gather_object(gathered, views)
    q.put((rank, worst, gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_render_disjoint_starts_and_time_is_max_over_ranks():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, worst, gathered in out:
        assert worst == 15.0                            # max over ranks, on every rank
        assert sorted(gathered[0]) == list(range(36)) and sorted(gathered[1]) == list(range(36))
        assert gathered[0][0] == 0 and gathered[1][0] == 18   # replicas start half an orbit apart
        assert all(a != b for a, b in zip(gathered[0], gathered[1]))
    assert replicas.aggregate_ms_per_frame(15.0 * 36, 36, 2) == 7.5


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.25, None) == 3.25
    assert [replicas.view_of(k, 0, 1, 36) for k in (0, 35, 36)] == [0, 35, 0]


def _run_bench(argv, extra_env):
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env.update(extra_env)
    return subprocess.run([sys.executable, os.path.join(root, "bench.py")] + argv, cwd=root, env=env, capture_output=True,
                          text=True, timeout=600)


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    r = _run_bench(["--gpus", "8", "--steps", "1"], {"WORLD_SIZE": "2", "RANK": "0"})
    assert r.returncode != 0 and "WORLD_SIZE=2" in r.stderr and "n_gpus" not in r.stdout


def test_bench_gpus_n_without_torchrun_launches_n_ranks_itself():
    """`python bench.py --gpus 2` by hand becomes a 2-rank job (here, without a GPU, both ranks stop with the
    no-device error): it must never answer with a single-replica line."""
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a GPU is present: the ranks would run the full benchmark")
    r = _run_bench(["--gpus", "2", "--steps", "1", "--no-cpu-baseline"], {})
    assert r.returncode != 0
    assert "n_gpus" not in r.stdout
    assert "no CUDA device" in r.stderr                  # a rank's own error (the launcher stops the others at the first)
    assert "torch.distributed" in r.stderr or "elastic" in r.stderr     # ... reported by the multi-rank launcher
