"""The N>1 harness logic on CPU: world_size 2, gloo backend."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    from paper_1304_0597_b200 import replicas, workloads as wl
    world, rank, local = replicas.env_world()
    dist.init_process_group("gloo")
    assert world == 2 and dist.get_world_size() == 2
    w = replicas.replica_workload(wl.config(1), rank)
    assert w.seed == 1 + 1000 * rank and w.N == 2100 and w.P == 20
    ms_local = 10.0 if rank == 0 else 25.0              # rank 1 is the slow one
    assert replicas.max_over_ranks(ms_local, world) == 25.0
    val, ms = replicas.job_throughput(1000.0, world, ms_local)
    assert ms == 25.0 and abs(val - 2 * 1000.0 / 0.025) < 1e-6
    dist.barrier()
    dist.destroy_process_group()
    print("rank", rank, "ok")
""") % ROOT


def test_two_rank_aggregation(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok" % r in o


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    from paper_1304_0597_b200 import replicas
    assert replicas.max_over_ranks(3.5, 1) == 3.5
    v, ms = replicas.job_throughput(100.0, 1, 50.0)
    assert ms == 50.0 and v == 2000.0
