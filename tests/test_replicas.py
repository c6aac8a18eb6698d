"""Multi-GPU = independent replicas: the only distributed
logic is the barrier and the max / sum of the timing report.  world_size-2
gloo run on CPU."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    from paper_2501_04456_b200 import replicas, workloads
    rank, local_rank, world = replicas.env_rank_world()
    assert world == 2 and rank == local_rank
    replicas.init("gloo")
    replicas.barrier()
    # each rank reports its own time and units; whole-job = sum(units) / max(time)
    ms, units = replicas.reduce_timing(10.0 * (rank + 1), 1000.0 * (rank + 1))
    assert ms == 20.0 and units == 3000.0, (ms, units)
    # distinct replicas: different seed -> different initial state and noise key
    base = workloads.make_workload("C1", state=False)
    s = replicas.replica_seed(base.seed, rank)
    w = workloads.make_workload("C1", 256, seed=s)
    import torch, torch.distributed as dist
    t = torch.tensor([float(w.pos[0, 0]), float(s)], dtype=torch.float64)
    got = [torch.zeros_like(t) for _ in range(world)]
    dist.all_gather(got, t)
    assert got[0][1] != got[1][1] and got[0][0] != got[1][0]
    replicas.barrier()
    print("rank", rank, "ok")
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_timing_reduction(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = []
    for p in procs:
        out, _ = p.communicate(timeout=240)
        outs.append(out)
    for r, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"rank {r} ok" in out


def test_single_process_passthrough():
    from paper_2501_04456_b200 import replicas
    assert replicas.reduce_timing(3.5, 7.0) == (3.5, 7.0)
    assert replicas.replica_seed(3, 0) == 3 and replicas.replica_seed(3, 2) != replicas.replica_seed(3, 1)
    replicas.barrier()   # no process group: a no-op
