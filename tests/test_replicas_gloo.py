"""N > 1 path of bench.py on CPU: the hot path has no exchange step ("replicas only"), so the only
multi-rank logic is the rendezvous, the barrier and the max-over-ranks of the per-rank time.  world_size 2, gloo."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import bench
    rank, local_rank, world = bench.dist_init("gloo")
    assert world == 2 and rank in (0, 1)
    bench.barrier()
    # every rank reports its own time; the job time is the slowest rank's
    t = bench.max_over_ranks(10.0 + 5.0 * rank)
    assert t == 15.0, t
    # aggregate throughput of replicas = world * per-rank units / max time
    units = 256
    value = world * units / t
    assert abs(value - 2 * 256 / 15.0) < 1e-12
    bench.barrier()
    print("rank", rank, "ok")
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replicas_rendezvous_barrier_and_max_over_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=120)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"rank {rank} ok" in out


def test_reference_arm_runs_on_rank0_only():
    """--impl reference under torchrun: rank 0 alone runs the oracle, the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
