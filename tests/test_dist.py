"""world_size-2 gloo test of the N>1 bench plumbing (replicas only: barrier + max/sum over ranks)."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_single_process_is_identity():
    from paper_2411_18511_b200.dist import Ranks, whole_job_throughput
    env = {k: os.environ.pop(k) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK") if k in os.environ}
    try:
        r = Ranks()
        assert r.world == 1 and r.max(3.5) == 3.5 and r.sum(2.0) == 2.0
        assert whole_job_throughput(r, 10.0, 2.0) == (5.0, 2.0)
    finally:
        os.environ.update(env)


def test_two_ranks_gloo():
    code = textwrap.dedent("""
        import os, sys
        sys.path.insert(0, %r)
        from paper_2411_18511_b200.dist import Ranks, whole_job_throughput
        r = Ranks(backend="gloo", device="cpu")
        r.barrier()
        # rank 0 processed 10 units in 1 s, rank 1 processed 10 units in 2 s: whole job = 20 units / 2 s
        v, t = whole_job_throughput(r, 10.0, 1.0 + r.rank)
        assert (v, t) == (10.0, 2.0), (v, t)
        r.barrier()
        r.close()
        print("rank", r.rank, "ok")
    """ % ROOT)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT))
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out.decode()
        assert b"ok" in out
