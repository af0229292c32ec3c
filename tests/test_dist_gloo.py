"""world_size-2 gloo test of the N>1 path's host logic (replicas only: units summed, time = max)."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_aggregate_two_ranks(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import os, sys
        sys.path.insert(0, %r)
        from paper_2607_07816_b200 import dist
        rank, lr, world = dist.init("gloo")
        dist.barrier()
        u, t = dist.aggregate(100.0 * (rank + 1), 5.0 + rank)
        assert world == 2 and u == 300.0 and t == 6.0, (u, t)
        dist.barrier()
        dist.shutdown()
        print("ok", rank)
    """ % ROOT))
    port = 29611 + (os.getpid() % 200)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT))
    for p in procs:
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0, out.decode()


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    from paper_2607_07816_b200 import dist
    assert dist.aggregate(7.0, 3.0) == (7.0, 3.0)
