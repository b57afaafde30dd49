"""The N > 1 path of bench.py on CPU: world_size-2 gloo processes exercise the rendezvous, the round-robin
segment assignment, the barrier and the max-over-ranks reduction (paper_2110_13115_b200/dist.py)."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(textwrap.dedent("""
        import sys
        sys.path.insert(0, %r)
        from paper_2110_13115_b200 import dist as rdist
        rank, local_rank, world = rdist.init(backend="gloo")
        assert world == 2 and rank in (0, 1)
        segs = [rdist.segment_index(rank, s, world) for s in range(3)]
        assert segs == [rank, 2 + rank, 4 + rank]
        rdist.barrier()
        assert rdist.max_over_ranks(10.0 + rank) == 11.0
        assert rdist.sum_over_ranks(1.0 + rank) == 3.0
        rdist.finalize()
        print("rank", rank, "ok")
    """ % ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0, out
        assert "rank %d ok" % r in out


def test_single_process_defaults():
    from paper_2110_13115_b200 import dist as rdist
    env = {k: os.environ.pop(k, None) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    try:
        assert rdist.env_world() == (0, 0, 1)
        assert rdist.max_over_ranks(3.5) == 3.5
        # every (rank, step) pair gets a distinct segment
        world = 4
        seen = {rdist.segment_index(r, s, world) for r in range(world) for s in range(5)}
        assert seen == set(range(20))
    finally:
        for k, v in env.items():
            if v is not None:
                os.environ[k] = v
