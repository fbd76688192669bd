"""world_size-2 gloo test of the N>1 bench plumbing (runs on CPU)."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_hermite_blocks_partition():
    from paper_2209_06731_b200 import dist as D
    world, Nm = 4, 8
    blocks = [D.hermite_block(Nm, r, world) for r in range(world)]
    assert blocks[0][0] == 0 and blocks[-1][1] == Nm * world
    for a, b in zip(blocks, blocks[1:]):
        assert a[1] == b[0]
    assert all(b[2] == Nm * world for b in blocks)


def test_two_rank_gloo_aggregate():
    script = textwrap.dedent("""
        import sys
        sys.path.insert(0, %r)
        from paper_2209_06731_b200 import dist as D
        rank, local, world = D.init("gloo")
        assert world == 2
        m0, m1, Nm = D.hermite_block(8, rank, world)
        assert (m0, m1, Nm) == (8 * rank, 8 * rank + 8, 16)
        D.barrier()
        # rank 0 takes 1.0 s for 10 units, rank 1 takes 2.0 s for 10 units -> 20 units / 2.0 s
        value, sec = D.aggregate_throughput(10.0, 1.0 + rank)
        assert abs(sec - 2.0) < 1e-12 and abs(value - 10.0) < 1e-12, (value, sec)
        D.barrier()
        D.finalize()
        print("ok", rank)
    """ % ROOT)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", script], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert "ok 0" in outs[0] and "ok 1" in outs[1]
