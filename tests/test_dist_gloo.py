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


def test_rank_blocks_are_slices_of_one_seeded_state():
    """bench.py --gpus N: rank r owns the Hermite block [m0, m1) of ONE global seeded state (weak scaling: Nm per
    rank fixed); the blocks of all ranks tile the single-process state bit for bit."""
    import numpy as np
    from paper_2209_06731_b200 import dist as D, inputs as I
    world = 2
    cfg = I.Config("t", 16, 16, 2, 2, 3, [I.Species()], seed=11)
    blocks = [D.hermite_block(cfg.Nm, r, world) for r in range(world)]
    cfg_global = I.Config(**{**cfg.__dict__, "Nm": blocks[0][2]})
    whole = I.make_state(cfg_global)
    for (m0, m1, _) in blocks:
        part = I.make_state(cfg_global, hermite_block=(m0, m1))
        assert part.shape[1] == cfg.Nm and np.array_equal(part, whole[:, m0:m1])
    # the m = 0 slab every rank uses for the replicated field solve is the global one
    assert np.array_equal(I.make_state(cfg_global, hermite_block=(0, 1)), whole[:, 0:1])


def test_bench_refuses_more_gpus_than_visible():
    import subprocess
    env = dict(os.environ)
    env.pop("WORLD_SIZE", None)
    env["CUDA_VISIBLE_DEVICES"] = ""
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode != 0 and "--gpus 2" in (res.stderr + res.stdout)


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
