"""Multi-rank host logic on CPU (gloo, world_size 2): the pixel partition, the gather of the outputs and
the max-over-ranks of the step time.  The per-pixel solve is stood in for by the oracle (test
infrastructure), because eq. 2 makes every pixel independent: sharded == unsharded."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1402_2518_b200.shard import cube_block, launch_plan, pixel_block


def test_pixel_block_partitions():
    for N in (0, 1, 5, 64, 1000, 131072 + 3):
        for world in (1, 2, 3, 8):
            blocks = [pixel_block(N, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == N
            for (a, b), (c, d) in zip(blocks, blocks[1:]):
                assert b == c and a <= b and c <= d
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        pixel_block(10, 2, 2)
    assert cube_block(3, 128) == (384, 512)


def test_bench_launch_plan():
    """`python bench.py --gpus N` must end up with N ranks: inline under torchrun or for one GPU, a torchrun command
    line otherwise, and a loud error when the node has fewer devices (never a silent one-rank run labelled N)."""
    argv = ["bench.py", "--gpus", "4", "--steps", "2"]
    assert launch_plan(1, {}, 0, argv, "python", 29500) == ("inline", None)
    assert launch_plan(4, {"WORLD_SIZE": "4", "RANK": "1"}, 8, argv, "python", 29500) == ("inline", None)
    kind, cmd = launch_plan(4, {}, 8, argv, "py", 29511)
    assert kind == "spawn" and cmd[:3] == ["py", "-m", "torch.distributed.run"] and cmd[-5:] == argv
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    with pytest.raises(ValueError, match="only 1 CUDA device"):
        launch_plan(8, {}, 1, argv, "python", 29500)
    with pytest.raises(ValueError, match="WORLD_SIZE=2"):
        launch_plan(4, {"WORLD_SIZE": "2"}, 8, argv, "python", 29500)
    with pytest.raises(ValueError):
        launch_plan(0, {}, 8, argv, "python", 29500)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_1402_2518_b200.shard import gather_blocks, max_over_ranks
        from paper_1402_2518_b200.synth import make_workload
        w = make_workload("tiny", N=N)                      # same seeded inputs on every rank
        lo, hi = pixel_block(N, rank, world)
        sol = oracle.solve(w.A, w.Y[lo:hi], w.sigma[lo:hi])
        coeffs = gather_blocks(torch.from_numpy(sol.coeffs), N)
        resid = gather_blocks(torch.from_numpy(sol.resid), N)
        tmax = max_over_ranks(1.0 + rank)
        dist.barrier()
        if rank == 0:
            q.put((coeffs.numpy(), resid.numpy(), tmax))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_gloo_sharded_equals_unsharded():
    import oracle
    from paper_1402_2518_b200.synth import make_workload
    oracle.build()
    N, world = 301, 2                                        # odd: the blocks differ in length
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N, q)) for r in range(world)]
    for p in procs:
        p.start()
    coeffs, resid, tmax = q.get()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    w = make_workload("tiny", N=N)
    ref = oracle.solve(w.A, w.Y, w.sigma)
    assert coeffs.shape == (N, w.A.shape[1])
    np.testing.assert_array_equal(coeffs, ref.coeffs)         # same code, same inputs: bit-identical
    np.testing.assert_array_equal(resid, ref.resid)
    assert tmax == 2.0
