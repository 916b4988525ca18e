"""-m "not gpu": the N>1 host logic on CPU, world_size 2 and 3, gloo.  Each rank walks its walker
range (with the oracle standing in for the device walk), compacts, and the ranks exchange the
compacted samples; the gathered cloud and its MEGB must equal the single-process result.  The
strong-scaling test drives sharding.strong_step, the very function bench.py --scaling strong calls."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2403_09990_b200 import instances as I
from paper_2403_09990_b200 import sharding


def test_walker_range_partitions_exactly():
    for W in (0, 1, 7, 1024, 65537):
        for world in (1, 2, 3, 8):
            spans = [sharding.walker_range(r, world, W) for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == W
            for (b0, c0), (b1, _) in zip(spans, spans[1:]):
                assert b0 + c0 == b1
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, W, steps, out_dir):
    import oracle
    from paper_2403_09990_b200 import binding as B
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 16)
    begin, cnt = sharding.walker_range(rank, world, W)
    smp, flag = oracle.walk(inst, inst.params, S0, begin + np.arange(cnt), steps, 42)
    if rank == 1:
        flag[::3] = 0                                   # ragged, rank-dependent counts
    comp = oracle.compact(smp, flag)
    gathered = sharding.gather_compacted(torch.from_numpy(comp), comp.shape[0])
    if rank == 0:
        np.save(os.path.join(out_dir, "gathered.npy"), gathered.numpy())
        c3, r3, _ = B.closure_miniball_host(gathered.numpy()[:, 9:])
        np.save(os.path.join(out_dir, "ball.npy"), np.concatenate([c3, [r3]]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gather_equals_single_process(tmp_path):
    import oracle
    W, steps = 96, 12
    mp.spawn(_worker, args=(2, _free_port(), W, steps, str(tmp_path)), nprocs=2, join=True)
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 16)
    smp, flag = oracle.walk(inst, inst.params, S0, np.arange(W), steps, 42)
    b1, _ = sharding.walker_range(1, 2, W)
    flag[b1::3] = 0
    expect = oracle.compact(smp, flag)
    got = np.load(tmp_path / "gathered.npy")
    assert np.array_equal(got, expect)
    ball = np.load(tmp_path / "ball.npy")
    c, r, _ = oracle.meb_welzl(expect[:, 9:])
    assert abs(ball[3] - r) <= 1e-12 * r and np.allclose(ball[:3], c, atol=1e-12)


def _strong_worker(rank, world, port, W, steps, out_dir):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 16)
    Rbar = oracle.mean_pose(S0)[0]

    def sample(begin, n):
        smp, flag = oracle.walk(inst, inst.params, S0, begin + np.arange(n), steps, 42)
        flag[(begin + np.arange(n)) % 5 == 0] = 0          # ragged counts that depend on the walker id only
        return torch.from_numpy(smp), torch.from_numpy(flag)

    def compact(smp, flag):
        comp = oracle.compact(smp.numpy(), flag.numpy())
        return torch.from_numpy(comp), torch.tensor([comp.shape[0]])

    def megb(cloud, count):
        return oracle.megb(cloud.numpy()[:count], Rbar)

    res = sharding.strong_step(sample, compact, megb, W, rank, world)
    if rank == 0:
        np.save(os.path.join(out_dir, "strong.npy"), np.array([res["rot_radius"], res["trans_radius"], res["count"]]))
        np.save(os.path.join(out_dir, "counts.npy"), np.array(res["counts"]))
    else:
        assert res is None
    dist.barrier()
    dist.destroy_process_group()


def test_strong_step_equals_single_process(tmp_path):
    """Range-split walk -> compaction per rank -> unpadded gather on rank 0 -> MEGB: radii and count equal the
    one-process run bit for bit (Philox makes walker w placement-independent).  W = 50 over 3 ranks
    gives uneven ranges (17, 17, 16)."""
    import oracle
    W, steps, world = 50, 10, 3
    mp.spawn(_strong_worker, args=(world, _free_port(), W, steps, str(tmp_path)), nprocs=world, join=True)
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 16)
    smp, flag = oracle.walk(inst, inst.params, S0, np.arange(W), steps, 42)
    flag[np.arange(W) % 5 == 0] = 0
    cloud = oracle.compact(smp, flag)
    ref = oracle.megb(cloud, oracle.mean_pose(S0)[0])
    got = np.load(tmp_path / "strong.npy")
    assert got[0] == ref["rot_radius"] and got[1] == ref["trans_radius"] and int(got[2]) == cloud.shape[0]
    counts = np.load(tmp_path / "counts.npy")
    assert counts.sum() == cloud.shape[0] and len(counts) == world
