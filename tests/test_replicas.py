"""The N > 1 path is "replicas only": its host-side logic -- which realisation a rank
takes, MAX of the timed region, SUM of the counts -- exercised with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    import torch.distributed as dist
    from paper_1908_03301_b200 import inputs, replicas
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, lr, w = replicas.env_rank_world()
        assert (r, lr, w) == (rank, rank, world)
        net = inputs.cfg4_fbm_cut_3d(12, 10, 8, seed=replicas.replica_seed(3, rank))
        shas = replicas.gather_list(net.sha256())
        t_max = replicas.reduce_max(1.5 * (rank + 1))
        n_sum = replicas.reduce_sum(100 + rank)
        mine = replicas.assign(5, rank, world)
        all_assigned = replicas.gather_list(mine)
        dist.barrier()
        q.put((rank, shas, t_max, n_sum, all_assigned))
    finally:
        dist.destroy_process_group()


def test_replicas_world2_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    res.sort()
    for rank, shas, t_max, n_sum, all_assigned in res:
        assert len(shas) == world and shas[0] != shas[1]          # every rank solves its own realisation
        assert t_max == pytest.approx(3.0)                         # the job is as slow as its slowest rank
        assert n_sum == pytest.approx(201.0)                       # whole-job counts are sums
        assert sorted(sum(all_assigned, [])) == [0, 1, 2, 3, 4]    # every problem owned exactly once
        assert all_assigned[0] == [0, 2, 4] and all_assigned[1] == [1, 3]
    assert res[0][1] == res[1][1]


def test_single_process_paths():
    from paper_1908_03301_b200 import replicas
    assert replicas.reduce_max(2.5) == 2.5
    assert replicas.reduce_sum(7) == 7.0
    assert replicas.gather_list("a") == ["a"]
    assert replicas.assign(3, 0, 1) == [0, 1, 2]
    assert replicas.replica_seed(3, 0) == 3
