"""The N > 1 path (replicas only): world_size-2 gloo processes on CPU."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_0909_0928_b200 import replicas
    r, w = replicas.init("gloo")
    assert (r, w) == (rank, world)
    replicas.barrier()
    # rank 1 is the slow one and does more work
    agg = replicas.aggregate(units_local=10.0 * (rank + 1), seconds_local=1.0 + rank)
    out.put((rank, agg, replicas.replica_seed(202, rank)))
    dist.destroy_process_group()


def test_aggregate_world_size_2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, agg, seed in res:
        assert agg["units"] == 30.0 and agg["seconds"] == 2.0 and agg["value"] == 15.0
    assert [s for _, _, s in res] == [202, 1202]


def test_single_process_is_identity():
    from paper_0909_0928_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert replicas.env_world() == (0, 0, 1)
    assert replicas.aggregate(6.0, 2.0) == {"units": 6.0, "seconds": 2.0, "value": 3.0}


def test_bench_spawns_its_own_ranks():
    """`python bench.py --gpus 2` outside torchrun must start the two ranks itself and report n_gpus = 2 only
    because two ranks reported (here with the CPU stub in place of the GPU step, gloo backend)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--stub", "--steps", "3"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=root)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1            # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["units"] == 6.0
    # max over ranks: rank 1 sleeps 20 ms per step
    assert line["ms_per_step"] >= 19.0


def test_slab_plan_covers_the_volume():
    from paper_0909_0928_b200 import slabs as SL
    assert SL.halo_planes(1.0) == 4 and SL.halo_planes(2.0) == 7
    for nz, world in ((256, 8), (100, 3), (44, 4), (37, 2), (9, 1)):
        plan = SL.plan(nz, world, 4)
        assert plan[0].own0 == 0 and plan[-1].own1 == nz
        for a, b in zip(plan, plan[1:]):
            assert a.own1 == b.own0                      # own ranges tile the volume
            assert a.hi == a.own1 + 4 and b.lo == b.own0 - 4
        assert plan[0].lo == 0 and plan[-1].hi == nz     # no halo beyond a face of the volume
        assert max(s.own_count for s in plan) - min(s.own_count for s in plan) <= 1
    with pytest.raises(ValueError):
        SL.plan(12, 4, 4)                                # 3 planes per rank cannot fill a 4-plane halo


def test_slab_loop_refuses_what_it_cannot_do():
    """iterate_slabs: eps > 0 (the stopping rule needs an all-reduce per iteration) and a halo thinner than the
    smoothing radius + 1 are refused before any kernel is launched."""
    from paper_0909_0928_b200 import slabs as SL
    plan = SL.plan(40, 2, SL.halo_planes(1.0))
    with pytest.raises(ValueError, match="stopping rule"):
        SL.iterate_slabs([], plan, None, None, [], [], 5, 1.0, SL.LocalExchange(plan), eps=1e-4)
    with pytest.raises(ValueError, match="halo"):
        SL.iterate_slabs([], plan, None, None, [], [], 5, 2.0, SL.LocalExchange(plan))
    with pytest.raises(ValueError, match="fewer than the halo"):
        SL.plan(256, 64, SL.halo_planes(2.0))            # 512x512x256 on 64 ranks at sigma 2: 4 planes < halo 7


def _slab_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    from paper_0909_0928_b200 import replicas, slabs as SL
    replicas.init("gloo")
    nz, ny, nx, halo = 23, 3, 5, 4
    s = SL.plan(nz, world, halo)[rank]
    # the "field": plane z of component c holds 100 c + z on own planes, -1 in the halos
    f = torch.full((3, s.count, ny, nx), -1.0)
    for c in range(3):
        for z in range(s.own0, s.own1):
            f[c, z - s.lo] = 100.0 * c + z
    SL.DistExchange(s).refresh(f)
    want = torch.stack([torch.stack([torch.full((ny, nx), 100.0 * c + z) for z in range(s.lo, s.hi)]) for c in range(3)])
    out.put((rank, bool(torch.equal(f, want))))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_slab_halo_exchange_over_gloo(world):
    """DistExchange (the NCCL path's bookkeeping) on CPU: after one refresh every halo plane holds the
    neighbour's own plane."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]
