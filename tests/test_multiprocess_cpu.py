"""N > 1 host logic on CPU: world_size-2 gloo run of the sharding + max-over-ranks timing reduction of bench.py,
and the state generator's sub-range property that weak scaling relies on."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import mechgen as mg
from paper_1809_01029_b200.sharding import shard_range, weak_scaling_offset


def test_shard_ranges_cover_and_align():
    for n, world, tile in ((1000, 3, 8), (262144, 8, 4), (5, 4, 1), (0, 2, 4), (17, 2, 16)):
        rs = [shard_range(n, r, world, tile) for r in range(world)]
        assert rs[0][0] == 0 and rs[-1][1] == n
        for (a, b), (c, d) in zip(rs, rs[1:]):
            assert b == c and a <= b
        assert all(a % tile == 0 or a == n for a, _ in rs)
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def test_state_subranges_are_consistent():
    """config_states(c, n, start) must equal the slice of the full set (each rank generates only its shard)."""
    full = mg.config_states(2, 3000)
    for r in range(2):
        off = weak_scaling_offset(1500, r)
        part = mg.config_states(2, 1500, start=off)
        assert np.array_equal(part["n"], full["n"][:, off:off + 1500]) and np.array_equal(part["T"], full["T"][off:off + 1500])


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    a, b = shard_range(1001, rank, world, 4)
    st = mg.config_states(1, b - a, start=a)
    t = torch.tensor([10.0 + rank], dtype=torch.float64)          # per-rank elapsed time
    dist.all_reduce(t, op=dist.ReduceOp.MAX)                        # bench.py: time = max over ranks
    cnt = torch.tensor([float(b - a)], dtype=torch.float64)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    chk = torch.tensor([float(st["T"].sum())], dtype=torch.float64)
    dist.all_reduce(chk, op=dist.ReduceOp.SUM)
    dist.barrier()
    if rank == 0:
        q.put((t.item(), cnt.item(), chk.item()))
    dist.destroy_process_group()


def test_two_rank_gloo_sharded_run():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    tmax, total, chk = q.get()
    assert tmax == 11.0 and total == 1001.0
    assert chk == pytest.approx(float(mg.config_states(1, 1001)["T"].sum()), rel=1e-12)


def _stub_rank(args):
    """What bench.rank_main does around its timed region, with the GPU step stubbed: gloo instead of nccl."""
    import json
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    assert int(os.environ["LOCAL_RANK"]) == rank and os.environ["MASTER_ADDR"] == "127.0.0.1"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n_per_rank, steps = 1000, 4
    off = weak_scaling_offset(n_per_rank, rank)                     # every rank owns its own states (weak scaling)
    dist.barrier()
    t = torch.tensor([0.5 + 0.25 * rank], dtype=torch.float64)      # stubbed per-rank elapsed seconds
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    offs = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(offs, torch.tensor([off]))
    if rank == 0:
        with open(args.out, "w") as f:
            json.dump({"n_gpus": world, "value": world * n_per_rank * steps / t.item(), "offsets": [int(o) for o in offs]}, f)
    dist.destroy_process_group()


def test_bench_gpus_n_spawns_its_own_ranks(tmp_path):
    """`python bench.py --gpus N` outside torchrun: bench.spawn_ranks starts N ranks with torchrun's environment."""
    import json
    import bench
    args = bench.parse_args(["--gpus", "2", "--steps", "4"])
    args.out = str(tmp_path / "line.json")
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    bench.spawn_ranks(args.gpus, _stub_rank, args, port=port)
    line = json.load(open(args.out))
    assert line["n_gpus"] == 2 and line["offsets"] == [0, 1000]
    assert line["value"] == pytest.approx(2 * 1000 * 4 / 0.75)
    # one GPU: no spawn, the rank runs in this process (main() -> rank_main directly)
    assert bench.parse_args([]).gpus == 1
