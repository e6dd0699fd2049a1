"""N > 1 path on CPU: world_size-2 `gloo` processes exercising the replica plumbing bench.py uses
(replicas only, no data-path collective)."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    sys.path.insert(0, str(ROOT))
    import torch.distributed as dist
    from paper_2011_01207_b200 import replicas
    env = replicas.RankEnv.from_env()
    assert (env.rank, env.world, env.local_rank) == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        # rank r "measured" (10 + r) ms in total and (20 + 2r) ms of wall clock
        total_ms, wall = replicas.max_over_ranks([10.0 + rank, 20.0 + 2 * rank], dist)
        assert total_ms == 10.0 + (world - 1) and wall == 20.0 + 2 * (world - 1)
        assert replicas.replicas_agree(9.0, -1234.5, dist)
        # one rank disagreeing on the energy, or on the iteration count, is detected on every rank
        assert not replicas.replicas_agree(9.0, -1234.5 - 1e-3 * rank, dist)
        assert not replicas.replicas_agree(9.0 + rank, -1234.5, dist)
        value = replicas.aggregate_throughput(1000.0, world, total_ms)
        assert abs(value - world * 1000.0 / (total_ms * 1e-3)) < 1e-9
        dist.barrier()
        Path(out_dir, f"ok{rank}").write_text(repr(value))
    finally:
        dist.destroy_process_group()


def test_two_gloo_replicas(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    v0, v1 = (float((tmp_path / f"ok{r}").read_text()) for r in (0, 1))
    assert v0 == v1 == pytest.approx(2 * 1000.0 / 11e-3)


def test_single_process_is_identity():
    from paper_2011_01207_b200 import replicas
    assert replicas.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert replicas.replicas_agree(3, 1.0)
    assert replicas.aggregate_throughput(10.0, 1, 2.0) == pytest.approx(5000.0)
    env = replicas.RankEnv.from_env({"RANK": "3", "WORLD_SIZE": "8", "LOCAL_RANK": "3"})
    assert (env.rank, env.world, env.local_rank) == (3, 8, 3)


def test_torchrun_command_uses_loopback():
    from paper_2011_01207_b200 import replicas
    cmd = replicas.torchrun_command("python", "bench.py", 4, ["--gpus", "4", "--steps", "2"], port=1234)
    assert "--nproc-per-node=4" in cmd and "127.0.0.1" in cmd and "1234" in cmd
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"]
