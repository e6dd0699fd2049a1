"""Host logic of the N > 1 launch: independent replicas, one process per GPU.

SURVEY 8(e) / BASELINE.json: "Everything runs on one GPU, with no sharding, no collectives between
GPUs".  ``bench.py --gpus N`` therefore runs N replicas of the same problem (weak scaling).  The only
inter-rank traffic is measurement plumbing: a barrier on both sides of the timed region, the MAX
over ranks of the device-timed duration, and a check that every replica solved the same problem
(iteration count and energy agree).  Nothing here touches the data path; the functions take any
initialised ``torch.distributed`` backend (``nccl`` on the GPU box, ``gloo`` in the CPU tests).
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass
class RankEnv:
    rank: int
    world: int
    local_rank: int

    @classmethod
    def from_env(cls, env=None) -> "RankEnv":
        env = os.environ if env is None else env
        return cls(int(env.get("RANK", "0")), int(env.get("WORLD_SIZE", "1")), int(env.get("LOCAL_RANK", "0")))


def torchrun_command(python: str, script: str, n_gpus: int, argv: list[str], port: int = 29531) -> list[str]:
    """The command ``python bench.py --gpus N`` re-launches itself with (one rank per GPU, 127.0.0.1)."""
    return [python, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), script] + list(argv)


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX over ranks of a list of floats (identity when dist is None)."""
    vals = [float(v) for v in values]
    if dist is None:
        return vals
    import torch
    t = torch.tensor(vals, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def replicas_agree(iters: float, energy: float, dist=None, device="cpu", rel_tol: float = 1e-9) -> bool:
    """True iff every replica reports the same PCG iteration count and the same energy."""
    if dist is None:
        return True
    import torch
    t = torch.tensor([iters, -iters, energy, -energy], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    hi_it, lo_it, hi_e, lo_e = float(t[0]), -float(t[1]), float(t[2]), -float(t[3])
    return hi_it == lo_it and abs(hi_e - lo_e) <= rel_tol * max(abs(hi_e), abs(lo_e), 1e-300)


def aggregate_throughput(units_per_rank_step: float, world: int, max_ms_per_step: float) -> float:
    """Whole-job rate: the units ALL ranks processed in one step / the slowest rank's step time."""
    return world * units_per_rank_step / (max_ms_per_step * 1e-3)
