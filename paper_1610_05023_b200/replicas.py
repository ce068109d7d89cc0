"""Multi-GPU plumbing of the bench: "replicas only" (BASELINE north_star: one GPU, no sharding, no
inter-GPU collective on the data path).  With N > 1 processes every rank runs the same independent problem on its
own GPU; the only communication is the barrier around the timed region and the max-over-ranks of the measured
time.  torch.distributed is the plumbing (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import dataclasses
import os


@dataclasses.dataclass
class Replicas:
    rank: int
    world: int
    local: int
    backend: str | None = None       # None: single process, torch.distributed not initialised

    @classmethod
    def from_env(cls, backend: str = "nccl") -> "Replicas":
        """Reads RANK / WORLD_SIZE / LOCAL_RANK (torchrun); initialises torch.distributed when WORLD_SIZE > 1."""
        rank = int(os.environ.get("RANK", "0"))
        world = int(os.environ.get("WORLD_SIZE", "1"))
        local = int(os.environ.get("LOCAL_RANK", "0"))
        if world == 1:
            return cls(rank, world, local, None)
        import torch
        import torch.distributed as dist
        if backend == "nccl":
            torch.cuda.set_device(local)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
        return cls(rank, world, local, backend)

    def _device(self):
        return f"cuda:{self.local}" if self.backend == "nccl" else "cpu"

    def barrier(self) -> None:
        """Process barrier, then a device synchronize where there is a device."""
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        if self.backend != "gloo":
            import torch
            if torch.cuda.is_available():
                torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        import torch
        import torch.distributed as dist
        t = torch.tensor([float(x)], dtype=torch.float64, device=self._device())
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def all_true(self, ok: bool) -> bool:
        return self.max_over_ranks(0.0 if ok else 1.0) == 0.0

    def aggregate_rate(self, units_per_rank: float, seconds: float) -> float:
        """Whole-job throughput: the units all ranks processed over the slowest rank's time."""
        return self.world * units_per_rank / self.max_over_ranks(seconds)

    @property
    def is_root(self) -> bool:
        return self.rank == 0

    def close(self) -> None:
        if self.world > 1:
            import torch.distributed as dist
            if dist.is_initialized():
                dist.destroy_process_group()
