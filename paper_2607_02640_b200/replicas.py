"""Multi-GPU = replicas only: sessions are independent, a session lives on one GPU
for life, there is no data-path collective.  This module holds the little host logic that exists:
the session -> rank map and the max-over-ranks reduction of the timed region.  It works with any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def session_rank(global_session: int, world: int) -> int:
    """A session is pinned to one GPU for life (its KV never moves: PAPER.md:L46-50)."""
    return global_session % world


def local_sessions(n_global: int, world: int, rank: int) -> list[int]:
    return [s for s in range(n_global) if session_rank(s, world) == rank]


def uid_base(rank: int) -> int:
    """Offset of a rank's session uids in the synthetic-input coordinate space, so replicas are
    not clones of each other."""
    return rank * 1_000_000


def aggregate(ms_local: float, session_frames_local: float, device="cpu"):
    """(whole-job session-frames/s, max-over-ranks milliseconds).  Every rank must call it."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([ms_local], dtype=torch.float64, device=device)
        n = torch.tensor([session_frames_local], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
        ms, frames = float(t.item()), float(n.item())
    else:
        ms, frames = float(ms_local), float(session_frames_local)
    return frames / (ms * 1e-3), ms
