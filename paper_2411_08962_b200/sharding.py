"""Timeslice sharding over ranks (the paper reports near-linear 2- and 4-node scaling
without describing the split).  Every (site, timeslice) is independent up to the sum over
sites of ONE timeslice (Eq. A2), so rank r contracts the timeslices t = r, r + N, r + 2N, ... of its own
propagator shard with no collective on the data path; the per-timeslice reduction order equals the single-GPU one
whenever the site batches have the same shape (always at BASELINE's sizes, where the batch is capped by the workspace
target), and then results are bitwise equal; otherwise they agree to rounding.  The only exchange is the final gather of C[p][t] (at most a few KB).

`torch.distributed` is plumbing here: any backend works (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import List, Optional

import torch
import torch.distributed as dist


def timeslices_of_rank(T: int, rank: int, world: int) -> List[int]:
    """Timeslices owned by `rank`: t = rank (mod world), ascending.  May be empty when T < world."""
    if T < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("need T >= 0, world >= 1, 0 <= rank < world")
    return list(range(rank, T, world))


def gather_correlator(C_local: torch.Tensor, T: int, group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """C_local: [n_mom][len(timeslices_of_rank(T, rank, world))] complex128, the rank's rows of C(t,p) in the order of
    timeslices_of_rank.  Returns the full [n_mom][T] tensor on every rank (one all_gather of padded shards)."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    mine = timeslices_of_rank(T, rank, world)
    if C_local.dim() != 2 or C_local.shape[1] != len(mine):
        raise ValueError(f"rank {rank}: expected [n_mom][{len(mine)}], got {tuple(C_local.shape)}")
    n_mom = C_local.shape[0]
    full = torch.zeros((n_mom, T), dtype=C_local.dtype, device=C_local.device)
    if world == 1:
        full[:, mine] = C_local
        return full
    width = (T + world - 1) // world                                 # every shard padded to the widest one
    send = torch.zeros((n_mom, width), dtype=torch.float64, device=C_local.device).repeat(1, 2)   # re | im
    send[:, :len(mine)] = C_local.real
    send[:, width:width + len(mine)] = C_local.imag
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send, group=group)
    for r in range(world):
        ts = timeslices_of_rank(T, r, world)
        full[:, ts] = torch.complex(recv[r][:, :len(ts)], recv[r][:, width:width + len(ts)])
    return full


def contract_sharded(U_local, D_local, terms, momenta, L: int, T: int, group: Optional[dist.ProcessGroup] = None, **kw):
    """U_local, D_local: [len(timeslices_of_rank)][L^3][12][12] complex128 on this rank's GPU (its timeslices, ascending).
    Contracts them with wick_contract and gathers C[p][t] for all T timeslices on every rank."""
    from . import binding
    n_local = U_local.shape[0]
    if n_local:
        C_local = binding.contract(U_local, D_local, terms, momenta, L, n_local, **kw)
    else:
        C_local = torch.zeros((len(momenta), 0), dtype=torch.complex128, device=U_local.device)
    return gather_correlator(C_local, T, group)
