"""Event-sharded evaluation across ranks ("treat different subsets of events
on different cores/machines ... then have a relatively lightweight piece of code perform a
synthesis").

One process per GPU.  Every rank holds a contiguous block of the data events and of the
accepted-MC events.  The only exchange per evaluation is the (2 + 2n)-double data-term record
{L_data, n_nonfinite, T}; per M build it is the n x n complex matrix.  Both are all-gathered and
summed IN RANK ORDER on every rank, so the result is bitwise identical on all ranks and from
run to run (a tree all-reduce would not fix the order).  torch.distributed is plumbing only:
all arithmetic on events happens in libpwa.so (pwa_data_term_enqueue / pwa_build_norm) and the
final assembly (step A7) in pwa_assemble_host.

Works with the nccl backend (CUDA tensors) and with gloo (CPU tensors; used by the tests).
"""
import numpy as np
import torch
import torch.distributed as dist


def world():
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def shard_bounds(n_events: int, rank: int, world_size: int):
    """Contiguous block [lo, hi) of rank `rank`; block sizes differ by at most one."""
    base, rem = divmod(int(n_events), int(world_size))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def sum_in_rank_order(x: torch.Tensor, group=None) -> torch.Tensor:
    """All-gather x (any shape, float64) and add the rank copies in rank order 0, 1, ..."""
    rank, ws = world()
    if ws == 1:
        return x.clone()
    x = x.contiguous()
    parts = [torch.empty_like(x) for _ in range(ws)]
    dist.all_gather(parts, x, group=group)
    out = parts[0].clone()
    for r in range(1, ws):
        out += parts[r]
    return out


def combine_norm(M_local: np.ndarray, n_gen_local: int, device=None, group=None):
    """M of the whole MC sample from per-shard matrices M_r = B_r^H B_r / N_gen,r:
    M = sum_r N_gen,r M_r / sum_r N_gen,r  (eq. 3 second term).
    -> (M [n, n, 2] float64 numpy, N_gen total)."""
    dev = device if device is not None else "cpu"
    t = torch.from_numpy(np.ascontiguousarray(M_local, dtype=np.float64) * float(n_gen_local)).to(dev)
    g = torch.tensor([float(n_gen_local)], dtype=torch.float64, device=dev)
    t = sum_in_rank_order(t, group)
    g = sum_in_rank_order(g, group)
    n_gen = int(round(float(g.item())))
    return (t / float(n_gen)).cpu().numpy(), n_gen


def reduce_terms(terms: torch.Tensor, group=None) -> torch.Tensor:
    """terms: [2 + 2n] float64 = {L_data, n_nonfinite, Re T_0, Im T_0, ...} of this rank's
    events (the record pwa_data_term_enqueue writes).  -> the same record for all events."""
    return sum_in_rank_order(terms, group)
