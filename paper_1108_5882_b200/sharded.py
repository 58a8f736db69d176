"""Event-sharded evaluation across ranks ("treat different subsets of events
on different cores/machines ... then have a relatively lightweight piece of code perform a
synthesis").

One process per GPU.  Every rank holds a contiguous block of the data events and of the
accepted-MC events.  The only exchange per evaluation is the (2 + 2n)-double data-term record
{L_data, n_nonfinite, T}; per M build it is the n x n complex matrix of sums and N_gen.  Both are
ALL-GATHERED (no reduction in the collective), and every rank hands the gathered array to
libpwa.so, which adds the shards in rank order (pwa_assemble_host_shards,
pwa_combine_norm_host): the result is bitwise identical on all ranks and from run to run (a tree
all-reduce would not fix the order).  This module is plumbing only: it moves buffers with
torch.distributed and calls the C ABI; it holds none of the method's arithmetic.

Works with the nccl backend (CUDA tensors) and with gloo (CPU tensors).
"""
import numpy as np
import torch
import torch.distributed as dist

from . import binding as pwa


def world():
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def shard_bounds(n_events: int, rank: int, world_size: int):
    """Contiguous block [lo, hi) of rank `rank`; block sizes differ by at most one."""
    base, rem = divmod(int(n_events), int(world_size))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather(x: torch.Tensor, group=None) -> np.ndarray:
    """All-gather x (any shape) -> numpy [world_size, *x.shape] on the host, rank r in row r."""
    _, ws = world()
    x = x.contiguous()
    if ws == 1:
        return x.detach().cpu().numpy()[None].copy()
    parts = [torch.empty_like(x) for _ in range(ws)]
    dist.all_gather(parts, x, group=group)
    return torch.stack(parts).cpu().numpy()


def _exchange_device(device):
    if device is not None:
        return device
    return "cuda" if dist.is_initialized() and dist.get_backend() == "nccl" else "cpu"


def combine_norm_sums(G: np.ndarray, n_gen: int, device=None, group=None):
    """Per-shard sums G_r = B_r^H B_r [n, n, 2] and N_gen,r of every rank -> (M [n, n, 2], N_gen total) with
    M = sum_r G_r / sum_r N_gen,r (eq. 3 second term; arithmetic in pwa_combine_norm_host)."""
    dev = _exchange_device(device)
    G_all = gather(torch.from_numpy(np.ascontiguousarray(G, dtype=np.float64)).to(dev), group)
    ng_all = gather(torch.tensor([int(n_gen)], dtype=torch.int64, device=dev), group).reshape(-1)
    return pwa.pwa_combine_norm_host(G_all, ng_all)


def combine_norm(ctx, device=None, group=None):
    """After pwa_build_norm on every rank: exchanges the per-shard sums and installs the M of ALL MC events in
    ctx (pwa_norm_sums -> all-gather -> pwa_combine_norm_host -> pwa_set_norm).  -> (M [n, n, 2], N_gen total)."""
    G, n_gen = pwa.pwa_norm_sums(ctx)
    M, n_gen_total = combine_norm_sums(G, n_gen, device, group)
    pwa.pwa_set_norm(ctx, M)
    return M, n_gen_total


def gather_terms(terms: torch.Tensor, group=None) -> np.ndarray:
    """terms: [2 + 2n] float64 = {L_data, n_nonfinite, Re T_0, Im T_0, ...} of this rank's events (the record
    pwa_data_term_enqueue writes; a CUDA tensor is gathered on the stream it was written on).
    -> [world_size, 2 + 2n] on the host, for pwa_assemble_host_shards."""
    return gather(terms, group)


def nll_grad(ctx, V, M, out_dev: torch.Tensor, likelihood=0, n_data_total=0.0, group=None):
    """One sharded evaluation: data term of this rank's events, exchange, synthesis (step A7) on every rank.
    out_dev: CUDA float64 tensor [2 + 2n] on the context's device, written on the context's stream (which must
    be torch's current stream, so that the gather is ordered behind the kernel).  -> (nll, grad[n, 2], parts[2])."""
    pwa.pwa_data_term_enqueue(ctx, V, out_dev)
    _, ws = world()
    if ws > 1 and dist.get_backend() != "nccl":
        terms = gather_terms(out_dev.cpu(), group)          # .cpu() synchronises with the current stream
    else:
        terms = gather_terms(out_dev, group)
    return pwa.pwa_assemble_host_shards(terms, M, V, likelihood, n_data_total)
