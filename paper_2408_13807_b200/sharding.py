"""Host-side plan of the multi-GPU runs; no arithmetic of the method lives here.

One process per GPU.  What shards, and how:
  * full IRE on one model couples all packages through the cell energies: it does NOT shard.
    `bench.py --gpus N` runs N independent replicas, each with its own seed (`replica_seed`);
  * fixed-temperature tracking: packages are independent, so the package ids [0, n) are cut into contiguous
    ranges (`package_range`), each rank follows its range with `dies_run(..., n_total=n, accumulate)` semantics
    (ids continue, energies are L / n_total), and the 64-bit integer tallies are summed with one all-reduce
    (`allreduce_tallies`): integer sums are order independent, so the result is bit-identical to one GPU;
  * config 5 (independent spheres): models are dealt to ranks (`model_range`, `batch_shard`; the shard's handle
    keeps the models' indices in the Philox counter with dies_set_model_offset), no collective at all.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def replica_seed(base_seed: int, step: int, rank: int) -> int:
    """Seed of replica `rank` at step `step`: distinct Philox keys for every (rank, step)."""
    return int(base_seed) + int(step) + 7919 * int(rank)


def package_range(n_packages: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range [first, first + count) of package ids of rank `rank`; ranges tile [0, n) exactly and
    differ in length by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    q, r = divmod(int(n_packages), int(world))
    first = rank * q + min(rank, r)
    return first, q + (1 if rank < r else 0)


def model_range(n_models: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range of model indices of rank `rank` (config 5: independent spheres, no exchange)."""
    return package_range(n_models, rank, world)


def batch_shard(batch, rank: int, world: int):
    """The spheres of a config-5 batch dealt to rank `rank`: (sub-batch, index of its first model).  The shard's handle
    takes that index with dies_set_model_offset, so that its packages are those the whole batch would follow."""
    import dataclasses
    first, count = model_range(batch.n_models, rank, world)
    sl = slice(first, first + count)
    meta = {k: (v[sl] if hasattr(v, "shape") and getattr(v, "shape", ()) and v.shape[0] == batch.n_models else v)
            for k, v in batch.meta.items()}
    return dataclasses.replace(batch, r_bounds=batch.r_bounds[sl], rho=batch.rho[sl],
                               ext_bin_intensity=batch.ext_bin_intensity[sl], meta=meta), first


def sum_over_ranks(x: float, device) -> float:
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def allreduce_tallies(*tallies: torch.Tensor) -> list[torch.Tensor]:
    """Sum int64 tally arrays (absorbed raw units per shell, escaped raw units per bin, counters) over all ranks
    with ONE all-reduce.  The tensors live where the backend wants them (CUDA for nccl, CPU for gloo)."""
    for t in tallies:
        if t.dtype != torch.int64:
            raise TypeError("tallies are 64-bit integers (fixed point): the sum over ranks must be exact")
    flat = torch.cat([t.reshape(-1) for t in tallies])
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(flat, op=dist.ReduceOp.SUM)
    out, o = [], 0
    for t in tallies:
        out.append(flat[o:o + t.numel()].reshape(t.shape))
        o += t.numel()
    return out


def max_over_ranks(ms: float, device) -> float:
    """Device time of a multi-rank step = the slowest rank's."""
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_fixed_T_shard(model, n_total: int, seed: int, rank: int, world: int, **opts):
    """Fixed-temperature tracking of this rank's share of an n_total-package run on `model` (a binding.Model whose
    fixed temperatures are set): follows the rank's package-id range, then sums the integer tallies over the ranks.
    Returns (absorbed raw units per shell summed over the ranks, this rank's escaped energy per bin, this rank's
    counters)."""
    import numpy as np
    from . import binding

    first, count = package_range(n_total, rank, world)
    if count > 0:
        model.dies_seek(first)
        model.dies_run(count, seed=seed, mode=binding.DIES_MODE_FIXED_T, n_total=n_total, **opts)
        raw, unit, _ = model.dies_get_absorbed()
        esc = model.dies_get_escape_spectrum()
        counters = model.dies_get_counters()
    else:
        raw, unit, esc, counters = np.zeros(model.N, dtype=np.int64), 0.0, np.zeros(model.K), {}
    dev = model.device if dist.is_available() and dist.is_initialized() and dist.get_backend() == "nccl" else "cpu"
    (raw_sum,) = allreduce_tallies(torch.as_tensor(np.ascontiguousarray(raw), dtype=torch.int64, device=dev))
    return raw_sum.cpu().numpy(), esc, counters
