"""One logical run over several GPUs, one process per GPU (include/anm.h "one logical run over
several GPUs").  Histories are independent and keyed by index, so the run shards by WHOLE BATCHES with no
data-path collective during transport; the one exchange step is the merge of the tallies at the end: an in-place
sum-all-reduce of the per-voxel sum and sum-of-squares volumes (NCCL over NVLink when the tensors are CUDA), and
the organ rows of every batch.  Everything here is plumbing over torch.distributed; the arithmetic (transport,
fold, finalize on the merged volumes) runs in libanm.so.
"""
from __future__ import annotations

from dataclasses import dataclass

# every additive field of anm_stats (tests/test_multi_gpu_host.py checks that no uint64 counter of the struct is left out;
# n_decays is set by anm_merge from the logical run, tally_binned is a flag)
STAT_SUM_KEYS = ("escaped_MeV", "n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff", "n_launches",
                 "n_electrons", "n_hbh_overflow", "n_tally_overflow", "n_fly_trips", "n_compton_tries", "n_rayleigh_tries",
                 "n_check_violations")
STAT_MAX_KEYS = ("ms_transport", "ms_fold", "ms_finalize", "ms_setup")


@dataclass(frozen=True)
class Shard:
    rank: int
    batch0: int            # first batch of this rank
    n_batches: int         # whole batches of this rank
    history_offset: int    # index of its first history = batch0 * decays_per_batch
    n_decays: int          # n_batches * decays_per_batch


def plan_shards(n_decays: int, n_batches: int, world: int) -> list[Shard]:
    """Whole batches per rank, as even as possible, in rank order; every rank needs >= 2 batches (the C ABI's
    minimum for the batch-method uncertainty), and n_decays must be a multiple of n_batches (reading C15)."""
    if world < 1 or n_batches < 2 * world:
        raise ValueError("need at least 2 batches per rank: n_batches = %d, world = %d" % (n_batches, world))
    if n_decays <= 0 or n_decays % n_batches:
        raise ValueError("n_decays must be a positive multiple of n_batches")
    per = n_decays // n_batches
    base, rem = divmod(n_batches, world)
    out, b0 = [], 0
    for r in range(world):
        k = base + (1 if r < rem else 0)
        out.append(Shard(r, b0, k, b0 * per, k * per))
        b0 += k
    return out


def merge_tallies(sum_t, sumsq_t, organ_rows, shard: Shard, n_batches: int, group=None):
    """The exchange step.  sum_t / sumsq_t: this rank's volumes, reduced IN PLACE (SUM over ranks); organ_rows: this
    rank's [shard.n_batches][K] rows.  Returns the [n_batches][K] rows of the whole run, in batch order, on every
    rank.  Works on CUDA tensors (NCCL) and CPU tensors (gloo)."""
    import torch
    import torch.distributed as dist
    if tuple(organ_rows.shape[:1]) != (shard.n_batches,):
        raise ValueError("organ_rows has %d rows, the shard has %d batches" % (organ_rows.shape[0], shard.n_batches))
    rows_all = torch.zeros((n_batches,) + tuple(organ_rows.shape[1:]), dtype=organ_rows.dtype, device=organ_rows.device)
    rows_all[shard.batch0:shard.batch0 + shard.n_batches] = organ_rows
    dist.all_reduce(sum_t, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(sumsq_t, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(rows_all, op=dist.ReduceOp.SUM, group=group)     # disjoint row ranges: a gather written as a sum
    return rows_all


def merge_stats(stats: dict, device, group=None) -> dict:
    """Counters and escaped energy summed over ranks, phase times as the max over ranks."""
    import torch
    import torch.distributed as dist
    s = torch.tensor([float(stats.get(k, 0)) for k in STAT_SUM_KEYS], dtype=torch.float64, device=device)
    m = torch.tensor([float(stats[k]) for k in STAT_MAX_KEYS], dtype=torch.float64, device=device)
    dist.all_reduce(s, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(m, op=dist.ReduceOp.MAX, group=group)
    out = dict(stats)
    for k, v in zip(STAT_SUM_KEYS, s.tolist()):
        out[k] = int(round(v)) if k.startswith("n_") else v
    out.update(zip(STAT_MAX_KEYS, m.tolist()))
    return out


def run_sharded(sim, n_decays: int, seed: int, n_batches: int, options: dict, group=None) -> Shard:
    """Run this rank's shard of the logical run (n_decays, n_batches, seed) on `sim` (inputs already loaded) and merge:
    afterwards every rank's `sim.get_*` returns the result of the whole run.  `options`: the anm_options fields other
    than n_batches / history_offset.  Where several ranks share one device (or one process holds several contexts), give
    each `sim.set_tally_budget(...)` before `set_grid`: every context otherwise sets 4 GiB of batch tallies aside."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    shard = plan_shards(n_decays, n_batches, world)[rank]
    opts = dict(options)
    opts.update(n_batches=shard.n_batches, history_offset=shard.history_offset)
    sim.set_options(**opts)
    sim.run(shard.n_decays, seed)
    s, q, rows = sim.get_tally_buffers()
    rows_all = merge_tallies(s, q, rows, shard, n_batches, group)
    stats = merge_stats(sim.get_stats(), s.device, group)
    if s.is_cuda:
        # the all-reduces ran on torch's current stream, anm_merge launches on the ctx stream: order them explicitly
        # (they are the same stream in bench.py; a ctx on another non-blocking stream would otherwise race)
        import torch
        torch.cuda.current_stream(s.device).synchronize()
    sim.merge(n_decays, n_batches, rows_all.cpu().numpy() if sim.n_organs else None, stats)
    return shard
