"""Host side of the multi-GPU path, on CPU: shard planning, and the exchange step
(`merge_tallies` / `merge_stats`) run by TWO gloo ranks on tallies the oracle computed for each rank's whole-batch
shard.  What must hold: merged sum / sum of squares / organ rows equal those of one undivided oracle run (the
histories are keyed by index, so the shards ARE the run), on every rank."""
import os
import socket

import numpy as np
import pytest

import anm_inputs
from paper_2111_11687_b200.multi_gpu import Shard, plan_shards


def test_plan_shards_partitions_whole_batches():
    for n_batches, world, per in ((100, 8, 10_000_000), (100, 1, 7), (10, 4, 3), (64, 8, 1), (17, 8, 5)):
        shards = plan_shards(n_batches * per, n_batches, world)
        assert [s.rank for s in shards] == list(range(world))
        assert shards[0].batch0 == 0 and shards[0].history_offset == 0
        for a, b in zip(shards, shards[1:]):
            assert b.batch0 == a.batch0 + a.n_batches                      # contiguous, in rank order
            assert b.history_offset == a.history_offset + a.n_decays
        assert sum(s.n_batches for s in shards) == n_batches
        assert sum(s.n_decays for s in shards) == n_batches * per
        assert all(s.n_batches >= 2 and s.n_decays == s.n_batches * per and s.history_offset == s.batch0 * per for s in shards)
        assert max(s.n_batches for s in shards) - min(s.n_batches for s in shards) <= 1


def test_plan_shards_rejects_bad_splits():
    with pytest.raises(ValueError):
        plan_shards(1000, 10, 6)          # fewer than 2 batches per rank
    with pytest.raises(ValueError):
        plan_shards(1001, 10, 2)          # N not a multiple of B
    with pytest.raises(ValueError):
        plan_shards(0, 10, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, n, B, out_dir):
    import torch
    import torch.distributed as dist
    from oracle import anm_oracle as O
    from paper_2111_11687_b200.multi_gpu import merge_stats, merge_tallies
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = anm_inputs.make_config(3, 16)
        o = O.Oracle(cfg, anm_inputs.make_tables(), n_decays=n, n_batches=B, seed=7)
        sh = plan_shards(n, B, world)[rank]
        r = o.run(sh.batch0, sh.batch0 + sh.n_batches)           # this rank's whole batches, histories keyed by index
        s, q = torch.from_numpy(r["sum"]), torch.from_numpy(r["sumsq"])
        rows = torch.from_numpy(r["organ_batch"][sh.batch0:sh.batch0 + sh.n_batches].copy())
        rows_all = merge_tallies(s, q, rows, sh, B)
        st = {"escaped_MeV": r["stats"]["escaped"], "n_steps": 0, "n_real": r["stats"]["n_collisions"], "n_pe": r["stats"]["n_pe"],
              "n_compton": r["stats"]["n_compton"], "n_rayleigh": r["stats"]["n_rayleigh"], "n_escaped": r["stats"]["n_escaped"],
              "n_cutoff": r["stats"]["n_cutoff"], "n_launches": 1, "ms_transport": 10.0 + rank, "ms_fold": 1.0, "ms_finalize": 0.5,
              "ms_setup": 2.0 - rank}
        ms = merge_stats(st, torch.device("cpu"))
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), sum=s.numpy(), sumsq=q.numpy(), rows=rows_all.numpy(),
                 n_pe=ms["n_pe"], n_compton=ms["n_compton"], escaped=ms["escaped_MeV"], ms_transport=ms["ms_transport"],
                 ms_setup=ms["ms_setup"], n_launches=ms["n_launches"])
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_merge_to_the_undivided_run(tmp_path):
    import torch.multiprocessing as mp
    from oracle import anm_oracle as O
    n, B, world = 40_000, 10, 2
    mp.spawn(_rank_main, args=(world, _free_port(), n, B, str(tmp_path)), nprocs=world, join=True)
    cfg = anm_inputs.make_config(3, 16)
    o = O.Oracle(cfg, anm_inputs.make_tables(), n_decays=n, n_batches=B, seed=7)
    full = o.run()
    for rank in range(world):
        z = np.load(os.path.join(str(tmp_path), "rank%d.npz" % rank))
        # batches are disjoint sets of histories: the merged volumes are the undivided run's up to fp64 summation order
        np.testing.assert_allclose(z["sum"], full["sum"], rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(z["sumsq"], full["sumsq"], rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(z["rows"], full["organ_batch"], rtol=1e-12, atol=0)
        assert int(z["n_pe"]) == full["stats"]["n_pe"] and int(z["n_compton"]) == full["stats"]["n_compton"]
        assert abs(float(z["escaped"]) - full["stats"]["escaped"]) < 1e-9 * full["stats"]["escaped"]
        assert float(z["ms_transport"]) == 11.0 and float(z["ms_setup"]) == 2.0 and int(z["n_launches"]) == 2
    assert full["sum"].sum() > 0 and np.count_nonzero(full["organ_batch"]) > 0


def test_merge_tallies_checks_row_count():
    import torch
    from paper_2111_11687_b200.multi_gpu import merge_tallies
    with pytest.raises(ValueError):
        merge_tallies(torch.zeros(4), torch.zeros(4), torch.zeros(3, 256), Shard(0, 0, 2, 0, 20), 4)


def test_every_counter_of_anm_stats_is_merged():
    """merge_stats must sum every additive uint64 counter of anm_stats over the ranks (a counter left out would report
    one rank's value beside globally summed ones); the few that are not additive are named here."""
    import ctypes as C
    from paper_2111_11687_b200 import binding
    from paper_2111_11687_b200.multi_gpu import STAT_MAX_KEYS, STAT_SUM_KEYS
    not_additive = {"n_decays",                    # set by anm_merge from the logical run
                    "tally_binned", "batches_per_launch", "texel_bits",      # how the run was made, the same on every rank
                    "n_voxels_gt10", "n_voxels_gt50"}                        # recomputed by anm_merge on the merged volumes
    fields = dict(binding.anm_stats._fields_)
    for name, typ in fields.items():
        if typ is C.c_uint64:
            assert name in STAT_SUM_KEYS or name in not_additive, name
    assert set(STAT_SUM_KEYS) <= set(fields) and set(STAT_MAX_KEYS) <= set(fields)
    assert not (set(STAT_SUM_KEYS) & not_additive)
