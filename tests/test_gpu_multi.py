"""The multi-GPU merge path through the C ABI on ONE GPU (`-m gpu`): the ranks of a sharded run are emulated one
after the other on cuda:0 (two contexts, no kernels waiting on one another), their tallies summed in place like the
all-reduce would, and the merged result compared with the undivided run -- the same histories, so equality holds up
to fp32 atomic order.  `run_sharded` itself is exercised end to end over NCCL with world_size 1."""
import os
import socket

import numpy as np
import pytest

import anm_inputs

pytestmark = pytest.mark.gpu

COUNTERS = ("n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff")


def _load(sim, cfg, tables, **opts):
    sim.load_config(cfg, tables, **opts)


@pytest.mark.parametrize("uncertainty", [0, 1])
def test_two_emulated_ranks_merge_to_the_undivided_run(tables, uncertainty):
    import torch
    from paper_2111_11687_b200 import Simulation
    from paper_2111_11687_b200.multi_gpu import STAT_SUM_KEYS, plan_shards
    cfg = anm_inputs.make_config(3, 4)
    n, B = 500_000, 10
    with Simulation(0) as one:
        _load(one, cfg, tables, n_batches=B, collect_stats=1, uncertainty=uncertainty)
        one.run(n, cfg["seed"])
        ref = {"energy": one.get_energy().astype(np.float64), "rel": one.get_uncertainty().astype(np.float64),
               "dose": one.get_dose().astype(np.float64), "organs": one.get_organ_doses(), "stats": one.get_stats()}
    shards = plan_shards(n, B, 2)
    sims = [Simulation(0), Simulation(0)]
    try:
        bufs, stats = [], []
        for sh, sim in zip(shards, sims):
            _load(sim, cfg, tables, n_batches=sh.n_batches, history_offset=sh.history_offset, collect_stats=1, uncertainty=uncertainty)
            sim.run(sh.n_decays, cfg["seed"])
            bufs.append(sim.get_tally_buffers())
            stats.append(sim.get_stats())
        (s0, q0, r0), (s1, q1, r1) = bufs
        assert s0.numel() == (one.V + 3) // 4 * 4 and r0.shape == (shards[0].n_batches, 256) and r0.dtype == torch.float64
        s0 += s1; q0 += q1                                       # what the sum-all-reduce leaves on rank 0
        rows_all = torch.cat([r0, r1]).cpu().numpy()             # organ rows of all batches in batch order
        summed = dict(stats[0])
        for k in STAT_SUM_KEYS:
            summed[k] = stats[0][k] + stats[1][k]
        torch.cuda.synchronize()
        sims[0].merge(n, B, rows_all, summed)
        got = {"energy": sims[0].get_energy().astype(np.float64), "rel": sims[0].get_uncertainty().astype(np.float64),
               "dose": sims[0].get_dose().astype(np.float64), "organs": sims[0].get_organ_doses(), "stats": sims[0].get_stats()}
    finally:
        for sim in sims:
            sim.close()
    assert np.allclose(got["energy"], ref["energy"], rtol=1e-4, atol=1e-3)
    assert np.allclose(got["dose"], ref["dose"], rtol=1e-4, atol=1e-12 * ref["dose"].max() + 1e-30)
    big = ref["energy"] > 0.05 * ref["energy"].max()
    assert np.allclose(got["rel"][big], ref["rel"][big], rtol=2e-3)
    for key in ("mean_Gy_per_decay", "sigma_mean", "mass_weighted_Gy_per_decay", "rms_voxel_rel_sigma"):
        assert np.allclose(got["organs"][key], ref["organs"][key], rtol=2e-4, atol=0), key
    assert np.array_equal(got["organs"]["n_voxels_nonzero"], ref["organs"]["n_voxels_nonzero"])
    for key in COUNTERS:
        assert got["stats"][key] == ref["stats"][key], key
    assert got["stats"]["n_decays"] == n and got["stats"]["emitted_MeV"] == ref["stats"]["emitted_MeV"]
    assert abs(got["stats"]["deposited_MeV"] / ref["stats"]["deposited_MeV"] - 1) < 1e-6
    assert abs(got["stats"]["escaped_MeV"] / ref["stats"]["escaped_MeV"] - 1) < 1e-6


def test_merge_error_codes(tables):
    from paper_2111_11687_b200 import AnmError, Simulation
    cfg = anm_inputs.make_config(3, 8)
    with Simulation(0) as sim:
        _load(sim, cfg, tables, n_batches=4)
        with pytest.raises(AnmError) as e:
            sim.get_tally_buffers()
        assert e.value.code == -2                                # ANM_E_STATE: no completed run
        sim.run(40_000, 1)
        rows = np.zeros((8, 256))
        with pytest.raises(AnmError) as e:
            sim.merge(80_000 + 8, 8, rows)                       # another decays-per-batch
        assert e.value.code == -1
        with pytest.raises(AnmError) as e:
            sim.merge(80_000, 8, None)                           # organs loaded: rows required
        assert e.value.code == -1
        with pytest.raises(AnmError) as e:
            sim.merge(20_000, 2, np.zeros((2, 256)))             # fewer batches than this run
        assert e.value.code == -1
        sim.merge(80_000, 8, rows)                               # a rank whose peers contributed nothing but zeros
        assert sim.get_stats()["n_decays"] == 80_000


def test_run_sharded_over_nccl_world_1(tables):
    import torch.distributed as dist
    import torch
    from paper_2111_11687_b200 import Simulation
    from paper_2111_11687_b200.multi_gpu import run_sharded
    cfg = anm_inputs.make_config(3, 4)
    n, B = 200_000, 10
    opts = dict(photons_per_decay=cfg["photons_per_decay"], rayleigh_on=cfg["rayleigh_on"],
                photon_cutoff_MeV=cfg["photon_cutoff_mev"], positron_ke_MeV=cfg["positron_ke_mev"], collect_stats=1)
    with Simulation(0) as one:
        _load(one, cfg, tables, n_batches=B, collect_stats=1)
        one.run(n, 5)
        ref_e, ref_o, ref_s = one.get_energy(), one.get_organ_doses(), one.get_stats()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        with Simulation(0) as sim:
            _load(sim, cfg, tables, n_batches=B)
            shard = run_sharded(sim, n, 5, B, opts)
            assert shard.n_batches == B and shard.history_offset == 0
            e, o, st = sim.get_energy(), sim.get_organ_doses(), sim.get_stats()
    finally:
        dist.destroy_process_group()
    assert np.allclose(e, ref_e, rtol=1e-4, atol=1e-3)
    assert np.allclose(o["mean_Gy_per_decay"], ref_o["mean_Gy_per_decay"], rtol=2e-4)
    assert np.allclose(o["sigma_mean"], ref_o["sigma_mean"], rtol=2e-3)
    for key in COUNTERS:
        assert st[key] == ref_s[key], key
