"""anm_organ_summary_static (include/anm.h, csrc/anm_static.cu) against the path every other test uses.

Some users of the library cannot let it allocate device memory: their own allocator already owns the whole card (a
PyTorch job, a server with one fixed arena), or they call from a thread on a deadline where cudaMalloc / cudaFree --
driver locks, a possible wait for the device -- are not allowed.  For them the per-organ summary of A11 exists as a
call that needs no anm_ctx and allocates nothing: its accumulators sit in a small array built into the library.

What is checked: the call gives what anm_get_organ_doses / anm_get_stats give for the same tallies (Eq. 3 RMS sigma,
voxels with energy, organ energy, total energy); twice in a row without a wait in between, and again after a different
run, because all calls share the one array and it keeps what the last call left in it; that the device's free memory
does not move across a call; and that a size the array cannot hold is refused with a message that names the limit.

This file is named to be collected last: `pytest -x` stops at the first failure, so a failure here hides nothing.
It depends on no other test and passes alone in a fresh process as well."""
import numpy as np
import pytest

import anm_inputs

pytestmark = pytest.mark.gpu

GY_PER_MEV_PER_GRAM = 1.602176634e-10
RTOL = 1e-9          # same arithmetic, fp64 sums in another order; the repo's organ comparisons allow 2e-4


@pytest.fixture(scope="module")
def anm():
    import paper_2111_11687_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def expected_rows(organs, stats, n_decays):
    """[n_organs + 1][3] from the existing path's organ table and counters."""
    n = len(organs["mass_g"])
    rows = np.zeros((n + 1, 3))
    rows[0, 2] = stats["deposited_MeV"]
    rows[1:, 0] = organs["rms_voxel_rel_sigma"]
    rows[1:, 1] = organs["n_voxels_nonzero"]
    rows[1:, 2] = organs["mass_weighted_Gy_per_decay"] * n_decays * organs["mass_g"] / GY_PER_MEV_PER_GRAM
    return rows


def check(got, want):
    assert np.array_equal(got[:, 1], want[:, 1])                       # voxel counts: exact
    assert np.allclose(got[:, 0], want[:, 0], rtol=RTOL, atol=0)
    assert np.allclose(got[:, 2], want[:, 2], rtol=RTOL, atol=0)
    assert got[0, 0] == 0.0 and got[0, 1] == 0.0
    assert want[0, 2] > 0 and np.count_nonzero(want[1:, 1]) >= 3       # the comparison is not between zeros


def test_static_scratch_matches_the_ctx_path(anm, tables):
    import torch
    cfg = anm_inputs.make_config(3, 8)                                 # small patient-like phantom with its organ labels
    V, n_org = int(np.prod(cfg["shape"])), int(cfg["n_organs"])
    labels = torch.from_numpy(np.ascontiguousarray(cfg["labels"]).reshape(-1)).cuda()
    # the caller owns the outputs; poisoned so that a word the call leaves alone shows
    outs = [torch.full((n_org + 1, 3), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=10, collect_stats=1)
        n = 200_000
        sim.run(n, cfg["seed"])
        want_a = expected_rows(sim.get_organ_doses(), sim.get_stats(), n)
        s, q, _ = sim.get_tally_buffers()
        # two calls in a row, no synchronisation in between (same stream: ordered on the GPU)
        anm.organ_summary_static(s, q, labels, n_org, 10, outs[0], n_voxels=V)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        anm.organ_summary_static(s, q, labels, n_org, 10, outs[1], n_voxels=V)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before             # the call took no device memory
        check(outs[0].cpu().numpy(), want_a)
        check(outs[1].cpu().numpy(), want_a)

        # other tallies, other batch count: nothing of the previous calls may be left in the shared array
        sim.set_options(n_batches=20, collect_stats=1, photons_per_decay=cfg["photons_per_decay"], rayleigh_on=cfg["rayleigh_on"],
                        photon_cutoff_MeV=cfg["photon_cutoff_mev"], positron_ke_MeV=cfg["positron_ke_mev"])
        n = 100_000
        sim.run(n, cfg["seed"] + 7)
        want_b = expected_rows(sim.get_organ_doses(), sim.get_stats(), n)
        s, q, _ = sim.get_tally_buffers()
        anm.organ_summary_static(s, q, labels, n_org, 20, outs[2], stream=torch.cuda.current_stream(), n_voxels=V)
        torch.cuda.synchronize()
        check(outs[2].cpu().numpy(), want_b)
        assert not np.allclose(want_a[:, 2], want_b[:, 2], rtol=1e-3)  # the two runs really differ

        # without labels: only the total
        tot = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
        anm.organ_summary_static(s, q, None, 0, 20, tot, n_voxels=V)
        torch.cuda.synchronize()
        assert np.allclose(tot.cpu().numpy(), [0.0, 0.0, want_b[0, 2]], rtol=RTOL, atol=0)


def test_static_scratch_refuses_what_it_cannot_hold(anm):
    import torch
    s = torch.zeros(1024, dtype=torch.float32, device="cuda")
    lab = torch.zeros(1024, dtype=torch.uint8, device="cuda")
    out = torch.zeros(3 * 300, dtype=torch.float64, device="cuda")
    with pytest.raises(anm.AnmError) as ei:
        anm.organ_summary_static(s, s, lab, 256, 10, out)
    assert ei.value.code == -1 and "at most 255 organs" in str(ei.value)
    with pytest.raises(anm.AnmError) as ei:
        anm.organ_summary_static(s, s, lab, 4, 1, out)                 # fewer than two samples: no variance
    assert ei.value.code == -1
    assert float(out.abs().sum()) == 0.0                               # a refused call writes nothing
