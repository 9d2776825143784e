"""The device random number generator, bit for bit (north_star (d): Philox4x32 keyed by history index; SURVEY.md §8(c)
P1): the known-answer vectors of tests/golden/philox4x32_10_kat.txt and the oracle's own Philox4x32-10 on random
counters and keys, through anm_philox_blocks -- the function the transport kernels call, with the round keys the
host side of anm_run prepares."""
import os

import numpy as np
import pytest

from oracle import anm_oracle as O

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_device_philox_known_answers_and_oracle():
    import paper_2111_11687_b200 as pkg
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    with pkg.Simulation(0) as sim:
        for r in rows:
            v = [int(x, 16) for x in r if x != "->"]
            ctr, key, want = v[0:4], v[4:6], v[6:10]
            got = sim.philox_blocks(key[0] | (key[1] << 32), [ctr])[0]
            assert [int(x) for x in got] == want, (r, [hex(int(x)) for x in got])
        rng = np.random.default_rng(9)
        for _ in range(8):
            seed = int(rng.integers(0, 2 ** 63)) * 2 + int(rng.integers(0, 2))
            ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
            # the layout the kernels use: counter = (history lo, history hi, block, stream)
            ctr[:500, 3] = rng.integers(0, 3, size=500)
            ctr[:500, 2] = rng.integers(0, 64, size=500)
            got = sim.philox_blocks(seed, ctr)
            key = [seed & 0xffffffff, seed >> 32]
            want = np.array([O.philox4x32_10(c, key) for c in ctr])
            assert np.array_equal(got, want)


def test_peaks_sweep_reports_saturated_rates():
    """anm_measure_peaks (include/anm.h): the gather / RED denominators are the best of a depth sweep, and the combined
    loads + REDs rate cannot beat the faster of the two alone and stays within a small factor of the slower one."""
    import paper_2111_11687_b200 as pkg
    with pkg.Simulation(0) as sim:
        p = sim.measure_peaks(64 << 20, 512 << 20)
    for k in range(2):
        assert p["gather_in_flight"][k] in (4, 8, 16, 32) and p["red_in_flight"][k] in (4, 8, 16, 32)
        assert p["gather_gps"][k] > 0 and p["red_gps"][k] > 0 and p["mix_gps"][k] > 0
        # (two arrays: twice the footprint of the single-array runs, so the mix may sit well below either of them)
        assert 0.2 * min(p["gather_gps"][k], p["red_gps"][k]) < p["mix_gps"][k] < 1.05 * max(p["gather_gps"][k], p["red_gps"][k])
    assert p["gather_gps"][0] > p["gather_gps"][1] and p["red_gps"][0] > p["red_gps"][1]     # L2-resident beats HBM
    assert p["issue_gtis"] > 1e3 and p["philox_gblocks"] > 10
