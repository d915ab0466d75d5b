"""Regression fixture of the oracle (tests/golden/oracle_regression.txt, written by tests/golden/make_golden.py)."""
import os

import numpy as np

import workloads

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_regression.txt")


def test_oracle_matches_its_frozen_fixture(oracle):
    x, _ = workloads.comb_batch_numpy(2, [7], 4096, 1.0, 50.0, 120.0, 0.10)
    rows = [l.split() for l in open(GOLD) if not l.startswith("#")]
    header = [l for l in open(GOLD) if l.startswith("# checksum")][0].split()[-1]
    assert workloads.checksum(x) == header
    outs = {v: oracle.harmonic_sum(x, 32, v, want_jpath=True) for v in ("standard", "max", "freqbin", "greedy")}
    assert len(rows) == 64
    for r in rows:
        v, n = r[0], int(r[1])
        h = np.array([float(t) for t in r[2:8]])
        np.testing.assert_array_equal(outs[v]["sums"][0, :, n], h)
        assert int(outs[v]["argmax"][0, n]) == int(r[8])
        assert int(outs[v]["jpath"][0, 5, n]) == int(r[9])
