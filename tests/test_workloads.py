"""The seeded input generators (workloads/): recipe constants of DESIGN.md section 5 and determinism.
Citations: PAPER.md:50 (von Mises pulsar + N(0,1) noise, 20 s at 64 us); BASELINE.json configs[0..3]."""
import math

import numpy as np
import pytest

import workloads as W


def test_kappa_values_from_duty_cycle():
    # full width at half maximum = duty:  exp(kappa (cos(pi duty) - 1)) = 1/2
    for duty, kappa in ((0.01, 1404.73), (0.03, 156.18), (0.05, 56.300), (0.10, 14.162), (0.20, 3.629)):
        k = W.von_mises_kappa(duty)
        assert k == pytest.approx(kappa, rel=2e-4)
        assert math.exp(k * (math.cos(math.pi * duty) - 1)) == pytest.approx(0.5, rel=1e-12)


def test_config0_is_seeded_and_carries_the_pulsar_near_bin_1251():
    x = W.config0()
    assert x.shape == (1, 1 << 18) and x.dtype == np.float32
    assert W.checksum(x) == W.checksum(W.config0())
    # white noise: normalised power has mean 0 and unit variance away from the pulsar's harmonics
    assert abs(float(x.mean())) < 0.02 and float(x.var()) == pytest.approx(1.0, abs=0.1)   # each bin ~ Exp(1) - 1
    f0_bin = 37.3 * W.NFFT * W.TSAMP
    assert f0_bin == pytest.approx(1251.58, abs=0.01)
    k = np.arange(1, 9) * f0_bin
    near = np.maximum(x[0, np.floor(k).astype(int)], x[0, np.floor(k).astype(int) + 1])
    assert near.mean() > 3.0                      # the first harmonics stand well above the noise floor
    prof = W.pulse_train(W.NSAMP, 37.3, 0.05, 0.0)
    assert W.pulsar_amplitude(prof, 10.0) == pytest.approx(0.0959, abs=5e-4)


def test_config1_streams_are_independent_and_ten_percent_injected():
    sub = [0, 1, 2, 3]
    x, params = W.config1(sub, nsamp=4096, nfft=8192, nbins=4096)
    x2, _ = W.config1([2], nsamp=4096, nfft=8192, nbins=4096)
    np.testing.assert_array_equal(x[2], x2[0])
    flags = [W.rng_for(1, b).random() < 0.10 for b in range(256)]
    assert 10 <= sum(flags) <= 45
    for b, p in zip(sub, params):
        assert (p is not None) == flags[b]


def test_comb_split_and_scale():
    rng = W.rng_for(2, 123)
    bins, vals, f0, S = W.comb(rng, 1 << 18, 50.0, 5000.0, 0.10)
    assert 50.0 <= f0 < 5000.0 and 5.0 <= S < 20.0
    assert bins.min() >= 0 and bins.max() < (1 << 18) and (vals >= 0).all()
    a = W.comb_powers(0.10)
    assert (np.diff(a) < 0).all()                 # von Mises coefficients decay monotonically
    # sinc^2 split keeps at most the harmonic's power and at least 81 % of it (scalloping at half a bin)
    tot = a * (S * math.sqrt(32) / a.sum())
    assert 0.8 * tot.sum() <= vals.sum() <= tot.sum() * (1 + 1e-6)


def test_exp_noise_numpy_and_torch_cpu():
    import torch
    x = W.exp_noise_numpy(W.rng_for(2, 0), 1 << 16)
    assert x.dtype == np.float32 and x.min() >= -1.0
    assert float(x.mean()) == pytest.approx(0.0, abs=0.02) and float(x.var()) == pytest.approx(1.0, abs=0.05)
    t = W.exp_noise_torch(4, 1 << 12, 2, "cpu")
    t2 = W.exp_noise_torch(4, 1 << 12, 2, "cpu")
    assert torch.equal(t, t2) and t.dtype == torch.float32 and float(t.min()) >= -1.0
    xb, inj = W.comb_batch_numpy(3, [0, 1], 1 << 14, 1.0, 100.0, 400.0, 0.03)
    assert inj.all() and xb.shape == (2, 1 << 14)
