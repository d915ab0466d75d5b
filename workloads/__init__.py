"""Seeded synthetic inputs for the harmonic-sum configs of BASELINE.json (configs[0..4]).

This module is the ONLY thing the oracle side and the CUDA side have in common, and it holds
none of the method's arithmetic: it produces normalised power spectra x[B][N] (the input of
eqs. 1-4) and nothing downstream of them.  The recipe follows PAPER.md:50
(modified von Mises pulse train + N(0,1) noise, 20 s at 64 us) and DESIGN.md section 5.

Seeding: base seed S0; the NumPy stream of (config c, spectrum b) is default_rng([S0, c, b]);
bulk noise generated with torch uses torch.Generator(device).manual_seed(S0 + c) and is
deterministic per device type.
"""
from __future__ import annotations

import math

import numpy as np

S0 = 181202647
TSAMP = 64e-6
NSAMP = 312500              # 20 s at 64 us
NFFT = 1 << 19              # zero-padded transform length (BASELINE.json configs[0])
NBINS0 = 1 << 18


def rng_for(config: int, spectrum: int) -> np.random.Generator:
    return np.random.default_rng([S0, int(config), int(spectrum)])


def von_mises_kappa(duty: float) -> float:
    """kappa such that exp(kappa(cos 2 pi phi - 1)) has full width at half maximum `duty` (in phase)."""
    return math.log(2.0) / (1.0 - math.cos(math.pi * duty))


def pulse_train(nsamp: int, f0_hz: float, duty: float, phi0: float, tsamp: float = TSAMP) -> np.ndarray:
    """Modified von Mises profile train I(phi) = exp(kappa(cos 2 pi (phi - phi0) - 1))."""
    t = np.arange(nsamp, dtype=np.float64) * tsamp
    return np.exp(von_mises_kappa(duty) * (np.cos(2.0 * np.pi * (f0_hz * t - phi0)) - 1.0))


def pulsar_amplitude(profile: np.ndarray, snr: float) -> float:
    """Amplitude giving matched-filter SNR `snr` against unit-variance white noise (reading R-A19)."""
    return snr / math.sqrt(float(np.sum((profile - profile.mean()) ** 2)))


def spectrum_from_series(series: np.ndarray, nfft: int = NFFT, nbins: int = NBINS0) -> np.ndarray:
    """Zero-pad, float64 FFT, P_k = |F_k|^2, x_k = P_k/len(series) - 1, cast to fp32 (configs[0])."""
    F = np.fft.rfft(series.astype(np.float64), n=nfft)[:nbins]
    P = F.real * F.real + F.imag * F.imag
    return (P / float(series.shape[0]) - 1.0).astype(np.float32)


def time_domain_spectrum(rng: np.random.Generator, f0_hz=None, duty=None, snr=None,
                         nsamp: int = NSAMP, nfft: int = NFFT, nbins: int = NBINS0) -> np.ndarray:
    """One spectrum built in the time domain; f0_hz=None gives noise only."""
    series = rng.standard_normal(nsamp)
    if f0_hz is not None:
        prof = pulse_train(nsamp, f0_hz, duty, rng.random())
        series = series + pulsar_amplitude(prof, snr) * prof
    return spectrum_from_series(series, nfft, nbins)


def config0(nsamp: int = NSAMP, nfft: int = NFFT, nbins: int = NBINS0) -> np.ndarray:
    """configs[0]: one spectrum, f0 = 37.3 Hz, 5 % duty cycle, time-domain SNR 10.  Returns x[1][nbins]."""
    return time_domain_spectrum(rng_for(0, 0), 37.3, 0.05, 10.0, nsamp, nfft, nbins)[None, :]


def config1(spectra, nsamp: int = NSAMP, nfft: int = NFFT, nbins: int = NBINS0):
    """configs[1]: DM-trial spectra `spectra` (indices in [0,256)); 10 % carry one pulsar with
    f0 ~ U[1,200) Hz, duty ~ U[0.01,0.20), SNR ~ U[5,20).  Returns (x[len][nbins], list of params or None)."""
    xs, params = [], []
    for b in spectra:
        rng = rng_for(1, b)
        if rng.random() < 0.10:
            f0, duty, snr = rng.uniform(1.0, 200.0), rng.uniform(0.01, 0.20), rng.uniform(5.0, 20.0)
            params.append((f0, duty, snr))
            xs.append(time_domain_spectrum(rng, f0, duty, snr, nsamp, nfft, nbins))
        else:
            params.append(None)
            xs.append(time_domain_spectrum(rng, None, None, None, nsamp, nfft, nbins))
    return np.stack(xs), params


def comb_powers(duty: float, nharm: int = 32, nphase: int = 4096) -> np.ndarray:
    """Relative harmonic powers |c_k|^2, k = 1..nharm, of the von Mises profile (DFT of the sampled profile)."""
    phi = np.arange(nphase, dtype=np.float64) / nphase
    prof = np.exp(von_mises_kappa(duty) * (np.cos(2.0 * np.pi * phi) - 1.0))
    c = np.fft.rfft(prof)[1:nharm + 1]
    return c.real ** 2 + c.imag ** 2


def comb(rng: np.random.Generator, nbins: int, f0_lo: float, f0_hi: float, duty: float, nharm: int = 32):
    """Injected pulsar comb (configs[2], configs[3]): harmonics at k*f0 bins, powers from comb_powers scaled so
    that sum_k a_k/sqrt(nharm) = S with S ~ U[5,20), each split over the two nearest bins with sinc^2 weights,
    harmonics beyond the spectrum dropped.  Returns (bins int64[], additive power fp32[], f0, S)."""
    f0 = rng.uniform(f0_lo, f0_hi)
    S = rng.uniform(5.0, 20.0)
    a = comb_powers(duty, nharm)
    a = a * (S * math.sqrt(nharm) / a.sum())
    bins, vals = [], []
    for k in range(1, nharm + 1):
        fk = k * f0
        lo = int(math.floor(fk))
        d = fk - lo
        for idx, w in ((lo, np.sinc(d) ** 2), (lo + 1, np.sinc(1.0 - d) ** 2)):
            if 0 <= idx < nbins:
                bins.append(idx)
                vals.append(a[k - 1] * w)
    return np.asarray(bins, np.int64), np.asarray(vals, np.float32), f0, S


def exp_noise_numpy(rng: np.random.Generator, nbins: int) -> np.ndarray:
    """x_k = E_k - 1, E_k ~ Exp(1) i.i.d.: the normalised white-noise power distribution (configs[2])."""
    return (rng.standard_exponential(nbins, dtype=np.float32) - np.float32(1.0)).astype(np.float32)


def comb_batch_numpy(config: int, spectra, nbins: int, frac: float, f0_lo: float, f0_hi: float, duty: float):
    """Host version of configs[2]/[3] for a list of spectrum indices (NumPy streams).  Returns (x, injected mask)."""
    xs, inj = [], []
    for b in spectra:
        rng = rng_for(config, b)
        x = exp_noise_numpy(rng, nbins)
        has = rng.random() < frac
        if has:
            bins, vals, _, _ = comb(rng, nbins, f0_lo, f0_hi, duty)
            np.add.at(x, bins, vals)
        xs.append(x)
        inj.append(has)
    return np.stack(xs), np.asarray(inj)


def exp_noise_torch(batch: int, nbins: int, config: int, device, out=None):
    """Bulk Exp(1)-1 noise generated directly on `device` (plumbing: torch RNG, no method arithmetic)."""
    import torch
    g = torch.Generator(device=device).manual_seed(S0 + int(config))
    x = out if out is not None else torch.empty((batch, nbins), dtype=torch.float32, device=device)
    rows = max(1, (1 << 26) // nbins)            # fill in slabs to bound temporary memory
    for r0 in range(0, batch, rows):
        x[r0:r0 + rows].exponential_(1.0, generator=g).sub_(1.0)
    return x


def inject_combs_torch(x, config: int, frac: float, f0_lo: float, f0_hi: float, duty: float):
    """Add combs (host-computed positions and powers, NumPy streams) to a device batch x[B][N] in place.
    Returns the list of injected spectrum indices."""
    import torch
    B, N = x.shape
    injected = []
    for b in range(B):
        rng = rng_for(config, b)
        if rng.random() < frac:
            bins, vals, _, _ = comb(rng, N, f0_lo, f0_hi, duty)
            x[b].index_add_(0, torch.as_tensor(bins, device=x.device),
                            torch.as_tensor(vals, device=x.device))
            injected.append(b)
    return injected


def config2_torch(device, batch: int = 4096, nbins: int = 1 << 18):
    """configs[2]: Exp(1)-1 noise, 1 % of spectra with a comb, f0 ~ U[50,5000) bins, 10 % duty."""
    x = exp_noise_torch(batch, nbins, 2, device)
    return x, inject_combs_torch(x, 2, 0.01, 50.0, 5000.0, 0.10)


def config3_torch(device, batch: int = 8, nbins: int = 1 << 23):
    """configs[3]: 8 x 2^23 Exp(1)-1 noise, one comb per spectrum, f0 ~ U[1000,100000) bins, 3 % duty."""
    x = exp_noise_torch(batch, nbins, 3, device)
    return x, inject_combs_torch(x, 3, 1.0, 1000.0, 100000.0, 0.03)


def checksum(x) -> str:
    """Order-independent 64-bit checksum of spectrum 0's bit patterns (printed by bench.py for reproducibility)."""
    a = np.ascontiguousarray(np.asarray(x)[0] if np.asarray(x).ndim == 2 else np.asarray(x), dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    idx = np.arange(u.shape[0], dtype=np.uint64)
    return f"{int(np.bitwise_xor.reduce((u + idx * np.uint64(2654435761)) & np.uint64(0xFFFFFFFFFFFF))):012x}"
