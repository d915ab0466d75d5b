"""Sensitivity sweep of BASELINE.json configs[4] (Figs. 1-2): recovered signal-to-noise ratio of the four
harmonic-sum variants (and of eq. 1 with interpolated terms) for a pulsar whose frequency lies between two Fourier bins,
relative to the standard sum (eq. 1).

    python -m paper_1812_02647_b200.sensitivity [--realisations 1024] [--out gpurun_out/sensitivity.json]

Recipe:
  * `R` noise series of 312 500 samples N(0,1) (20 s at 64 us), zero-padded to 2^19, transformed ONCE (common random
    numbers); for each sweep point (fractional bin offset delta of f0 in 0, 0.05 .. 0.5; duty cycle in 1 .. 40 %) the
    von Mises pulse train of matched-filter SNR 8 is transformed once and added in the Fourier domain (the transform is
    linear), then x = |F|^2 / 312500 - 1 as fp32: R x 2^18 bins per point.  f0 = (1251 + delta) bins of the padded transform.
  * The library (hs_execute, full planes, Hmax = 32) runs the four variants on the R spectra.
  * h is turned into a signal-to-noise ratio per variant and level with the mean and standard deviation of the same
    variant and level on the noise-only spectra (A17: the maximum of i noise bins has a positive mean), the candidate is
    the best (level, bin) with the fundamental within +-1 bin of the truth (eq. 1 at level H: top harmonic at H f0).
Input generation (series, transforms) uses torch on the device: plumbing, none of the method's arithmetic.  Everything
downstream of x runs in libhs.so; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# "standard_interp": eq. 1 with its terms read on the line between the two neighbouring bins (HS_TERM_INTERP,
# CONVENTIONS.md C15) instead of at the nearest bin
VARIANTS = ["standard", "max", "freqbin", "greedy", "standard_interp"]
K0 = 1251                                   # integer part of the fundamental bin (configs[0]: 37.3 Hz -> bin 1251.58)
DELTAS = [0.05 * k for k in range(11)]
DUTIES = [0.01, 0.02, 0.05, 0.10, 0.20, 0.40]
LEVELS = 6


def noise_transforms(R, dev, slab=64):
    """F[R][2^18] complex64-pair (float64 transform, kept as complex128) of R seeded N(0,1) series."""
    import torch

    import workloads as W
    g = torch.Generator(device=dev).manual_seed(W.S0 + 4)
    out = torch.empty((R, W.NBINS0), dtype=torch.complex128, device=dev)
    for r0 in range(0, R, slab):
        n = min(slab, R - r0)
        s = torch.randn((n, W.NSAMP), dtype=torch.float64, device=dev, generator=g)
        out[r0:r0 + n] = torch.fft.rfft(s, n=W.NFFT, dim=1)[:, :W.NBINS0]
    return out


def signal_transform(delta, duty, snr, dev):
    """Transform of the pulse train with f0 = (K0 + delta) bins of the padded transform, matched-filter SNR `snr`."""
    import torch

    import workloads as W
    f0_hz = (K0 + delta) / (W.NFFT * W.TSAMP)
    prof = W.pulse_train(W.NSAMP, f0_hz, duty, 0.25)
    amp = W.pulsar_amplitude(prof, snr)
    s = torch.from_numpy(prof * amp).to(dev)
    return torch.fft.rfft(s, n=W.NFFT)[:W.NBINS0]


def spectra_of(Fn, Fs):
    """x = |Fn + Fs|^2 / NSAMP - 1 as fp32 (Fs may be None: noise only)."""
    import torch

    import workloads as W
    x = torch.empty(Fn.shape, dtype=torch.float32, device=Fn.device)
    for r0 in range(0, Fn.shape[0], 64):
        F = Fn[r0:r0 + 64] if Fs is None else Fn[r0:r0 + 64] + Fs
        x[r0:r0 + 64] = ((F.real * F.real + F.imag * F.imag) / float(W.NSAMP) - 1.0).to(torch.float32)
    return x


def level_planes(hs, x, variant):
    """h[R][6][N] of one variant through the C ABI (hs_execute, full output, Hmax = 32)."""
    import torch
    R, N = x.shape
    if variant == "standard_interp":
        plan = hs.hs_plan_create_ex(N, R, 32, "standard", "full", "dyadic", "interp")
    else:
        plan = hs.hs_plan_create(N, R, 32, variant, "full")
    plan.ensure_workspace(x.device)
    sums = torch.empty((R, LEVELS, N), dtype=torch.float32, device=x.device)
    plan.hs_execute(x, sums, None, None)
    torch.cuda.synchronize()
    plan.hs_destroy()
    return sums


def calibration(hs, x_noise):
    """mean and standard deviation of h per (variant, level) on noise-only spectra, over bins where every harmonic is
    in range (eqs. 2-4: 256 <= n < N/32; eq. 1: N/32 <= n < N)."""
    N = x_noise.shape[1]
    cal = {}
    for v in VARIANTS:
        h = level_planes(hs, x_noise, v)
        lo, hi = (N // 32, N) if v.startswith("standard") else (256, N // 32)
        part = h[:, :, lo:hi].double()
        cal[v] = (part.mean(dim=(0, 2)), part.std(dim=(0, 2)))
        del h, part
    return cal


def recovered_snr(hs, x, cal, f_true):
    """Per variant: mean over the realisations of max over (level, bin within +-1 fundamental bin of f_true) of the
    calibrated SNR; for eq. 1 at level H the bin is that of the top harmonic, so the window is H (f_true +- 1)."""
    import torch
    out = {}
    for v in VARIANTS:
        h = level_planes(hs, x, v)
        mu, sd = cal[v]
        best = torch.full((x.shape[0],), -1e30, dtype=torch.float64, device=x.device)
        for l in range(LEVELS):
            H = 1 << l
            scale = H if v.startswith("standard") else 1
            lo = int(math.ceil(scale * (f_true - 1.0)))
            hi = int(math.floor(scale * (f_true + 1.0)))
            z = (h[:, l, lo:hi + 1].double() - mu[l]) / sd[l]
            best = torch.maximum(best, z.max(dim=1).values)
        out[v] = float(best.mean())
        del h
    return out


def run(realisations=1024, snr=8.0, deltas=DELTAS, duties=DUTIES, device="cuda:0"):
    import torch

    from paper_1812_02647_b200 import binding as hs
    dev = torch.device(device)
    torch.cuda.set_device(dev)
    Fn = noise_transforms(realisations, dev)
    cal = calibration(hs, spectra_of(Fn, None))
    points = []
    for duty in duties:
        for delta in deltas:
            x = spectra_of(Fn, signal_transform(delta, duty, snr, dev))
            rec = recovered_snr(hs, x, cal, K0 + delta)
            points.append({"duty": duty, "delta": delta, "snr": rec,
                           "relative_to_standard": {v: rec[v] / rec["standard"] for v in VARIANTS}})
            del x
    return {"realisations": realisations, "input_snr": snr, "k0": K0, "points": points,
            "calibration": {v: {"mean": cal[v][0].tolist(), "std": cal[v][1].tolist()} for v in VARIANTS}}


def summarise(res):
    """Markdown: recovered SNR relative to eq. 1 per duty cycle, on-bin (delta = 0), worst offset and mean over offsets."""
    lines = ["| duty | variant | on-bin SNR | SNR at delta = 0.5 | mean over delta | mean relative to eq. 1 |", "|---:|---|---:|---:|---:|---:|"]
    duties = sorted({p["duty"] for p in res["points"]})
    for d in duties:
        pts = sorted((p for p in res["points"] if p["duty"] == d), key=lambda p: p["delta"])
        for v in VARIANTS:
            s = [p["snr"][v] for p in pts]
            ref = [p["snr"]["standard"] for p in pts]
            lines.append(f"| {100 * d:.0f} % | {v} | {s[0]:.2f} | {s[-1]:.2f} | {sum(s) / len(s):.2f} | "
                         f"{sum(s) / sum(ref):.3f} |")
    return "\n".join(lines)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--realisations", type=int, default=1024)
    ap.add_argument("--snr", type=float, default=8.0)
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    res = run(args.realisations, args.snr)
    if args.out:
        with open(args.out, "w") as f:
            json.dump(res, f)
    print(summarise(res))


if __name__ == "__main__":
    main()
