"""Parity of the SURVEY.md section 8(f) rows on the GPU (through the C ABI) with oracle/hs_oracle_ext.c: every integer H
up to 64, eq. 2 with the window as printed, the two-dimensional sum over the f - fdot plane, and the fused power-spectrum
front end.  Tolerances as CONVENTIONS.md C10."""
import numpy as np
import pytest
import torch

import workloads as W
from parity import argmax_from_levels, check_argmax, check_sums

pytestmark = pytest.mark.gpu
VARIANTS = ["standard", "max", "freqbin", "greedy"]


@pytest.fixture(scope="module")
def hs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1812_02647_b200 import build
    build.build()
    import paper_1812_02647_b200.binding as binding
    return binding


@pytest.fixture(scope="module")
def ext():
    from oracle import ext as _ext
    _ext.build()
    return _ext


def compare(plan, got, ref, what, x_np=None, printed=False):
    sums, vmax, amax = got
    if sums is not None:
        check_sums(sums.cpu().numpy(), ref["sums"], what + " sums")
        if x_np is not None and not printed:
            np.testing.assert_array_equal(sums[:, 0].cpu().numpy(), x_np)          # h_1 = x bit-exactly
    if vmax is not None:
        check_sums(vmax.cpu().numpy(), ref["max"], what + " max")
        check_argmax(amax.cpu().numpy(), ref["argmax"], ref["second"], ref["gap"], ref["max"], what + " argmax")
    if sums is not None and vmax is not None:
        pick = torch.gather(sums, 1, amax.long().unsqueeze(1)).squeeze(1)
        assert torch.equal(pick, vmax), what + " max != sums[argmax]"


# ------------------------------------------------------------------------------------------ every integer H, printed window
@pytest.mark.parametrize("variant", VARIANTS)
def test_every_integer_H_whole_batch(hs, ext, variant):
    rng = np.random.default_rng(41)
    for N, B, Hmax in ((4, 1, 64), (100, 2, 64), (4100, 2, 64), (20000, 3, 24), (1 << 15, 2, 7), (2052, 5, 1)):
        x, _ = W.comb_batch_numpy(2, list(range(B)), N, 0.5, 5.0, max(6.0, N / 40), 0.10) if N >= 256 else \
            ((rng.standard_exponential((B, N)) - 1).astype(np.float32), None)
        d_x = torch.from_numpy(x).cuda()
        for out_mode in ("both", "reduced", "full"):
            plan = hs.hs_plan_create_ex(N, B, Hmax, variant, out_mode, "all", "c2")
            assert plan.levels == Hmax and plan.algo == hs.HS_ALGO_GENERAL and plan.workspace_bytes() == 0
            got = plan.run(d_x)
            plan.device_status()
            ref = ext.harmonic_sum_all(x, Hmax, variant, want_jpath=(variant == "greedy"))
            compare(plan, got, ref, f"all-H {variant}/{out_mode}/N={N}/Hmax={Hmax}", x)
            if variant == "greedy" and out_mode == "full":
                d_j = torch.empty((B, Hmax, N), dtype=torch.uint8, device="cuda")
                plan.hs_debug_greedy_paths(d_x, d_j)
                torch.cuda.synchronize()
                np.testing.assert_array_equal(d_j.cpu().numpy(), ref["jpath"])
            plan.hs_destroy()


def test_every_integer_H_degenerate_spectra_and_ties(hs, ext):
    N = 3000
    rng = np.random.default_rng(42)
    cases = [np.zeros(N), -np.ones(N), np.ones(N), np.arange(N), np.arange(N)[::-1], rng.integers(-2, 3, N)]
    x = np.stack(cases).astype(np.float32)
    d_x = torch.from_numpy(x).cuda()
    for variant in VARIANTS:
        plan = hs.hs_plan_create_ex(N, len(cases), 48, variant, "both", "all", "c2")
        compare(plan, plan.run(d_x), ext.harmonic_sum_all(x, 48, variant), f"all-H degenerate {variant}", x)


def test_eq2_window_as_printed(hs, ext):
    for N, B, Hmax, levels in ((20000, 3, 32, "dyadic"), (4100, 2, 64, "all"), (100, 1, 16, "dyadic"), (1 << 15, 2, 40, "all")):
        x, _ = W.comb_batch_numpy(2, list(range(B)), N, 1.0, 5.0, max(6.0, N / 40), 0.10) if N >= 256 else \
            ((np.random.default_rng(43).standard_exponential((B, N)) - 1).astype(np.float32), None)
        d_x = torch.from_numpy(x).cuda()
        ref = ext.harmonic_sum_all(x, Hmax, "max", "printed")
        if levels == "dyadic":                                   # the dyadic levels of the all-H oracle
            pick = [h - 1 for h in (1, 2, 4, 8, 16, 32, 64) if h <= Hmax]
            ref_sums = ref["sums"][:, pick]
            best, second, gap, m = argmax_from_levels(np.moveaxis(ref_sums, 1, -1))
            ref = {"sums": ref_sums, "max": m, "argmax": best, "second": second, "gap": gap}
        shifted = np.concatenate([x[:, 1:], np.zeros((B, 1), np.float32)], axis=1)          # h_1(n) = x(n + 1)
        # ("reduced" alone is the only mode in which the kernel stops at the first harmonic that is out of range for the warp
        # and emits the first and the last remaining level only)
        for out_mode in ("both", "reduced", "full"):
            plan = hs.hs_plan_create_ex(N, B, Hmax, "max", out_mode, levels, "printed")
            sums, vmax, amax = plan.run(d_x)
            torch.cuda.synchronize()
            compare(plan, (sums, vmax, amax), ref, f"printed window N={N} Hmax={Hmax} {levels} {out_mode}", printed=True)
            if sums is not None:
                np.testing.assert_array_equal(sums[:, 0].cpu().numpy(), shifted)
            plan.hs_destroy()
    with pytest.raises(hs.HsError) as e:
        hs.hs_plan_create_ex(4096, 1, 32, "greedy", "full", "dyadic", "printed")
    assert e.value.code == hs.HS_ERR_INVALID_ARG


def test_eq1_interpolated_terms(hs, ext):
    """HS_TERM_INTERP (CONVENTIONS.md C15): eq. 1 read on the line between the two bins around n i / H, every integer H and
    the dyadic levels, all three output modes, whole batches against the oracle; candidates too."""
    from parity import check_candidates
    rng = np.random.default_rng(45)
    for N, B, Hmax, levels in ((4, 1, 64, "all"), (100, 2, 64, "all"), (4100, 2, 64, "all"), (20000, 3, 32, "dyadic"),
                               (1 << 15, 2, 7, "all"), (2052, 5, 1, "dyadic"), (12000, 2, 16, "dyadic")):
        x, _ = W.comb_batch_numpy(2, list(range(B)), N, 0.5, 5.0, max(6.0, N / 40), 0.10) if N >= 256 else \
            ((rng.standard_exponential((B, N)) - 1).astype(np.float32), None)
        d_x = torch.from_numpy(x).cuda()
        ref = ext.harmonic_sum_all(x, Hmax, "standard", "interp")
        if levels == "dyadic":
            pick = [h - 1 for h in (1, 2, 4, 8, 16, 32) if h <= Hmax]
            ref_sums = ref["sums"][:, pick]
            best, second, gap, m = argmax_from_levels(np.moveaxis(ref_sums, 1, -1))
            ref = {"sums": ref_sums, "max": m, "argmax": best, "second": second, "gap": gap}
        for out_mode in ("both", "reduced", "full"):
            plan = hs.hs_plan_create_ex(N, B, Hmax, "standard", out_mode, levels, "interp")
            assert plan.algo == hs.HS_ALGO_GENERAL and plan.workspace_bytes() == 0
            assert plan.levels == (Hmax if levels == "all" else len(pick))
            got = plan.run(d_x)
            plan.device_status()
            compare(plan, got, ref, f"interp eq. 1 {levels}/{out_mode}/N={N}/Hmax={Hmax}", x)
            if out_mode == "reduced" and N >= 4100:
                thr = 4.0
                b, n = np.nonzero(ref["max"] > thr)
                cref = {"spectrum": b.astype(np.int64), "bin": n.astype(np.int64), "margin": np.abs(ref["max"] - thr),
                        "max": ref["max"], "argmax_all": ref["argmax"], "second": ref["second"], "gap": ref["gap"]}
                count, rec = plan.run_candidates(d_x, thr, capacity=B * N)
                check_candidates(count, {k: v.cpu().numpy() for k, v in rec.items()}, cref, (B, N), f"interp candidates N={N}")
            plan.hs_destroy()
    # a ramp is reproduced exactly by the line between bins: S_H(n) = a n (H + 1)/2 + b H (the nearest-bin sum is not)
    N = 4096
    ramp = (0.25 * np.arange(N) - 3.0).astype(np.float32)
    plan = hs.hs_plan_create_ex(N, 1, 64, "standard", "full", "all", "interp")
    sums, _, _ = plan.run(torch.from_numpy(ramp[None]).cuda())
    H = np.arange(1, 65)[:, None]
    check_sums(sums[0].cpu().numpy(), (0.25 * np.arange(N)[None, :] * (H + 1) / 2 - 3.0 * H) / np.sqrt(H), "interp ramp")
    for variant in ("max", "freqbin", "greedy"):                        # only eq. 1 has an argument between bins
        with pytest.raises(hs.HsError) as e:
            hs.hs_plan_create_ex(4096, 1, 32, variant, "full", "all", "interp")
        assert e.value.code == hs.HS_ERR_INVALID_ARG


def test_eq1_interpolated_terms_sampled_at_bench_size(hs, ext):
    """256 x 2^18, Hmax 64, reduced output (the shape of bench.py --workload allh), sampled outputs."""
    B, N, Hmax = 256, 1 << 18, 64
    d_x = W.exp_noise_torch(B, N, 7, "cuda")
    rng = np.random.default_rng(46)
    spectra = np.array([0, 1, 100, 255])
    bidx = np.concatenate([rng.choice(spectra, 1200), rng.choice(spectra, 400)])
    nidx = np.concatenate([rng.integers(0, N, 1200), rng.integers(0, 4096, 400)])
    x_rows = d_x[spectra].cpu().numpy()
    remap = {int(b): i for i, b in enumerate(spectra)}
    plan = hs.hs_plan_create_ex(N, B, Hmax, "standard", "reduced", "all", "interp")
    _, vmax, amax = plan.run(d_x)
    plan.device_status()
    h, _ = ext.points_all(x_rows, Hmax, "standard", np.array([remap[int(b)] for b in bidx]), nidx, "interp")
    best, second, gap, m = argmax_from_levels(h)
    tb, tn = torch.as_tensor(bidx, device="cuda"), torch.as_tensor(nidx, device="cuda")
    check_sums(vmax[tb, tn].cpu().numpy(), m, "interp sampled max")
    check_argmax(amax[tb, tn].cpu().numpy(), best, second, gap, m, "interp sampled argmax")
    assert bool((vmax >= d_x).all())                                    # h_1 = x is one of the levels
    plan.hs_destroy()


def test_general_plans_reject_other_families_and_bad_arguments(hs):
    plan = hs.hs_plan_create_ex(4096, 2, 64, "freqbin", "reduced", "all", "c2")
    for algo in ("direct", "tiled", "gather"):
        with pytest.raises(hs.HsError):
            plan.set_algo(algo)
    plan.set_algo("auto")
    for bad in ((4096, 1, 65, "max", "full", "all", "c2"), (4096, 1, 0, "max", "full", "all", "c2"),
                (1 << 25, 1, 8, "max", "reduced", "all", "c2")):
        with pytest.raises(hs.HsError) as e:
            hs.hs_plan_create_ex(*bad)
        assert e.value.code == hs.HS_ERR_INVALID_ARG
    for bad in ((4096, 4, 1, 32, "standard", "full"), (4096, 5, 1, 32, "max", "full"), (4096, 5, 1, 3, "standard", "full")):
        with pytest.raises(hs.HsError) as e:
            hs.hs_plan_create_2d(*bad)
        assert e.value.code == hs.HS_ERR_INVALID_ARG
    d = hs.hs_plan_create_ex(4096, 1, 32, "max", "full", "dyadic", "c2")          # the plain plan: not general
    assert d.algo != hs.HS_ALGO_GENERAL


@pytest.mark.parametrize("variant", VARIANTS)
def test_candidates_on_every_integer_H_plans(hs, ext, variant):
    """hs_execute_candidates on HS_LEVELS_ALL plans (level = H - 1) and on the printed window: the records are the bins
    whose reduced maximum, as the all-H oracle gives it, exceeds the threshold."""
    from parity import check_candidates
    for N, B, Hmax, window in ((20000, 3, 48, "c2"), (4100, 2, 64, "c2"), (1 << 15, 2, 17, "printed")):
        if window == "printed" and variant != "max":
            continue
        x, _ = W.comb_batch_numpy(2, list(range(B)), N, 1.0, 5.0, max(6.0, N / 40), 0.10)
        d_x = torch.from_numpy(x).cuda()
        full = ext.harmonic_sum_all(x, Hmax, variant, window)
        plan = hs.hs_plan_create_ex(N, B, Hmax, variant, "reduced", "all", window)
        for thr in (3.0, 8.0, 40.0):
            m = full["max"]
            b, n = np.nonzero(m > thr)
            ref = {"spectrum": b.astype(np.int64), "bin": n.astype(np.int64), "margin": np.abs(m - thr), "max": m,
                   "argmax_all": full["argmax"], "second": full["second"], "gap": full["gap"]}
            count, rec = plan.run_candidates(d_x, thr, capacity=B * N)
            check_candidates(count, {k: v.cpu().numpy() for k, v in rec.items()}, ref, (B, N),
                             f"all-H candidates {variant}/N={N}/Hmax={Hmax}/{window}/thr={thr}")
        plan.hs_destroy()


def test_every_integer_H_sampled_at_bench_size(hs, ext):
    """The shape bench.py --workload allh times (256 spectra x 2^18 bins, Hmax 64, reduced), sampled outputs."""
    B, N, Hmax = 256, 1 << 18, 64
    d_x = W.exp_noise_torch(B, N, 7, "cuda")
    rng = np.random.default_rng(44)
    spectra = np.array([0, 1, 100, 255])
    bidx = np.concatenate([rng.choice(spectra, 1200), rng.choice(spectra, 400)])
    nidx = np.concatenate([rng.integers(0, N, 1200), rng.integers(0, N // 64, 400)])
    x_rows = d_x[spectra].cpu().numpy()
    remap = {int(b): i for i, b in enumerate(spectra)}
    tb, tn = torch.as_tensor(bidx, device="cuda"), torch.as_tensor(nidx, device="cuda")
    for variant in VARIANTS:
        plan = hs.hs_plan_create_ex(N, B, Hmax, variant, "reduced", "all", "c2")
        _, vmax, amax = plan.run(d_x)
        plan.device_status()
        h, _ = ext.points_all(x_rows, Hmax, variant, np.array([remap[int(b)] for b in bidx]), nidx)
        best, second, gap, m = argmax_from_levels(h)
        check_sums(vmax[tb, tn].cpu().numpy(), m, f"all-H bench shape {variant} max")
        check_argmax(amax[tb, tn].cpu().numpy(), best, second, gap, m, f"all-H bench shape {variant} argmax")
        assert bool((vmax >= d_x).all()) and int(amax.max()) <= Hmax - 1


# ------------------------------------------------------------------------------------------ two-dimensional sum
@pytest.mark.parametrize("variant", ["standard", "freqbin"])
def test_2d_whole_batch(hs, ext, variant):
    rng = np.random.default_rng(51)
    # (8192 and 2^15 bins at Hmax 32, reduced: the standard sum then runs eq. 1's register-blocked kernel, one harmonic
    # window per plane row; 24 rows x 8 tiles x 3 planes = 576 tiles, more than the resident CTAs)
    for N, Z, B, Hmax in ((8, 1, 2, 32), (100, 3, 2, 32), (4100, 9, 2, 32), (1000, 41, 1, 8), (2052, 5, 3, 2), (20000, 7, 1, 16),
                          (8192, 9, 2, 32), (1 << 15, 25, 3, 32)):
        x = (rng.standard_exponential((B, Z, N)) - 1).astype(np.float32)
        x[0, Z // 2, N // 3] += 30.0
        d_x = torch.from_numpy(x).cuda()
        for out_mode in ("both", "reduced", "full"):
            plan = hs.hs_plan_create_2d(N, Z, B, Hmax, variant, out_mode)
            assert (plan.algo == hs.HS_ALGO_GENERAL) == (Z > 1)        # a one-row plane is the 1-D problem
            got = plan.run(d_x if Z > 1 else d_x.view(B, N))
            got = tuple(None if t is None else (t if Z > 1 else t.unsqueeze(-2)) for t in got)
            plan.device_status()
            ref = ext.harmonic_sum_2d(x, Hmax, variant)
            compare(plan, got, ref, f"2-D {variant}/{out_mode}/N={N}/Z={Z}/Hmax={Hmax}", x)


@pytest.mark.parametrize("variant", ["standard", "freqbin"])
def test_2d_host_buffer_entry_and_launch_count(hs, variant):
    """hs_execute_host on 2-D plans (the slab layout counts nz rows per entry; the standard sum at 8192 bins, Hmax 32,
    reduced output runs eq. 1's register-blocked kernel and needs its tile counter in every lane's workspace), and
    hs_plan_launches against the kernels a 2-D execute really enqueues (counted by the CUDA profiler)."""
    N, B, slab = 8192, 5, 2
    for Z in (3, 9):
        x = W.exp_noise_torch(B, Z * N, 9, "cpu").view(B, Z, N).contiguous().pin_memory()
        plan = hs.hs_plan_create_2d(N, Z, B, 32, variant, "reduced")
        d_x = x.cuda()
        _, vmax_d, amax_d = plan.run(d_x)
        staging = torch.empty(plan.host_staging_bytes(slab), dtype=torch.uint8, device="cuda")
        plan.set_host_staging(staging, slab)
        h_max = torch.empty((B, Z, N), dtype=torch.float32).pin_memory()
        h_amax = torch.empty((B, Z, N), dtype=torch.uint8).pin_memory()
        plan.hs_execute_host(x, None, h_max, h_amax)
        assert plan.device_status() == hs.HS_OK
        assert torch.equal(h_max, vmax_d.cpu()) and torch.equal(h_amax, amax_d.cpu())
        # launches: the standard sum = memset node + rb_kernel; freq-bin = hs_2d_kernel + the streaming kernel for the outer
        # rows, which exist from Z = 3 on
        assert plan.launches() == 2
        vmax = torch.empty_like(vmax_d)
        amax = torch.empty_like(amax_d)
        torch.cuda.synchronize()
        try:
            from torch.profiler import ProfilerActivity, profile
            with profile(activities=[ProfilerActivity.CUDA]) as prof:
                plan.hs_execute(d_x, None, vmax, amax)
                torch.cuda.synchronize()
            names = [e.name for e in prof.events()
                     if e.name.startswith("Memset") or "hs_2d_" in e.name or "rb_kernel" in e.name]
        except Exception:                                           # (no CUPTI on this box: the count above stands alone)
            names = []
        if names:
            assert len(names) == plan.launches(), names
        plan.hs_destroy()
    full = hs.hs_plan_create_2d(N, 3, B, 32, variant, "full")       # full output: the general kernels for both variants
    assert full.launches() == (2 if variant == "freqbin" else 1)
    one = hs.hs_plan_create_2d(N, 3, B, 1, "freqbin", "full")       # a single level: nothing to stream separately
    assert one.launches() == 1


def test_2d_recovers_an_integer_harmonic_track_and_matches_1d_on_the_zero_drift_row(hs):
    Z, N, r0, z0, Zc = 129, 8192, 100, -2, 64
    amp = (5.0 * 0.9 ** np.arange(32) + 0.25).astype(np.float32)
    plane = np.zeros((1, Z, N), np.float32)
    for k in range(1, 33):
        plane[0, k * z0 + Zc, k * r0] = amp[k - 1]
    rng = np.random.default_rng(52)
    plane[0, Zc] = (rng.standard_exponential(N) - 1).astype(np.float32)           # noise on the zero-drift row only
    d = torch.from_numpy(plane).cuda()
    std, _, _ = hs.hs_plan_create_2d(N, Z, 1, 32, "standard", "full").run(d)
    fb, _, _ = hs.hs_plan_create_2d(N, Z, 1, 32, "freqbin", "full").run(d)
    for l, H in enumerate((1, 2, 4, 8, 16, 32)):
        want = float(np.cumsum(amp.astype(np.float64))[H - 1]) / np.sqrt(H)
        assert float(std[0, l, H * z0 + Zc, H * r0]) == pytest.approx(want, rel=1e-5)
        assert float(fb[0, l, z0 + Zc, r0]) == pytest.approx(want, rel=1e-5)
    one_d, _, _ = hs.hs_plan_create(N, 1, 32, "standard", "full").run(d[:, Zc].contiguous())
    assert torch.equal(std[0, :, Zc], one_d[0])                                    # z = 0: the 1-D kernels' result, bit for bit


def test_2d_sampled_at_bench_size(hs, ext):
    """The shape bench.py --workload plane times: 8 planes of 129 drifts x 2^18 bins, reduced output."""
    B, Z, N = 8, 129, 1 << 18
    d_x = W.exp_noise_torch(B * Z, N, 8, "cuda").view(B, Z, N)
    rng = np.random.default_rng(53)
    planes = [0, 7]
    x_rows = d_x[planes].cpu().numpy()
    P = 1500
    pb, pz, pn = rng.integers(0, 2, P), rng.integers(0, Z, P), rng.integers(0, N, P)
    for variant in ("standard", "freqbin"):
        plan = hs.hs_plan_create_2d(N, Z, B, 32, variant, "reduced")
        _, vmax, amax = plan.run(d_x)
        plan.device_status()
        h = np.array([[ext.partial_sum_2d(x_rows[b], n, z, H, variant) / np.sqrt(H) for H in (1, 2, 4, 8, 16, 32)]
                      for b, z, n in zip(pb, pz, pn)])
        best, second, gap, m = argmax_from_levels(h)
        tb = torch.as_tensor(np.array(planes)[pb], device="cuda")
        tz, tn = torch.as_tensor(pz, device="cuda"), torch.as_tensor(pn, device="cuda")
        check_sums(vmax[tb, tz, tn].cpu().numpy(), m, f"2-D bench shape {variant} max")
        check_argmax(amax[tb, tz, tn].cpu().numpy(), best, second, gap, m, f"2-D bench shape {variant} argmax")
        assert bool((vmax >= d_x).all())


# ------------------------------------------------------------------------------------------ fused front end
def complex_batch(B, N, seed, n_norm=312500.0):
    """Fourier series whose normalised power is Exp(1) - 1 noise plus a few bright harmonics: F = sqrt(n/2) (g1 + i g2)."""
    rng = np.random.default_rng(seed)
    F = (rng.standard_normal((B, N)) + 1j * rng.standard_normal((B, N))) * np.sqrt(n_norm / 2)
    for b in range(B):
        m = int(rng.integers(20, max(21, N // 40)))
        k = m * np.arange(1, 33)
        k = k[k < N]
        F[b, k] += np.sqrt(n_norm) * (6.0 * 0.9 ** np.arange(k.size)) * np.exp(2j * np.pi * rng.random(k.size))
    return F.astype(np.complex64), np.float32(1.0 / n_norm)


@pytest.mark.parametrize("variant", VARIANTS)
def test_complex_input_whole_batch(hs, ext, oracle, variant):
    """hs_execute_complex against the oracle composition power spectrum (fp32, step by step) -> harmonic sum, and against
    hs_execute on the same x: the kernels that form x themselves must reproduce it bit for bit."""
    for N, B, Hmax in ((20000, 3, 32), (1 << 15, 5, 32), (4100, 2, 8), (2052, 3, 2), (1 << 15, 17, 16)):
        F, scale = complex_batch(B, N, 60 + Hmax)
        x = ext.power_spectrum(F, float(scale))
        d_F = torch.view_as_real(torch.from_numpy(F)).contiguous().cuda()
        d_x = torch.from_numpy(x).cuda()
        for out_mode in ("both", "reduced"):
            plan = hs.hs_plan_create(N, B, Hmax, variant, out_mode)
            got = plan.run_complex(d_F, float(scale))
            plan.device_status()
            ref = oracle.harmonic_sum(x, Hmax, variant)
            what = f"complex {variant}/{out_mode}/N={N}/Hmax={Hmax}"
            compare(plan, got, ref, what, x if out_mode == "both" else None)
            plain = plan.run(d_x)
            torch.cuda.synchronize()
            if variant != "standard":                            # eq. 1's tuned kernels stage x by TMA: the direct family runs instead
                for a, b_ in zip(got, plain):
                    assert (a is None and b_ is None) or torch.equal(a, b_), what + ": differs from hs_execute on the same x"
            plan.hs_destroy()
    g = hs.hs_plan_create_ex(4096, 1, 8, "max", "full", "all", "c2")
    with pytest.raises(hs.HsError) as e:
        g.run_complex(torch.zeros((1, 4096, 2), device="cuda"), 1.0)
    assert e.value.code == hs.HS_ERR_INVALID_ARG


def test_complex_input_every_family(hs, ext, oracle):
    N, B = 1 << 14, 4
    F, scale = complex_batch(B, N, 77)
    x = ext.power_spectrum(F, float(scale))
    d_F = torch.view_as_real(torch.from_numpy(F)).contiguous().cuda()
    for variant in VARIANTS:
        ref = oracle.harmonic_sum(x, 32, variant)
        for algo in ("direct", "tiled", "gather", "grouped", "twophase"):
            plan = hs.hs_plan_create(N, B, 32, variant, "both")
            try:
                plan.set_algo(algo)
            except hs.HsError:
                continue
            compare(plan, plan.run_complex(d_F, float(scale)), ref, f"complex {variant}/{algo}", x)
            plan.device_status()


def test_complex_input_sampled_at_bench_size(hs, ext, oracle):
    """The shape bench.py --workload complex times: 1024 spectra x 2^18 bins from their Fourier series, reduced output."""
    B, N = 1024, 1 << 18
    g = torch.Generator(device="cuda").manual_seed(181202647 + 9)
    d_F = torch.randn((B, N, 2), generator=g, device="cuda") * float(np.sqrt(312500.0 / 2))
    scale = float(np.float32(1.0 / 312500.0))
    rng = np.random.default_rng(78)
    spectra = np.array([0, 1, 500, 1023])
    bidx = np.concatenate([rng.choice(spectra, 1500), rng.choice(spectra, 500)])
    nidx = np.concatenate([rng.integers(0, N, 1500), rng.integers(0, N // 32, 500)])
    x_rows = ext.power_spectrum(d_F[spectra].cpu().numpy(), scale)
    remap = {int(b): i for i, b in enumerate(spectra)}
    tb, tn = torch.as_tensor(bidx, device="cuda"), torch.as_tensor(nidx, device="cuda")
    for variant in VARIANTS:
        plan = hs.hs_plan_create(N, B, 32, variant, "reduced")
        _, vmax, amax = plan.run_complex(d_F, scale)
        plan.device_status()
        h, _ = oracle.points(x_rows, 32, variant, np.array([remap[int(b)] for b in bidx]), nidx)
        best, second, gap, m = argmax_from_levels(h)
        check_sums(vmax[tb, tn].cpu().numpy(), m, f"complex bench shape {variant} max")
        check_argmax(amax[tb, tn].cpu().numpy(), best, second, gap, m, f"complex bench shape {variant} argmax")
