"""Parity of the CUDA path (through the C ABI, include/hs.h) with the oracle, element by element on the same seeded
inputs.  Tolerances are those of BASELINE.json north_star / CONVENTIONS.md C10:
    sums and maxima  |gpu - ref| <= 1e-5 (1 + |ref|);   Greedy j exact;
    best level exact unless the oracle's top two levels differ by less than the tolerance.
"""
import math

import numpy as np
import pytest
import torch

import workloads as W
from parity import check_candidates, argmax_from_levels, check_argmax, check_sums

pytestmark = pytest.mark.gpu

VARIANTS = ["standard", "max", "freqbin", "greedy"]
ALGOS = ["direct", "tiled", "twophase", "gather", "grouped"]


def by_contract(variant, algo, Hmax=32, N=4096):
    """What hs_plan_set_algo accepts by contract (include/hs.h, enum hs_algo): the two-phase families cover eqs. 2-3
    (the grouped one spectra of up to 2^23 bins and Hmax >= 2), the plain gather eqs. 3-4 and eq. 2 up to Hmax = 4.
    Everything else must run: a rejected set_algo is a failure."""
    if algo in ("twophase", "grouped"):
        return variant in ("max", "freqbin") and not (algo == "grouped" and (Hmax < 2 or N > (1 << 23)))
    if algo == "gather":
        return variant in ("freqbin", "greedy") or (variant == "max" and Hmax <= 4)
    return True


# every (variant, family) pair some plan exists for; a pair absent here is rejected by contract for every Hmax
PAIRS = [pytest.param(v, a, id=f"{v}-{a}") for v in VARIANTS for a in ALGOS if any(by_contract(v, a, h) for h in (2, 32))]
FAMILIES = [pytest.param(a, id=a) for a in ALGOS]


@pytest.fixture(scope="module")
def hs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1812_02647_b200 import build
    build.build()
    import paper_1812_02647_b200.binding as binding
    return binding


def make_plan(hs, N, B, Hmax, variant, out_mode, algo):
    """The plan, or None where the contract says the family does not cover (variant, Hmax): callers `continue`.
    Never skips: a test that loops over shapes or variants must run every combination the family supports."""
    plan = hs.hs_plan_create(N, B, Hmax, variant, out_mode)
    if not by_contract(variant, algo, Hmax, N):
        with pytest.raises(hs.HsError):
            plan.set_algo(algo)
        return None
    plan.set_algo(algo)
    return plan


def run_and_compare(hs, oracle, x_np, Hmax, variant, out_mode, algo, check_j=True):
    """Run the whole batch on the GPU and compare every element with the oracle."""
    B, N = x_np.shape
    d_x = torch.from_numpy(x_np).cuda()
    plan = make_plan(hs, N, B, Hmax, variant, out_mode, algo)
    if plan is None:
        return 0
    sums, vmax, amax = plan.run(d_x)
    plan.device_status()                                                             # synchronises; no wait timed out
    ref = oracle.harmonic_sum(x_np, Hmax, variant, want_jpath=(variant == "greedy"))
    what = f"{variant}/{algo}/{out_mode}/N={N}/B={B}/Hmax={Hmax}"
    if sums is not None:
        check_sums(sums.cpu().numpy(), ref["sums"], what + " sums")
        np.testing.assert_array_equal(sums[:, 0].cpu().numpy(), x_np)               # h_1(n) = x(n) bit-exactly
    if vmax is not None:
        check_sums(vmax.cpu().numpy(), ref["max"], what + " max")
        check_argmax(amax.cpu().numpy(), ref["argmax"], ref["second"], ref["gap"], ref["max"], what + " argmax")
    if sums is not None and vmax is not None:                                        # P13: max is one of the planes
        pick = torch.gather(sums, 1, amax.long().unsqueeze(1)).squeeze(1)
        assert torch.equal(pick, vmax), what + " max != sums[argmax]"
    if variant == "greedy" and check_j:
        d_j = torch.empty((B, plan.levels, N), dtype=torch.uint8, device="cuda")
        plan.hs_debug_greedy_paths(d_x, d_j)                      # the plan's own kernel family and launch shape
        plan.device_status()
        np.testing.assert_array_equal(d_j.cpu().numpy(), ref["jpath"])
    plan.hs_destroy()
    return 1


# ---------------------------------------------------------------------------------------------------- small and ragged
@pytest.mark.parametrize("variant,algo", PAIRS)
def test_small_and_ragged_sizes(hs, oracle, variant, algo):
    rng = np.random.default_rng(1)
    ran = 0
    for Hmax in (32, 4):
        for N, B in ((4, 1), (8, 3), (12, 1), (36, 2), (100, 1), (1000, 3), (4100, 2), (33000, 1), (2052, 37)):
            x = (rng.standard_exponential((B, N)) - 1).astype(np.float32)
            ran += run_and_compare(hs, oracle, x, Hmax, variant, "both", algo)
    assert ran >= 9


@pytest.mark.parametrize("variant,algo", PAIRS)
def test_every_hmax_and_out_mode(hs, oracle, variant, algo):
    rng = np.random.default_rng(2)
    x = rng.standard_normal((2, 20000)).astype(np.float32)
    ran = 0
    for Hmax in (1, 2, 4, 8, 16, 32):
        for out_mode in ("full", "reduced", "both"):
            ran += run_and_compare(hs, oracle, x, Hmax, variant, out_mode, algo, check_j=(out_mode == "full"))
    assert ran == 3 * sum(by_contract(variant, algo, h) for h in (1, 2, 4, 8, 16, 32)) > 0


@pytest.mark.parametrize("variant,algo", PAIRS)
def test_reduced_hmax32_whole_batch_across_tiles_and_spectra(hs, oracle, variant, algo):
    """The headline mode (Hmax 32, reduced output) compared element by element on whole batches whose spectra are made
    of whole 4096-bin tiles: the shape that takes eq. 1's register-blocked kernel (hs_standard_rb.cu) and the persistent
    ring kernels of eqs. 2-4.  64 x 2^15 bins = 512 tiles, more than the resident CTAs, so tiles are handed over
    between CTAs and the ring runs across spectrum boundaries (PAPER.md:17 eq. 1, :33, :38, :43)."""
    if not by_contract(variant, algo, 32):
        pytest.skip("the family does not cover this variant at Hmax = 32 (include/hs.h, enum hs_algo)")
    for N in (4096, 8192, 1 << 15):
        for B in (1, 5, 64):
            x, _ = W.comb_batch_numpy(2, list(range(B)), N, 0.25, 50.0, float(N // 40), 0.10)
            assert run_and_compare(hs, oracle, x, 32, variant, "reduced", algo, check_j=(B == 5)) == 1


@pytest.mark.parametrize("variant,algo", PAIRS)
def test_degenerate_spectra(hs, oracle, variant, algo):
    ran = 0
    for N, Hmax in ((6000, 32), (8192, 32), (6000, 4)):
        rng = np.random.default_rng(3)
        cases = [np.zeros(N), -np.ones(N), np.ones(N), np.arange(N), np.arange(N)[::-1],
                 rng.integers(-2, 3, N), np.where(np.arange(N) % 7 == 0, 5.0, -1.0)]
        x = np.stack(cases).astype(np.float32)
        ran += run_and_compare(hs, oracle, x, Hmax, variant, "both", algo)
        ran += run_and_compare(hs, oracle, x, Hmax, variant, "reduced", algo)
        # all levels tie on the zero spectrum: the smallest level wins (C8)
        plan = make_plan(hs, N, 1, Hmax, variant, "reduced", algo)
        if plan is None:
            continue
        _, vmax, amax = plan.run(torch.zeros((1, N), device="cuda"))
        assert int(amax.max()) == 0 and float(vmax.abs().max()) == 0.0
    assert ran >= 2


@pytest.mark.parametrize("algo", FAMILIES)
def test_integer_bin_comb_all_variants_agree(hs, algo):
    N, m = 1 << 16, 1251
    a = (10.0 * 0.9 ** np.arange(32) + 0.5).astype(np.float32)
    x = np.zeros((1, N), np.float32)
    x[0, m * np.arange(1, 33)] = a
    d_x = torch.from_numpy(x).cuda()
    vals = {}
    for v in VARIANTS:
        plan = make_plan(hs, N, 1, 32, v, "full", algo)
        if plan is None:
            continue
        sums, _, _ = plan.run(d_x)
        plan.device_status()
        vals[v] = sums[0].cpu().numpy()
    assert vals
    for l, H in enumerate((1, 2, 4, 8, 16, 32)):
        ref = float(np.cumsum(a.astype(np.float64))[H - 1] / math.sqrt(H))
        for v in vals:
            assert vals[v][l, H * m if v == "standard" else m] == pytest.approx(ref, rel=1e-5)


# ---------------------------------------------------------------------------------------------------- configs 0 and 1
@pytest.mark.parametrize("variant,algo", PAIRS)
def test_config0_full_output(hs, oracle, variant, algo):
    if not by_contract(variant, algo, 32):
        pytest.skip("the family does not cover this variant at Hmax = 32 (include/hs.h, enum hs_algo)")
    assert run_and_compare(hs, oracle, W.config0(), 32, variant, "full", algo) == 1


@pytest.mark.parametrize("variant,algo", PAIRS)
def test_config1_subset_full_and_reduced(hs, oracle, variant, algo):
    if not by_contract(variant, algo, 32):
        pytest.skip("the family does not cover this variant at Hmax = 32 (include/hs.h, enum hs_algo)")
    flags = [W.rng_for(1, b).random() < 0.10 for b in range(256)]
    chosen = [b for b in range(256) if flags[b]][:2] + [0, 255]
    x, _ = W.config1(chosen)
    assert run_and_compare(hs, oracle, x, 32, variant, "both", algo, check_j=False) == 1
    assert run_and_compare(hs, oracle, x, 32, variant, "reduced", algo, check_j=True) == 1


# ---------------------------------------------------------------------------------------------------- full-size configs
def sampled_compare(hs, oracle, d_x, variant, out_mode, algo, spectra, npoints, seed, Hmax=32, check_j=True):
    """At sizes the oracle cannot cover: launch on the whole batch exactly as bench.py does, then compare sampled
    outputs (whole rows of a few spectra's low bins plus random points) computed one by one by the oracle."""
    B, N = d_x.shape
    plan = make_plan(hs, N, B, Hmax, variant, out_mode, algo)
    if plan is None:
        return 0
    sums, vmax, amax = plan.run(d_x)
    plan.device_status()
    rng = np.random.default_rng(seed)
    bidx = np.concatenate([rng.choice(spectra, npoints), np.repeat(spectra[:4], 64)])
    nidx = np.concatenate([rng.integers(0, N, npoints), np.tile(np.arange(64), len(spectra[:4]))])
    # low bins (all 32 harmonics in range) are a tiny fraction of uniform samples: add some explicitly
    extra = npoints // 4
    bidx = np.concatenate([bidx, rng.choice(spectra, extra)])
    nidx = np.concatenate([nidx, rng.integers(0, N // 32, extra)])
    rows = sorted(set(int(b) for b in bidx))
    x_rows = d_x[rows].cpu().numpy()
    remap = {b: i for i, b in enumerate(rows)}
    h, jref = oracle.points(x_rows, Hmax, variant, np.array([remap[int(b)] for b in bidx]), nidx)
    tb, tn = torch.as_tensor(bidx, device="cuda"), torch.as_tensor(nidx, device="cuda")
    what = f"{variant}/{algo}/{out_mode} sampled B={B} N={N}"
    if sums is not None:
        check_sums(sums[tb, :, tn].cpu().numpy(), h, what + " sums")
    if vmax is not None:
        best, second, gap, m = argmax_from_levels(h)
        check_sums(vmax[tb, tn].cpu().numpy(), m, what + " max")
        check_argmax(amax[tb, tn].cpu().numpy(), best, second, gap, m, what + " argmax")
        assert int(amax.max()) <= plan.levels - 1
    # properties that hold at any size: h_1 = x, and the reduced maximum is at least x
    if sums is not None:
        assert torch.equal(sums[:, 0], d_x)
    if vmax is not None:
        assert bool((vmax >= d_x).all())
    del sums, vmax, amax
    torch.cuda.empty_cache()
    if variant == "greedy" and check_j:                              # Greedy j of the same launch shape, sampled
        d_j = torch.empty((B, plan.levels, N), dtype=torch.uint8, device="cuda")
        plan.hs_debug_greedy_paths(d_x, d_j)
        plan.device_status()
        np.testing.assert_array_equal(d_j[tb, :, tn].cpu().numpy(), jref)
        del d_j
        torch.cuda.empty_cache()
    plan.hs_destroy()
    return 1


def _variants_of(algo, Hmax=32, N=4096):
    return [v for v in VARIANTS if by_contract(v, algo, Hmax, N)]


@pytest.mark.parametrize("algo", FAMILIES)
def test_config2_full_size_reduced_sampled(hs, oracle, algo):
    d_x, injected = W.config2_torch("cuda")
    assert d_x.shape == (4096, 1 << 18) and 20 <= len(injected) <= 70
    spectra = np.array(sorted(set(injected[:12] + [0, 4095] + list(range(64, 4096, 512)))))
    for v in _variants_of(algo):
        assert sampled_compare(hs, oracle, d_x, v, "reduced", algo, spectra, 4000, 22) == 1


@pytest.mark.timeout(900, method="thread")
def test_config1_shape_full_and_reduced_output_repeated_launches(hs, oracle):
    """configs[1]'s shape in bench's launch configuration (256 x 2^18, full + reduced output).  With both outputs the
    warps of a CTA of the interleaved kernel (eq. 3) progress at very different speeds: the launch that once hung when
    item completion was a running sum over the warps.  Five launches per variant, the last one compared with the oracle."""
    d_x = W.exp_noise_torch(256, 1 << 18, 6, "cuda")
    for v in VARIANTS:
        plan = make_plan(hs, 1 << 18, 256, 32, v, "both", "tiled")
        for _ in range(4):
            plan.run(d_x)
        plan.device_status()
        plan.hs_destroy()
        assert sampled_compare(hs, oracle, d_x, v, "both", "tiled", np.arange(0, 256, 37), 1500, 55) == 1


@pytest.mark.parametrize("algo", FAMILIES)
def test_config3_long_spectra_full_output_sampled(hs, oracle, algo):
    d_x, injected = W.config3_torch("cuda")
    assert d_x.shape == (8, 1 << 23) and len(injected) == 8
    for v in _variants_of(algo):
        assert sampled_compare(hs, oracle, d_x, v, "full", algo, np.arange(8), 3000, 33) == 1


@pytest.mark.parametrize("algo", FAMILIES)
def test_scaling_shapes_short_and_long_spectra(hs, oracle, algo):
    # configs[4] scaling sweep shapes, shrunk in batch: 2^16-bin and 2^24-bin spectra, Hmax 32 and 4
    for N, B in ((1 << 16, 64), (1 << 19, 40), (1 << 24, 2)):       # (2^19: the longest spectra the interleaved kernel takes)
        d_x = W.exp_noise_torch(B, N, 4, "cuda")
        for Hmax in (32, 4):
            for v in _variants_of(algo, Hmax, N):
                assert sampled_compare(hs, oracle, d_x, v, "reduced", algo, np.arange(min(B, 8)), 1500, 44, Hmax=Hmax) == 1


@pytest.mark.parametrize("algo", FAMILIES)
def test_scaling_sweep_every_hmax_with_slot_reuse(hs, oracle, algo):
    """`bench.py --sweep scaling` also times Hmax 2, 8 and 16 (configs[4]).  The grouped kernel of eq. 2 keeps a different
    set of per-harmonic arrays at Hmax 8 and 16 than at 32; 160 spectra of 2^18 bins give each of its groups several
    spectra in a row, so every workspace slot is refilled while neighbouring groups still read theirs."""
    N, B = 1 << 18, 160
    d_x = W.exp_noise_torch(B, N, 8, "cuda")
    W.inject_combs_torch(d_x, 2, 0.05, 50.0, 5000.0, 0.10)
    ran = 0
    for Hmax in (2, 8, 16):
        for v in _variants_of(algo, Hmax, N):
            ran += sampled_compare(hs, oracle, d_x, v, "reduced", algo, np.array([0, 1, 17, 18, 19, 77, 158, 159]), 1500, 66,
                                   Hmax=Hmax, check_j=(Hmax == 16))
    assert ran >= 3


@pytest.mark.timeout(900, method="thread")
def test_interleaved_kernel_soak_identical_outputs_over_many_launches(hs):
    """The interleaved ring kernel of eq. 3 hands items between a scheduler warp and the worker warps and between CTAs
    through counters; a hand-over bug shows up once in tens of launches (it did: 128 x 2^18 with both outputs once hung).
    40 launches per output mode on that shape, on 2^16-bin spectra (several groups per ring step) and on 2^19-bin spectra
    (two big slots): no wait may time out and every launch must reproduce the first one bit for bit."""
    for B, N in ((128, 1 << 18), (512, 1 << 16), (48, 1 << 19)):
        d_x = W.exp_noise_torch(B, N, 10, "cuda")
        for out_mode in ("both", "reduced"):
            plan = make_plan(hs, N, B, 32, "freqbin", out_mode, "tiled")
            first = plan.run(d_x)
            plan.device_status()
            for it in range(40):
                again = plan.run(d_x)
                if it % 8 == 7:
                    plan.device_status()
                    for a, b in zip(first, again):
                        assert (a is None and b is None) or torch.equal(a, b), f"launch {it + 2} differs ({B}x{N}, {out_mode})"
                del again
            plan.hs_destroy()
            del first
        del d_x
        torch.cuda.empty_cache()


@pytest.mark.parametrize("algo", [pytest.param("tiled", id="tiled"), pytest.param("direct", id="direct")])
def test_scaling_point_with_2_to_32_input_elements(hs, oracle, algo):
    """configs[4]'s largest-offset point: 65536 spectra x 2^16 bins = 2^32 input elements (16 GiB), reduced output, as
    `bench.py --sweep scaling` times it.  Element offsets b N + n pass 2^31 and 2^32: the sampled spectra include the
    last ones of the batch (offsets just below 2^32) and the ones around the 2^31 boundary."""
    B, N = 65536, 1 << 16
    free, _ = torch.cuda.mem_get_info()
    if free < 44 * (1 << 30):
        pytest.skip("needs 44 GiB of free device memory")
    d_x = W.exp_noise_torch(1, B * N, 4, "cuda").view(B, N)
    spectra = np.array([0, 1, 32766, 32767, 32768, 32769, 49151, 65534, 65535])
    for v in VARIANTS:
        assert sampled_compare(hs, oracle, d_x, v, "reduced", algo, spectra, 2500, 55, check_j=False) == 1
    del d_x
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------------------------- ABI behaviour on the device
def test_error_paths_on_device(hs):
    plan = hs.hs_plan_create(1024, 2, 32, "max", "both")
    x = torch.zeros((2, 1024), device="cuda")
    sums = torch.empty((2, 6, 1024), device="cuda")
    vmax = torch.empty((2, 1024), device="cuda")
    amax = torch.empty((2, 1024), dtype=torch.uint8, device="cuda")
    plan.ensure_workspace()
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute(x, None, vmax, amax)
    assert e.value.code == hs.HS_ERR_NULL_POINTER
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute(x, sums, vmax, None)
    assert e.value.code == hs.HS_ERR_NULL_POINTER
    off = torch.zeros(2 * 1024 + 1, device="cuda")[1:].view(2, 1024)
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute(off, sums, vmax, amax)
    assert e.value.code == hs.HS_ERR_MISALIGNED
    plan.hs_execute(x, sums, vmax, amax)
    torch.cuda.synchronize()
    g = hs.hs_plan_create(1024, 2, 32, "standard", "full")
    with pytest.raises(hs.HsError) as e:
        g.hs_debug_greedy_paths(x, amax)
    assert e.value.code == hs.HS_ERR_INVALID_ARG
    assert plan.launches() >= 1 and plan.levels == 6
    with pytest.raises(hs.HsError):
        plan.set_algo(8)
    with pytest.raises(hs.HsError):
        g.set_algo("twophase")            # eq. 1 has no two-phase kernel
    assert plan.device_status() == hs.HS_OK
    with pytest.raises(hs.HsError) as e:
        hs.hs_plan_create(4, 1 << 31, 2, "max", "full")           # spectrum indices are int32
    assert e.value.code == hs.HS_ERR_INVALID_ARG


def test_host_staging_must_be_set_again_after_set_algo(hs):
    """staging sized for one algorithm must not be used by another (the workspace per slab differs)."""
    B, N = 6, 1 << 14
    plan = hs.hs_plan_create(N, B, 32, "max", "reduced")
    plan.set_algo("direct")
    st = torch.empty(plan.host_staging_bytes(2), dtype=torch.uint8, device="cuda")
    plan.set_host_staging(st, 2)
    plan.set_algo("tiled")                                             # needs a workspace per slab: staging is invalidated
    h_x = torch.zeros((B, N)).pin_memory()
    h_max = torch.empty((B, N)).pin_memory()
    h_amax = torch.empty((B, N), dtype=torch.uint8).pin_memory()
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute_host(h_x, None, h_max, h_amax)
    assert e.value.code == hs.HS_ERR_WORKSPACE
    st2 = torch.empty(plan.host_staging_bytes(2), dtype=torch.uint8, device="cuda")
    plan.set_host_staging(st2, 2)
    plan.hs_execute_host(h_x, None, h_max, h_amax)
    assert plan.device_status() == hs.HS_OK and float(h_max.abs().max()) == 0.0


def test_a_timed_out_wait_is_reported_by_device_status():
    """A persistent kernel that gives up a wait sets the error word; hs_plan_device_status turns it into
    HS_ERR_DEVICE_TIMEOUT.  Forced in the tuning build (libhs_tuning.so, -DHS_TUNING) with a spin limit of 0 in a
    subprocess: the product library reads no environment variable."""
    import os
    import subprocess
    import sys
    from paper_1812_02647_b200 import build
    build.build(tuning=True)
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = (
        "import torch, paper_1812_02647_b200 as pkg\n"
        "pkg.LIBRARY = 'libhs_tuning.so'\n"
        "import paper_1812_02647_b200.binding as hs\n"
        "assert hs.LIB_PATH.endswith('libhs_tuning.so')\n"
        "x = torch.randn(64, 1 << 15, device='cuda')\n"
        "bad = 0\n"
        "for v in ('max', 'freqbin', 'greedy'):\n"
        "    p = hs.hs_plan_create(1 << 15, 64, 32, v, 'reduced')\n"
        "    if p.workspace_bytes() == 0: continue\n"
        "    p.run(x)\n"
        "    try:\n"
        "        p.device_status()\n"
        "    except hs.HsError as e:\n"
        "        assert e.code == hs.HS_ERR_DEVICE_TIMEOUT\n"
        "        bad += 1\n"
        "print('TIMEOUTS', bad)\n")
    env = dict(os.environ, HS_SPIN_LIMIT="0", PYTHONPATH=root)        # (only the tuning build reads HS_SPIN_LIMIT)
    out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    assert int(out.stdout.split("TIMEOUTS")[1]) >= 1, out.stdout
    env["HS_SPIN_LIMIT"] = str(1 << 23)                                # the default limit: nothing times out
    out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and int(out.stdout.split("TIMEOUTS")[1]) == 0, out.stdout + out.stderr[-2000:]


@pytest.mark.parametrize("variant", VARIANTS)
def test_workspace_is_required_when_the_algorithm_needs_one(hs, variant):
    plan = hs.hs_plan_create(1 << 14, 4, 32, variant, "reduced")
    if plan.workspace_bytes() == 0:
        return
    x = torch.zeros((4, 1 << 14), device="cuda")
    vmax = torch.empty((4, 1 << 14), device="cuda")
    amax = torch.empty((4, 1 << 14), dtype=torch.uint8, device="cuda")
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute(x, None, vmax, amax)
    assert e.value.code == hs.HS_ERR_WORKSPACE
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(hs.HsError) as e:
        plan.set_workspace(small)
    assert e.value.code == hs.HS_ERR_WORKSPACE


@pytest.mark.parametrize("variant", VARIANTS)
def test_non_default_stream_and_repeat_calls(hs, oracle, variant):
    rng = np.random.default_rng(9)
    x = (rng.standard_exponential((5, 50000)) - 1).astype(np.float32)
    d_x = torch.from_numpy(x).cuda()
    plan = hs.hs_plan_create(50000, 5, 32, variant, "reduced")
    plan.ensure_workspace()
    vmax = torch.empty((5, 50000), device="cuda")
    amax = torch.empty((5, 50000), dtype=torch.uint8, device="cuda")
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        for _ in range(3):                                   # the workspace is reused across calls
            vmax.fill_(float("nan"))
            plan.hs_execute(d_x, None, vmax, amax, stream=s)
    assert plan.device_status(stream=s) == hs.HS_OK          # synchronises s
    ref = oracle.harmonic_sum(x, 32, variant, want_sums=False)
    check_sums(vmax.cpu().numpy(), ref["max"], variant + " stream max")
    check_argmax(amax.cpu().numpy(), ref["argmax"], ref["second"], ref["gap"], ref["max"], variant + " stream argmax")


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("out_mode", ["reduced", "both"])
def test_host_buffer_entry_matches_device_entry(hs, variant, out_mode):
    B, N, slab = 11, 1 << 15, 4                               # ragged last slab, more slabs than lanes
    x = W.exp_noise_torch(B, N, 5, "cpu").pin_memory()
    plan = hs.hs_plan_create(N, B, 32, variant, out_mode)
    sums_d, vmax_d, amax_d = plan.run(x.cuda())
    staging = torch.empty(plan.host_staging_bytes(slab), dtype=torch.uint8, device="cuda")
    plan.set_host_staging(staging, slab)
    h_sums = torch.empty((B, 6, N), dtype=torch.float32).pin_memory() if out_mode == "both" else None
    h_max = torch.empty((B, N), dtype=torch.float32).pin_memory()
    h_amax = torch.empty((B, N), dtype=torch.uint8).pin_memory()
    plan.hs_execute_host(x, h_sums, h_max, h_amax)
    assert plan.device_status() == hs.HS_OK
    assert torch.equal(h_max, vmax_d.cpu()) and torch.equal(h_amax, amax_d.cpu())
    if h_sums is not None:
        assert torch.equal(h_sums, sums_d.cpu())


def test_sensitivity_sweep_small_instance(hs):
    """configs[4] sensitivity harness on 24 realisations: on a Fourier bin freq-bin recovers what the standard sum does,
    half a bin off it loses clearly more than Max HRMS does."""
    from paper_1812_02647_b200 import sensitivity
    res = sensitivity.run(realisations=24, snr=8.0, deltas=[0.0, 0.5], duties=[0.02])
    on, off = res["points"]
    assert on["delta"] == 0.0 and off["delta"] == 0.5
    assert abs(on["snr"]["freqbin"] / on["snr"]["standard"] - 1.0) < 0.1
    assert off["snr"]["freqbin"] < 0.75 * on["snr"]["freqbin"]
    assert off["snr"]["max"] > 0.8 * on["snr"]["max"]
    for p in (on, off):
        assert p["snr"]["standard"] >= p["snr"]["max"] - 0.5


# ---------------------------------------------------------------------------------------------------- candidates (fused back end)
def _records(rec):
    return {k: v.cpu().numpy() for k, v in rec.items()}


@pytest.mark.parametrize("variant,algo", PAIRS)
def test_candidates_match_the_oracle(hs, oracle, variant, algo):
    """hs_execute_candidates against oracle.candidates on noise + combs: several tiles, ragged tail, both halves of the
    spectrum (bins >= N/2 are emitted by other code than the bins below), thresholds from 'a few' to 'thousands'."""
    ran = 0
    for N, B, Hmax in ((20000, 3, 32), (1 << 15, 5, 32), (4100, 2, 8), (4100, 2, 4)):
        x, _ = W.comb_batch_numpy(2, list(range(B)), N, 1.0, 50.0, 500.0, 0.10)
        d_x = torch.from_numpy(x).cuda()
        plan = make_plan(hs, N, B, Hmax, variant, "reduced", algo)
        if plan is None:
            continue
        for thr in (2.5, 6.0, 40.0):
            ref = oracle.candidates(x, Hmax, variant, thr)
            count, rec = plan.run_candidates(d_x, thr, capacity=B * N)
            check_candidates(count, _records(rec), ref, (B, N), f"{variant}/{algo}/N={N}/thr={thr}")
            assert plan.device_status() == hs.HS_OK
        plan.hs_destroy()
        ran += 1
    assert ran >= 1


def test_candidates_at_the_bench_size(hs, oracle):
    """hs_execute_candidates on configs[2]'s full shape (4096 x 2^18, the launch bench.py times): the count equals the
    number of bins of the plan's own reduced maximum above the threshold (another instantiation of the same kernel: a
    whole-batch property), and the records of a few spectra, injected ones included, are the oracle's candidates."""
    d_x, injected = W.config2_torch("cuda")
    B, N = d_x.shape
    chosen = np.array(sorted(set(list(injected[:3]) + [0, 4095])))
    x_rows = d_x[chosen].cpu().numpy()
    for v in VARIANTS:
        # eq. 2 sums block maxima: on noise alone its h_32 sits near 12.4 at the bins whose 32 harmonics are all in range
        thr = 22.0 if v == "max" else 12.0
        plan = make_plan(hs, N, B, 32, v, "reduced", "tiled")
        _, vmax, _ = plan.run(d_x)
        plan.device_status()
        expected = int((vmax > thr).sum().item())
        del vmax
        count, rec = plan.run_candidates(d_x, thr, capacity=1 << 22)
        plan.device_status()
        assert count == expected and 0 < count <= (1 << 22), (v, count, expected)
        rec = _records(rec)
        keep = np.isin(rec["spectrum"], chosen)
        sel = {k: a[keep] for k, a in rec.items()}
        sel["spectrum"] = np.searchsorted(chosen, sel["spectrum"])
        ref = oracle.candidates(x_rows, 32, v, thr)
        check_candidates(int(keep.sum()), sel, ref, (len(chosen), N), f"{v} candidates at 4096 x 2^18")
        assert v == "max" or len(ref["spectrum"]) > 0
        plan.hs_destroy()
    del d_x
    torch.cuda.empty_cache()


def test_candidates_capacity_count_and_errors(hs, oracle):
    N, B = 1 << 14, 4
    x, _ = W.comb_batch_numpy(2, list(range(B)), N, 1.0, 50.0, 500.0, 0.10)
    d_x = torch.from_numpy(x).cuda()
    plan = hs.hs_plan_create(N, B, 32, "freqbin", "reduced")
    ref = oracle.candidates(x, 32, "freqbin", 3.0)
    total = ref["spectrum"].shape[0]
    assert total > 100
    count, rec = plan.run_candidates(d_x, 3.0, capacity=64)          # more candidates than room: count is the total
    assert abs(count - total) <= 2 and rec["bin"].shape[0] == 64
    count0, _ = plan.run_candidates(d_x, 3.0, capacity=0)
    assert abs(count0 - total) <= 2
    count_none, rec_none = plan.run_candidates(d_x, 1e30, capacity=16)
    assert count_none == 0 and rec_none["bin"].shape[0] == 0
    full = hs.hs_plan_create(N, B, 32, "freqbin", "full")
    with pytest.raises(hs.HsError) as e:
        full.run_candidates(d_x, 3.0)
    assert e.value.code == hs.HS_ERR_INVALID_ARG


# ---------------------------------------------------------------------------------------------------- guard bands
@pytest.mark.parametrize("variant,algo", PAIRS)
def test_no_writes_outside_the_output_and_workspace_buffers(hs, variant, algo):
    """Every output and the workspace sit between canary bands inside one allocation; after hs_execute (both output
    modes at once) and hs_execute_candidates the bands are untouched.  (compute-sanitizer is not available on the box.)"""
    G = 4096                                                      # guard elements on either side
    Hmax = 32 if by_contract(variant, algo, 32) else 4
    for N, B in ((20000, 3), (1 << 15, 5), (4100, 2)):
        x = (torch.empty((B, N), device="cuda").exponential_() - 1)
        for out_mode in ("both", "reduced"):
            plan = make_plan(hs, N, B, Hmax, variant, out_mode, algo)
            assert plan is not None
            L = plan.levels

            def guarded(nelem, dtype, fill):
                buf = torch.full((nelem + 2 * G,), fill, dtype=dtype, device="cuda")
                return buf, buf[G:G + nelem]

            sums_all, sums = guarded(B * L * N, torch.float32, -777.0)
            vmax_all, vmax = guarded(B * N, torch.float32, -777.0)
            amax_all, amax = guarded(B * N, torch.uint8, 0xAB)
            ws_bytes = plan.workspace_bytes()
            ws_all, ws = guarded(max(ws_bytes, 256), torch.uint8, 0xCD)
            assert ws.data_ptr() % 256 == 0                       # (torch allocations are 512-byte aligned, G = 4096)
            if ws_bytes:
                plan.set_workspace(ws)
            plan.hs_execute(x, sums.view(B, L, N) if out_mode == "both" else None, vmax.view(B, N), amax.view(B, N))
            if out_mode == "reduced":
                cand = torch.full((64 + 2 * G, 4), -5, dtype=torch.int32, device="cuda")
                count = torch.zeros(1, dtype=torch.int64, device="cuda")
                plan.hs_execute_candidates(x, 1.5, cand[G:G + 64], 64, count)
            torch.cuda.synchronize()
            what = f"{variant}/{algo}/{out_mode}/N={N}"
            for name, whole, fill in (("sums", sums_all, -777.0), ("max", vmax_all, -777.0), ("argmax", amax_all, 0xAB),
                                      ("workspace", ws_all, 0xCD)):
                assert bool((whole[:G] == fill).all()) and bool((whole[-G:] == fill).all()), f"{what}: wrote outside {name}"
            if out_mode == "reduced":
                assert bool((cand[:G] == -5).all()) and bool((cand[G + 64:] == -5).all()), f"{what}: wrote outside the records"
                assert int(count.item()) > 64                     # (more candidates than room: the rest must be dropped)
            else:
                assert bool((sums != -777.0).all()), f"{what}: a plane element was not written"
            assert bool((vmax != -777.0).all()), f"{what}: a max element was not written"
            plan.hs_destroy()
