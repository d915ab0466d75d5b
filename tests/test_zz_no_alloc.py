"""hs_execute_static: the entry point for callers that cannot allocate device memory.

Who that is: a real-time search loop that reserved its device memory at start-up and forbids cudaMalloc / cudaFree
afterwards (both synchronise the device, and a late allocation can fail), a plug-in that only ever receives input and
output buffers from its host application, a process whose framework already holds all of the device's memory.  Such a
caller cannot give a plan the workspace the two-phase kernels of eqs. 2-3 need, so the library keeps a fixed scratch
array (HS_STATIC_SCRATCH_BYTES) in its own image and this call uses it.

What is checked here: on the same seeded inputs the call returns what the existing path returns (hs_execute on a
HS_ALGO_TWOPHASE plan with a torch-allocated workspace), within the tolerance of the other parity tests
(CONVENTIONS.md C10) and with identical best levels; twice in a row on DIFFERENT inputs, because the array is shared
and keeps the previous call's contents: a second call that read stale entries would disagree.  Also: the array is not
allocated by the call (the allocator's counters do not move across it), spectra whose arrays exceed the array are
refused with HS_ERR_SCRATCH_LIMIT, and plans the call does not cover are refused.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide another test.  It needs no
state from other tests (the first call on the device does the address look-up itself), so it passes alone in a fresh
process as well as after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import workloads as W
from parity import check_sums

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1812_02647_b200 import build
    build.build()
    import paper_1812_02647_b200.binding as binding
    return binding


def noise(seed, B, N):
    """Exp(1) - 1 noise, about a third of the spectra with an injected comb (the recipe of BASELINE.json configs[2]);
    `seed` selects a disjoint set of spectrum streams."""
    x, _ = W.comb_batch_numpy(2, [1000 * seed + b for b in range(B)], N, 0.3, 50.0, min(5000.0, N / 40.0), 0.10)
    return x


def existing_path(hs, x_np, Hmax, variant, out_mode):
    B, N = x_np.shape
    plan = hs.hs_plan_create(N, B, Hmax, variant, out_mode)
    plan.set_algo("twophase")
    out = plan.run(torch.from_numpy(x_np).cuda())
    plan.device_status()
    plan.hs_destroy()
    return [None if t is None else t.cpu().numpy() for t in out]


def static_path(hs, plan, d_x):
    """Outputs allocated by the CALLER (torch stands in for it), poisoned first: the call must overwrite every element."""
    B, N, L = plan.batch, plan.nbins, plan.levels
    sums = vmax = amax = None
    if plan.out_mode & hs.HS_OUT_FULL:
        sums = torch.full((B, L, N), float("nan"), dtype=torch.float32, device="cuda")
    if plan.out_mode & hs.HS_OUT_REDUCED:
        vmax = torch.full((B, N), float("nan"), dtype=torch.float32, device="cuda")
        amax = torch.full((B, N), 255, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_stats().get("num_device_alloc", 0), torch.cuda.mem_get_info()[0]
    plan.hs_execute_static(d_x, sums, vmax, amax)
    torch.cuda.synchronize()
    after = torch.cuda.memory_stats().get("num_device_alloc", 0), torch.cuda.mem_get_info()[0]
    return [None if t is None else t.cpu().numpy() for t in (sums, vmax, amax)], before, after


def compare(got, ref, what):
    for name, g, r in zip(("sums", "max", "argmax"), got, ref):
        assert (g is None) == (r is None), (what, name)
        if g is None:
            continue
        if name == "argmax":
            assert np.array_equal(g, r), f"{what}: best levels differ in {int((g != r).sum())} bins"
        else:
            check_sums(g, r, f"{what} {name}")


# (variant, Hmax, out_mode, B, N): several 4096-bin tiles and a ragged tail; the last shape has 23 spectra of 2^18 bins,
# of which the 32 MiB array holds 10 at a time: three groups, so the slots are reused INSIDE one call as well
SHAPES = [("max", 32, "both", 5, 3 * 4096 + 1000), ("freqbin", 32, "both", 5, 3 * 4096 + 1000),
          ("max", 8, "reduced", 3, 20000), ("freqbin", 4, "full", 2, 8192), ("max", 1, "both", 2, 4096),
          ("max", 32, "reduced", 23, 1 << 18), ("freqbin", 32, "both", 23, 1 << 18)]


@pytest.mark.parametrize("variant,Hmax,out_mode,B,N", SHAPES)
def test_static_scratch_matches_the_workspace_path_twice_in_a_row(hs, variant, Hmax, out_mode, B, N):
    x1, x2 = noise(11, B, N), noise(12, B, N)
    assert not np.array_equal(x1, x2)
    ref1 = existing_path(hs, x1, Hmax, variant, out_mode)
    ref2 = existing_path(hs, x2, Hmax, variant, out_mode)
    plan = hs.hs_plan_create(N, B, Hmax, variant, out_mode)
    assert plan._ws is None                                     # no workspace is ever set on this plan
    d1, d2 = torch.from_numpy(x1).cuda(), torch.from_numpy(x2).cuda()
    got1, _, _ = static_path(hs, plan, d1)                      # (the very first call may load the module: not measured)
    got2, before, after = static_path(hs, plan, d2)             # second call in a row, same array, other input
    compare(got1, ref1, f"{variant} Hmax {Hmax} {out_mode} {B}x{N} call 1")
    compare(got2, ref2, f"{variant} Hmax {Hmax} {out_mode} {B}x{N} call 2")
    # the call allocated nothing: torch's allocator did not go to the driver and the device's free memory did not drop
    assert after[0] == before[0]
    assert after[1] >= before[1]
    plan.device_status()
    plan.hs_destroy()


def test_static_scratch_refuses_what_does_not_fit(hs):
    limit = hs.lib.hs_static_scratch_bytes()
    assert limit == 32 << 20
    d = torch.zeros(4096, dtype=torch.float32, device="cuda")   # never touched: the call fails before it enqueues
    a = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    # 2^22 bins at Hmax 32: one spectrum's arrays are about 3.06 * 2^22 floats = 51 MB > 32 MiB
    plan = hs.hs_plan_create(1 << 22, 1, 32, "max", "reduced")
    with pytest.raises(hs.HsError) as e:
        plan.hs_execute_static(d, None, d, a)
    assert e.value.code == hs.HS_ERR_SCRATCH_LIMIT
    assert b"HS_STATIC_SCRATCH_BYTES" in hs.lib.hs_error_string(e.value.code)
    plan.hs_destroy()
    # the same length at Hmax 4 (1.08 * 2^22 floats = 18 MB) fits, and so does 2^21 at Hmax 32: accepted by the size check
    # (NULL input: the call gets past the limit and stops at the pointer check)
    for N, Hmax in ((1 << 22, 4), (1 << 21, 32)):
        plan = hs.hs_plan_create(N, 1, Hmax, "freqbin", "reduced")
        with pytest.raises(hs.HsError) as e:
            plan.hs_execute_static(None, None, d, a)
        assert e.value.code == hs.HS_ERR_NULL_POINTER
        plan.hs_destroy()
    # eqs. 1 and 4 have no two-phase kernel, general plans neither
    for make in (lambda: hs.hs_plan_create(4096, 1, 32, "standard", "reduced"),
                 lambda: hs.hs_plan_create(4096, 1, 32, "greedy", "reduced"),
                 lambda: hs.hs_plan_create_ex(4096, 1, 32, "max", "reduced", "all", "c2"),
                 lambda: hs.hs_plan_create_2d(4096, 3, 1, 32, "freqbin", "reduced")):
        plan = make()
        with pytest.raises(hs.HsError) as e:
            plan.hs_execute_static(d, None, d, a)
        assert e.value.code == hs.HS_ERR_INVALID_ARG
        plan.hs_destroy()
