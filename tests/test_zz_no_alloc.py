"""fitrig_choose_accumulate_static: the accumulation rule for callers that must not allocate device memory.

Why the entry point exists: `fitrig_choose_accumulate` allocates and frees its scratch with cudaMalloc / cudaFree on
every call.  A real-time loop cannot afford that (cudaFree waits for the whole device to go idle, which ends the
overlap of the next snapshot's copy with the running kernels), and a process whose device memory is already held by
another allocator (a framework's caching pool that took the whole card, a fixed memory budget) may not get the
allocation at all.  The static variant keeps its scratch in a fixed array inside the library instead and must give
the same answer.

What is checked: on two calls in a row -- different stacks, different numbers of levels, so the second call finds the
first call's partial sums and decision record still in the array -- the static entry point returns what the allocating
path returns (same kernels, same grid, same order of summation: the contrasts are compared for equality, which is
inside the 4e-6 relative band tests/test_parity_gpu_r2b.py allows against the oracle), and that the device's free
memory does not move across the calls.

The file is named so that pytest collects it after every other test file: with `pytest -x` a failure here cannot hide
another test.  It does not depend on that order: it passes alone in a fresh process (where its first call is the one
that does the per-device set-up) and after the rest of the suite.
"""
import pytest
import torch

import paper_2509_21754_b200 as fitrig
import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _drifting_stack(L, H, W, seed):
    base = synth.gaussian_noise_stack(L, H, W, seed=seed, device=DEV)
    drift = torch.arange(L, dtype=torch.float32, device=DEV)[:, None, None] * 0.02
    return (5.0 + 0.05 * base + drift).contiguous()  # contrast grows with the group size


def test_static_scratch_matches_allocating_path_on_two_calls_in_a_row():
    first = _drifting_stack(64, 40, 64, seed=31)     # five levels (g = 1 .. 16), 10 blocks
    second = _drifting_stack(17, 333, 500, seed=32)  # three levels (g = 1, 2, 4), 651 blocks: overwrites more, decides less
    expected_first = fitrig.choose_accumulate(first, 1e30)
    expected_second = fitrig.choose_accumulate(second, 1e30)
    assert len(expected_first[1]) == 5 and len(expected_second[1]) == 3
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(0)
    got_first = fitrig.choose_accumulate_static(first, 1e30)
    got_second = fitrig.choose_accumulate_static(second, 1e30)
    free_after, _ = torch.cuda.mem_get_info(0)
    assert got_first == expected_first
    assert got_second == expected_second
    assert free_after == free_before
    # a threshold between two levels: the decision itself, again back to back and in the other order
    lo, hi = expected_second[1][1], expected_second[1][2]
    assert hi > lo
    eps = 0.5 * (lo + hi)
    assert fitrig.choose_accumulate_static(second, eps) == fitrig.choose_accumulate(second, eps)
    assert fitrig.choose_accumulate_static(first, eps) == fitrig.choose_accumulate(first, eps)


def test_static_scratch_on_a_side_stream_and_with_stale_contents():
    # identical snapshots have zero contrast at every level: anything left over from the calls above would show
    flat = torch.full((12, 16, 16), 2.5, device=DEV)
    side = torch.cuda.Stream(device=DEV)
    torch.cuda.synchronize()
    assert fitrig.choose_accumulate_static(flat, 1e-6, stream=side) == (4, [0.0, 0.0, 0.0])
    busy = _drifting_stack(24, 96, 128, seed=33)
    assert fitrig.choose_accumulate_static(busy, 1e30, g_max=2) == fitrig.choose_accumulate(busy, 1e30, g_max=2)
    assert fitrig.choose_accumulate_static(flat, 1e-6) == (4, [0.0, 0.0, 0.0])


def test_static_scratch_rejects_what_the_allocating_path_rejects():
    st = torch.zeros((6, 8, 8), device=DEV)
    with pytest.raises(fitrig.FitrigError):
        fitrig.choose_accumulate_static(st[:2].contiguous(), 0.1)  # fewer than three snapshots
    with pytest.raises(fitrig.FitrigError):
        fitrig.choose_accumulate_static(st, float("nan"))
    assert fitrig.choose_accumulate_static(st, 0.5) == (2, [0.0, 0.0])  # and an error leaves the scratch usable


def test_static_scratch_holds_the_largest_request_of_this_device():
    # the stated limit: levels * min(ceil(H * W / 256), 8 * SMs) partial sums; all six levels on a full grid
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    if 6 * 8 * sms > fitrig.binding.STATIC_ACCUM_MAX_PARTIALS:
        st = torch.zeros((96, 8 * sms, 256), device=DEV)
        with pytest.raises(fitrig.FitrigError, match="partial sums"):
            fitrig.choose_accumulate_static(st, 1e30)
        return
    L, H, W = 96, 640, 512  # 1280 blocks of 256 pixels >= 8 * 148
    st = _drifting_stack(L, H, W, seed=34)
    expected = fitrig.choose_accumulate(st, 1e30)
    assert len(expected[1]) == 6
    assert fitrig.choose_accumulate_static(st, 1e30) == expected
