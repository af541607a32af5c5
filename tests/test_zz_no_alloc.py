"""vmg_norm_inf_static (include/vmg.h): the entry point that allocates nothing, against the existing path.

Collected last on purpose (the suite runs with pytest -x).  The existing path is vmg_step_norm_inf, whose scratch is the
handle's cudaMalloc'ed scalar block; the maximum norm is taken on bit patterns on both sides, so the bar is the one
tests/test_gpu_parity.py uses for it: equality (and NaN for NaN).
"""
import ctypes
import gc

import numpy as np
import pytest

from paper_2507_08200_b200 import binding

CHUNK = 4096   # elements per CTA of the static kernel = elements per partial maximum in the static scratch


def test_sizes_beyond_the_static_scratch_are_rejected_before_any_cuda_call():
    lib = binding.load()
    why = ctypes.c_char_p()
    fake = ctypes.c_void_p(256)          # never dereferenced: the argument checks come first
    assert lib.vmg_norm_inf_static(fake, binding.NORM_INF_STATIC_MAX_N + 1, fake, None, ctypes.byref(why)) == -2
    assert b"VMG_NORM_INF_STATIC_MAX_N" in why.value and b"134217728" in why.value
    assert lib.vmg_norm_inf_static(fake, -1, fake, None, ctypes.byref(why)) == -1
    assert lib.vmg_norm_inf_static(fake, 8, None, None, ctypes.byref(why)) == -1 and b"out" in why.value
    assert lib.vmg_norm_inf_static(None, 8, fake, None, None) == -1


def _arrays(torch):
    rng = np.random.default_rng(2507)
    sizes = [40 * CHUNK + 77, 3 * CHUNK + 1, 1, CHUNK, 5_000_003, 0]       # several CTAs and ragged tails; long before short
    out = []
    for n in sizes:
        x = rng.standard_normal(n)
        if n > 10:
            x[n - 3] = -(7.0 + n * 1e-9)      # the maximum sits in the ragged tail, with a minus sign, different per array
        out.append(torch.from_numpy(x).cuda())
    return out


@pytest.mark.gpu
def test_static_norm_matches_the_existing_path_on_calls_in_a_row():
    torch = pytest.importorskip("torch")
    s = binding.Vmg(8, 8, 8, 0.125, 0.125, 0.125)
    arrays = _arrays(torch)
    outs = torch.full((len(arrays),), -1.0, dtype=torch.float64, device="cuda")
    binding.norm_inf_static(arrays[0], outs[0:1])      # first call on this device: looks the scratch up
    torch.cuda.synchronize()
    gc.collect()
    free_before = torch.cuda.mem_get_info()[0]
    # calls in a row on ONE stream, no synchronisation in between: each sees the scratch the previous one left
    for r in range(2):
        for t, v in enumerate(arrays):
            binding.norm_inf_static(v, outs[t:t + 1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the calls took device memory"
    got = outs.cpu().numpy()
    for t, v in enumerate(arrays):
        want = s.step_norm_inf(v) if v.numel() else 0.0
        assert got[t] == want, (t, v.numel(), got[t], want)
        assert got[t] == (np.abs(v.cpu().numpy()).max() if v.numel() else 0.0)
    # a shorter array right after a longer one with a larger maximum: stale partials must not leak
    big, small = arrays[4], arrays[1]
    o2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    binding.norm_inf_static(big, o2[0:1])
    binding.norm_inf_static(small, o2[1:2])
    a, b = o2.cpu().numpy()
    assert a == s.step_norm_inf(big) and b == s.step_norm_inf(small) and b < a
    # NaN propagates as in the existing path
    bad = arrays[1].clone()
    bad[5] = float("nan")
    binding.norm_inf_static(bad, o2[0:1])
    assert np.isnan(o2[0].item()) and np.isnan(s.step_norm_inf(bad))
    s.destroy()


@pytest.mark.gpu
def test_static_norm_runs_under_stream_capture():
    torch = pytest.importorskip("torch")
    s = binding.Vmg(8, 8, 8, 0.125, 0.125, 0.125)
    v = _arrays(torch)[0]
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    binding.norm_inf_static(v[:0], out)                 # set-up (symbol look-up) outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.graph(g, stream=side):
        binding.norm_inf_static(v, out, stream=torch.cuda.current_stream())
    assert out.item() == 0.0                            # captured, not run
    for _ in range(2):
        v.mul_(1.5)
        g.replay()
        torch.cuda.synchronize()
        assert out.item() == s.step_norm_inf(v)
    s.destroy()
