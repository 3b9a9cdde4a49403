"""GPU test (-m gpu) of landau_moments_noalloc, the one entry point of liblandau.so that allocates no
device memory (include/landau.h; csrc/moments_noalloc.cu).

It exists for callers that cannot call cudaMalloc: a host code whose own arrays (or whose framework's
fixed pool) already own all of HBM, or a diagnostics hook inside an asynchronous time loop, where a
cudaMalloc / cudaFree would synchronise the whole device.  Its scratch is a fixed 640 KiB __device__
array inside the library, shared by every call and never cleared between calls, so what is checked here
is: the result equals the context path's (landau_set_markers + landau_moments, which the other GPU
tests compare with the oracle) within the moments tolerance of tests/test_gpu_parity.py, on TWO calls
in a row -- the second smaller than the first, with fewer species, so that anything the first call
left behind in the scratch would show -- and that sizes beyond the array are refused, not truncated.

This file is named to be collected last (pytest -x stops at the first failure; a failure here must
not hide the parity tests), and it passes alone in a fresh process as well as after the others: it
makes no assumption on whether the first call on the device has already happened.
"""
import numpy as np
import pytest

from paper_2212_00663_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-12, 1e-13   # the bounds test_moments_match_oracle uses for n, K (P: 1e-13 of sum |w m|)


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the CUDA path has no fallback")
    from paper_2212_00663_b200 import binding
    binding.load()
    return binding


def context_path(B, wl):
    g = B.Landau(wl.mass, wl.charge, wl.eps)
    g.set_markers(wl.v, wl.w, wl.species_id)
    m = g.moments(with_entropy=False)
    g.close()
    return m


def device_inputs(wl):
    import torch
    dev = torch.device("cuda", 0)
    v = torch.as_tensor(wl.v, dtype=torch.float64, device=dev).contiguous()
    w = torch.as_tensor(wl.w, dtype=torch.float64, device=dev).contiguous()
    sid = torch.as_tensor(wl.species_id, dtype=torch.int32, device=dev).contiguous()
    out = torch.full((len(wl.mass), 5), -7.0, dtype=torch.float64, device=dev)
    return v, w, sid, out


def assert_same_moments(out, ref, wl):
    got = out.cpu().numpy()
    assert np.all(np.isfinite(got))
    np.testing.assert_allclose(got[:, 0], ref["n"], rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(got[:, 4], ref["K"], rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(got[:, 1:4], ref["P"], rtol=0,
                               atol=1e-13 * np.abs(wl.w * wl.mass[wl.species_id]).sum())


def test_noalloc_moments_equal_context_path_on_two_calls_in_a_row(B):
    import torch
    # first call: 3 species x 33 333 markers (49 blocks, ragged tail), caller order shuffled
    wl1 = W.make(4, n_per_species=33333, shuffled=True)
    # second call: 2 species x 3000 markers -- fewer blocks and fewer species than what call 1 left behind
    wl2 = W.make(1, n_per_species=3000, shuffled=True)
    ref1, ref2 = context_path(B, wl1), context_path(B, wl2)
    in1, in2 = device_inputs(wl1), device_inputs(wl2)
    torch.cuda.synchronize()

    B.moments_noalloc(in1[0], in1[1], in1[2], wl1.mass, in1[3])
    # by now the per-device set-up has happened, whichever test ran first: from here on the entry
    # point must leave the amount of free device memory exactly where it was
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    B.moments_noalloc(in2[0], in2[1], in2[2], wl2.mass, in2[3])
    B.moments_noalloc(in1[0], in1[1], in1[2], wl1.mass, in1[3])   # and back to the large one, in place
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before

    assert_same_moments(in1[3], ref1, wl1)
    assert_same_moments(in2[3], ref2, wl2)


def test_noalloc_refuses_what_does_not_fit_and_flags_bad_species(B):
    import torch
    wl = W.make(0, n_per_species=300, shuffled=True)
    v, w, sid, out = device_inputs(wl)
    with pytest.raises(B.LandauError) as e:
        B.moments_noalloc(v, w, sid, wl.mass, out, N=B.MOMENTS_NOALLOC_MAX_N + 1)   # size check comes first
    assert e.value.code == B.EINVAL and "LANDAU_MOMENTS_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(B.LandauError):
        B.moments_noalloc(v, w, sid, list(wl.mass) * 9, torch.empty(5 * 9 * len(wl.mass), dtype=torch.float64,
                                                                    device=v.device))   # > 16 species
    torch.cuda.synchronize()
    assert float(out[0, 0]) == -7.0   # nothing was launched
    # a species id outside 0..S-1 poisons the output instead of being summed somewhere
    bad = sid.clone()
    bad[17] = len(wl.mass)
    B.moments_noalloc(v, w, bad, wl.mass, out)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())
    # ... and the flag does not stick: the next call clears it
    B.moments_noalloc(v, w, sid, wl.mass, out)
    assert_same_moments(out, context_path(B, wl), wl)
