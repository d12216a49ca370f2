"""woden_truncate_select_static: the Eq 23-24 selection for callers that cannot
allocate device memory -- a stage inside a host framework's fixed device arena, a plug-in called while
the allocator is locked, a process under a GPU memory quota, a loop that cannot take cudaMalloc's
device-wide stall.  Its ranked list sits in a fixed 16384-entry array built into the library instead of
the context arena woden_truncate_select grows with cudaMalloc.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  The GPU test has to pass both alone in a fresh process (where its first call
does the per-device address look-up) and after every other test has used the library."""
import numpy as np
import pytest

from paper_2005_09316_b200 import binding


def test_sizes_beyond_the_built_in_array_are_refused_before_any_cuda_work():
    L = binding.load()
    too_long = binding.WODEN_STATIC_TRUNCATE_MAX + 1
    assert L.woden_truncate_select_static(too_long, None, 0.5, None, None, None) == binding.WODEN_ERR_STATIC_LIMIT
    msg = L.woden_static_last_error().decode()
    assert "WODEN_STATIC_TRUNCATE_MAX" in msg and "woden_truncate_select" in msg
    assert "built-in scratch" in L.woden_strerror(binding.WODEN_ERR_STATIC_LIMIT).decode()
    assert L.woden_truncate_select_static(-1, None, 0.5, None, None, None) == binding.WODEN_ERR_DIM
    assert L.woden_truncate_select_static(4, None, float("nan"), None, None, None) == binding.WODEN_ERR_DIM
    assert L.woden_truncate_select_static(4, None, 0.5, None, None, None) == binding.WODEN_ERR_NULL
    assert L.woden_static_last_error().decode() != ""


def _weights(seed, n):
    rng = np.random.default_rng(seed)
    w = rng.normal(0.0, 1.0, n) * rng.lognormal(0.0, 2.0, n)
    w[rng.integers(0, n, max(1, n // 16))] = w[0]            # equal values: Eq 24 ties keep list order
    return w


@pytest.mark.gpu
def test_static_scratch_selection_equals_the_allocating_path_on_two_calls_in_a_row():
    import torch
    from oracle import truncate as otrunc
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    ctx = binding.Woden(0)
    # second call shorter than the first (the array then still holds the first call's tail), then the limit
    cases = [(11, 5000, 0.9), (12, 777, 0.35), (13, binding.WODEN_STATIC_TRUNCATE_MAX, 0.999), (14, 1, 0.5),
             (15, 300, 1.0), (16, 300, 0.0)]
    tensors = []
    for seed, n, f in cases:
        w = torch.from_numpy(_weights(seed, n)).to(dev)
        tensors.append((w, f, torch.full((n,), -7, dtype=torch.int32, device=dev),
                        torch.full((1,), -7, dtype=torch.int32, device=dev)))
    w0, f0, keep0, nk0 = tensors[0]
    binding.truncate_select_static(w0, f0, keep0, nk0)           # first call on this device: address look-up
    torch.cuda.synchronize()
    keep0.fill_(-7); nk0.fill_(-7)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    for w, f, keep, nk in tensors:                               # back to back on one stream, no sync between
        binding.truncate_select_static(w, f, keep, nk)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] >= free_before        # nothing was taken from the device
    for w, f, keep, nk in tensors:
        ref_keep, ref_nk = ctx.truncate_select(w, f)             # the existing, allocating path
        torch.cuda.synchronize()
        assert int(nk.item()) == int(ref_nk.item())              # integer work: bit-exact
        assert torch.equal(keep, ref_keep)
        mask = otrunc.keep_mask(w.cpu().numpy(), f)              # and both equal the oracle
        assert np.array_equal(keep.cpu().numpy().astype(bool), mask)
        assert int(nk.item()) == int(mask.sum())
    # an empty list writes N_comp = 0 and touches nothing else
    nk = torch.full((1,), -7, dtype=torch.int32, device=dev)
    binding.truncate_select_static(torch.empty(0, dtype=torch.float64, device=dev), 0.5,
                                   torch.empty(0, dtype=torch.int32, device=dev), nk)
    assert int(nk.item()) == 0
    with pytest.raises(binding.WodenError) as e:
        n = binding.WODEN_STATIC_TRUNCATE_MAX + 1
        binding.truncate_select_static(torch.zeros(n, dtype=torch.float64, device=dev), 0.5,
                                       torch.zeros(n, dtype=torch.int32, device=dev), nk)
    assert e.value.status == binding.WODEN_ERR_STATIC_LIMIT
    ctx.close()
