"""dp_scan_exclusive_static (include/dp.h): the exclusive prefix sum of the neighbour-list build from an entry point that
allocates nothing (its scratch is a static device array inside the library), against the existing path dp_scan_exclusive
(caller-owned scratch; the scan dp_compute runs).  Integer work: the comparison is bit-exact.  Collected last on purpose
(the suite runs with pytest -x).  The file depends on no other test: it passes alone in a fresh process and after the rest."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SIZES = [1, 5, 4095, 4096, 4097, 3 * 4096 + 17, 1_000_003]


def _inputs(torch, n, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return torch.randint(0, 100, (n,), generator=g, dtype=torch.int32).cuda()


def _existing(torch, binding, cnt):
    n = cnt.numel()
    out = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    scratch = torch.empty(int(binding.lib().dp_scan_scratch_bytes(n)) // 4 + 1, dtype=torch.int32, device="cuda")
    binding.scan_exclusive(cnt, out, scratch)
    return out


def test_static_scan_matches_existing_path_on_two_calls_in_a_row():
    import torch
    from paper_2005_00223_b200 import binding
    # two calls in a row on one stream, the second on a SHORTER input than the first: the shared scratch still holds the first
    # call's tile sums beyond the second call's range, and they must not leak into its result
    big, small = _inputs(torch, 1_000_003, 1), _inputs(torch, 3 * 4096 + 17, 2)
    out_big = torch.full((big.numel() + 1,), -7, dtype=torch.int32, device="cuda")
    out_small = torch.full((small.numel() + 1,), -7, dtype=torch.int32, device="cuda")
    binding.scan_exclusive_static(big, out_big)
    binding.scan_exclusive_static(small, out_small)
    torch.cuda.synchronize()
    for cnt, out in ((big, out_big), (small, out_small)):
        ref = _existing(torch, binding, cnt)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        # and both agree with the definition (int64 cumulative sum on the host)
        host = np.concatenate([[0], np.cumsum(cnt.cpu().numpy().astype(np.int64))])
        assert np.array_equal(out.cpu().numpy().astype(np.int64), host)
    # the same input again gives the same output again
    again = torch.full_like(out_small, -7)
    binding.scan_exclusive_static(small, again)
    torch.cuda.synchronize()
    assert torch.equal(again, out_small)


@pytest.mark.parametrize("n", SIZES)
def test_static_scan_sizes(n):
    """one element, a ragged tail, exactly one tile, one past a tile, several tiles"""
    import torch
    from paper_2005_00223_b200 import binding
    cnt = _inputs(torch, n, 100 + n)
    out = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    binding.scan_exclusive_static(cnt, out)
    ref = _existing(torch, binding, cnt)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    assert int(out[0].item()) == 0 and int(out[n].item()) == int(cnt.sum().item())


def test_static_scan_maximum_size_and_rejection():
    import torch
    from paper_2005_00223_b200 import binding
    L = binding.lib()
    nmax = binding.SCAN_STATIC_MAX
    cnt = torch.ones(nmax, dtype=torch.int32, device="cuda")
    out = torch.empty(nmax + 1, dtype=torch.int32, device="cuda")
    binding.scan_exclusive_static(cnt, out)                   # the largest size the static scratch serves
    torch.cuda.synchronize()
    assert torch.equal(out, torch.arange(nmax + 1, dtype=torch.int32, device="cuda"))
    st = torch.cuda.current_stream().cuda_stream
    # one more element: rejected with DP_ENOMEM before anything is launched (pointers are not touched)
    assert L.dp_scan_exclusive_static(nmax + 1, cnt.data_ptr(), out.data_ptr(), st) == -3
    assert L.dp_scan_exclusive_static(0, cnt.data_ptr(), out.data_ptr(), st) == -1
    assert L.dp_scan_exclusive_static(16, None, out.data_ptr(), st) == -1
    assert L.dp_scan_exclusive_static(16, cnt.data_ptr(), None, st) == -1
    with pytest.raises(binding.DPError) as ei:
        binding.scan_exclusive_static(torch.ones(nmax + 1, dtype=torch.int32, device="cuda"),
                                      torch.empty(nmax + 2, dtype=torch.int32, device="cuda"))
    assert ei.value.code == -3
    torch.cuda.synchronize()
    assert torch.equal(out, torch.arange(nmax + 1, dtype=torch.int32, device="cuda"))      # untouched by the rejected calls


def test_static_scan_allocates_no_device_memory():
    """free device memory (driver view, cudaMemGetInfo) is the same before and after calls of the entry point"""
    import torch
    from paper_2005_00223_b200 import binding
    cnt = _inputs(torch, 200_000, 7)
    out = torch.empty(cnt.numel() + 1, dtype=torch.int32, device="cuda")
    binding.scan_exclusive_static(cnt, out)                   # first call: symbol look-up, module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        binding.scan_exclusive_static(cnt, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
