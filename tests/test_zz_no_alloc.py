"""cb_permutation_static: the allocation-free variant of the PPO permutation (static device scratch, include/cleanba.h) against
the existing path (cb_permutation, which allocates its scratch per call) -- bit-exact, as for every integer result (A15) --
on two calls in a row.  Collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _setup():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no GPU")
    from paper_2310_00036_b200 import binding
    return torch, binding


def test_permutation_static_matches_existing_path_two_calls_in_a_row():
    torch, binding = _setup()
    # 8192 = config 3 (T=128, B=64); up to 51200 indices the swap loop runs in shared memory, the maximum takes the global-memory branch
    for N in (1, 2, 7, 8192, 40000, binding.PERM_STATIC_MAX):
        out = torch.full((N,), -1, dtype=torch.int32, device="cuda")
        for seed, epoch in ((11, 0), (11, 1)):      # two calls in a row on the same output and the same (shared) scratch
            want = binding.permutation(seed, epoch, N).cpu().numpy()
            got = binding.permutation_static(seed, epoch, N, out=out)
            torch.cuda.synchronize()
            got = got.cpu().numpy()
            assert np.array_equal(got, want), (N, seed, epoch)
            assert np.array_equal(np.sort(got), np.arange(N, dtype=np.int32))
    # a smaller N after a larger one: what the larger call left in the scratch is never read
    a = binding.permutation_static(5, 3, 8192).cpu().numpy()
    assert np.array_equal(a, binding.permutation(5, 3, 8192).cpu().numpy())


def test_permutation_static_allocates_nothing_and_rejects_large_N():
    torch, binding = _setup()
    N = 8192
    out = torch.empty((N,), dtype=torch.int32, device="cuda")
    binding.permutation_static(1, 0, N, out=out)      # set-up (symbol address, shared-memory opt-in) happens on the first call
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for e in range(8):
        binding.permutation_static(1, e, N, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0      # no device memory taken by the calls (the driver's pools included)
    with pytest.raises(RuntimeError, match="CB_PERM_STATIC_MAX"):
        binding.permutation_static(1, 0, binding.PERM_STATIC_MAX + 1, out=torch.empty((binding.PERM_STATIC_MAX + 1,), dtype=torch.int32, device="cuda"))
    binding.permutation_static(1, 0, 0, out=out)      # empty: nothing launched
