"""lofar_trigger_static -- the allocation-free entry point (fixed file-scope device scratch, no plan, no cudaMalloc)
against the existing path lofar_trigger on the same series, two calls in a row: the second call is smaller and has
other data, so anything left in the shared scratch by the first call would show.  Collected last on purpose (the
suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes

import numpy as np
import pytest

from paper_1612_06592_b200 import binding

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    binding.load()
    return t


def _series(torch, nseries, n, seed, spikes):
    g = torch.Generator(device="cuda").manual_seed(seed)
    x = torch.randn((nseries, n), generator=g, device="cuda", dtype=torch.float32) * 37.0
    rng = np.random.default_rng(seed)
    for _ in range(spikes):                     # a few samples far above 6 sigma, also in the ragged last chunk
        s, i = int(rng.integers(nseries)), int(rng.integers(n))
        x[s, i] = float(rng.choice([-1.0, 1.0])) * float(rng.uniform(260.0, 900.0))
    x[nseries - 1, n - 1] = 700.0
    x[0, 0] = -650.0
    return x.contiguous()


def _outputs(torch, nseries, cap):
    return (torch.full((cap, 24), 0xAB, dtype=torch.uint8, device="cuda"),       # stale bytes on purpose
            torch.full((1,), 12345, dtype=torch.int32, device="cuda"),
            torch.full((nseries,), -1.0, dtype=torch.float32, device="cuda"))


def test_static_trigger_matches_the_plan_path_twice(torch):
    nseries, kappa, cap = 5, 6.0, 4096
    plan = binding.Plan(2, 4, nseries, 16, 0.0)                 # the existing path: a plan with 5 series
    plan.set_input(binding.LOFAR_CI8, 64)
    plan.set_trigger(kappa, 1, cap)
    offset = 0
    for call, (slices, seed) in enumerate(((50, 11), (20, 12))):   # 51200 and 20480 samples: ragged last chunks
        n = slices * 1024
        x = _series(torch, nseries, n, seed, spikes=9)
        cand_r, count_r, sigma_r = _outputs(torch, nseries, cap)
        plan.trigger(x, slices, cand_r, count_r, sigma_r)
        torch.cuda.synchronize()
        cand_s, count_s, sigma_s = _outputs(torch, nseries, cap)
        free0, _ = torch.cuda.mem_get_info()
        binding.trigger_static(x, n, kappa, cand_s, count_s, sigma_s, offset=offset)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        if call == 1:                            # everything lazy (module load) happened in the first call
            assert free0 - free1 < (1 << 20), "device memory was allocated inside lofar_trigger_static"
        # sigma: same kernels, same summation order -> the tolerance the other trigger tests use is 5e-6
        np.testing.assert_allclose(sigma_s.cpu().numpy(), sigma_r.cpu().numpy(), rtol=5e-6)
        ref = float(x.double().pow(2).mean(dim=1).sqrt()[2].item())
        assert abs(float(sigma_s[2].item()) / ref - 1.0) < 5e-6
        assert int(count_s.item()) == int(count_r.item()) >= 10
        rec_s = binding.candidates_to_numpy(cand_s, count_s)
        rec_r = binding.candidates_to_numpy(cand_r, count_r)
        assert rec_s.size == rec_r.size
        for f in ("series", "trial", "sample", "env", "sigma"):
            assert np.array_equal(rec_s[f], rec_r[f]), f
        assert np.all(rec_s["sample"] >= offset) and np.all(rec_s["sample"] < offset + n)
        key = rec_s["series"].astype(np.int64) * (1 << 40) + rec_s["sample"].astype(np.int64)
        assert np.all(np.diff(key) > 0), "sorted by (series, sample)"
        offset += n
    plan.destroy()


def test_static_trigger_rejects_sizes_beyond_its_scratch(torch):
    lib = binding.load()
    x = torch.zeros((2, 1024), dtype=torch.float32, device="cuda")
    cand = torch.zeros((16, 24), dtype=torch.uint8, device="cuda")
    count = torch.zeros(1, dtype=torch.int32, device="cuda")
    sigma = torch.zeros(2, dtype=torch.float32, device="cuda")
    too_many = (binding.STATIC_MAX_CHUNKS // 2 + 1) * 16384      # 2 series: one chunk more than the array holds
    st = lib.lofar_trigger_static(x.data_ptr(), 2, too_many, too_many, 6.0, 0, cand.data_ptr(), 16, count.data_ptr(),
                                  sigma.data_ptr(), None)
    assert st == binding.LOFAR_E_SHAPE            # rejected before anything is launched or read
    assert binding.status_string(st) == "shape out of range"
    st = lib.lofar_trigger_static(None, 2, 1024, 1024, 6.0, 0, cand.data_ptr(), 16, count.data_ptr(), sigma.data_ptr(), None)
    assert st == binding.LOFAR_E_INVALID
    torch.cuda.synchronize()
    assert int(count.item()) == 0
