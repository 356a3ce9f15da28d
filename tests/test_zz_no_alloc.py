"""mf_vegas_iterate_static (include/mf.h): the iteration call for callers that must not allocate; its scratch is a file-scope
static __device__ array inside the library.  Checked against the existing mf_vegas_iterate on the same inputs, two calls in a
row (the array keeps the first call's contents when the second one starts), plus the refusals.  Collected last on purpose: the
suite runs with pytest -x.  Own handles (no session fixtures), so it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2106_10279_b200 import workloads as W

pytestmark = pytest.mark.gpu
REL_ITER = 1e-9          # the per-iteration tolerance of tests/test_gpu_parity.py


def _run(proc, call, grid, seed, it, first, n):
    import torch
    hist, res = proc.new_hist(), proc.new_result()
    call(grid, seed, it, first, n, hist, res)
    torch.cuda.synchronize()
    return hist.cpu().numpy(), proc.result_to_host(res)


@pytest.mark.parametrize("wl", [W.C1, W.C5, W.C0], ids=["gg_tt", "pp_tt", "ee_mumu"])
def test_static_scratch_iteration_equals_the_existing_path(wl):
    import torch
    from paper_2106_10279_b200 import api
    proc = api.Process(wl, W.pdf_for(wl.process))
    try:
        grid = torch.from_numpy(W.uniform_grid(wl.n_dims, wl.n_bins)).cuda()
        # two calls in a row with different streams of events and sizes (the second one smaller and ragged: whatever the first
        # one left in the shared array must not leak into it), then the first one again
        for seed, it, first, n in [(0, 0, 0, 300000), (7, 3, (1 << 33) + 5, 4099), (0, 0, 0, 300000)]:
            h_ref, r_ref = _run(proc, proc.vegas_iterate, grid, seed, it, first, n)
            h_new, r_new = _run(proc, proc.vegas_iterate_static, grid, seed, it, first, n)
            assert r_new.n_pass == r_ref.n_pass and r_new.n_accept == r_ref.n_accept
            assert abs(r_new.sum_w - r_ref.sum_w) <= REL_ITER * abs(r_ref.sum_w)
            assert abs(r_new.sum_w2 - r_ref.sum_w2) <= REL_ITER * r_ref.sum_w2
            assert abs(r_new.max_abs_w - r_ref.max_abs_w) <= REL_ITER * r_ref.max_abs_w
            np.testing.assert_allclose(h_new, h_ref, rtol=REL_ITER, atol=1e-14 * h_ref.max())
            assert r_ref.n_pass > 0 and h_ref.max() > 0
        # without a histogram, and an empty range
        res = proc.new_result()
        proc.vegas_iterate_static(grid, 1, 1, 0, 1000, None, res)
        ref = proc.new_result()
        proc.vegas_iterate(grid, 1, 1, 0, 1000, None, ref)
        torch.cuda.synchronize()
        assert abs(proc.result_to_host(res).sum_w - proc.result_to_host(ref).sum_w) <= REL_ITER * abs(proc.result_to_host(ref).sum_w)
        h0, r0 = _run(proc, proc.vegas_iterate_static, grid, 0, 0, 0, 0)
        assert r0.sum_w == 0 and r0.n_pass == 0 and not h0.any()
    finally:
        proc.close()


def test_static_scratch_refusals():
    """beyond the array's size, and for the kernels whose scratch is tens of MB: MF_EINVAL with the reason, nothing launched"""
    import dataclasses
    import torch
    from paper_2106_10279_b200 import api
    big = dataclasses.replace(W.C1, n_bins=128)          # 444 blocks x (40 + 8 x 4 x 128) bytes = 1.8 MB > 1 MiB
    for wl, word in [(big, "static"), (W.C2, "thread-per-event")]:
        proc = api.Process(wl, W.pdf_for(wl.process))
        try:
            grid = torch.from_numpy(W.uniform_grid(wl.n_dims, wl.n_bins)).cuda()
            hist, res = proc.new_hist(), proc.new_result()
            with pytest.raises(api.MfError) as err:
                proc.vegas_iterate_static(grid, 0, 0, 0, 1000, hist, res)
            assert "EINVAL" in str(err.value) and word in str(err.value)
            proc.vegas_iterate(grid, 0, 0, 0, 1000, hist, res)        # the existing path still serves the same handle
            torch.cuda.synchronize()
            assert proc.result_to_host(res).n_pass > 0
        finally:
            proc.close()
