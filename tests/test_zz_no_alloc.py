"""mg_sigma_batch_noalloc: the entry point that allocates nothing (README, "callers that cannot call cudaMalloc").

It runs g g -> t tbar g g g g with the generic diagram kernel's scratch in a file-scope `static __device__` array
(csrc/hsg_kernel.cu) instead of the handle's cudaMalloc'ed scratch areas.  Checked against the existing path
(mg_sigma_batch) on two calls in a row -- the array keeps the previous call's contents -- within the fp64 tolerance of
tests/test_gpu_parity.py (1e-10; the kernels are the same, so the numbers are in fact identical), plus the size limit.
Collected last on purpose (pytest -x): it must pass alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_2510_05392_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def test_no_alloc_entry_point_matches_the_existing_path():
    from paper_2510_05392_b200 import binding as B
    B.load_library()
    assert torch.cuda.is_available()
    process = "gg_ttxgggg"
    max_evt = B.NOALLOC_MAX_EVENTS
    for prec, tol in (("fp64", 1e-10), ("mixed", 1e-10)):          # same kernels on both paths in either precision
        proc = B.init_process(process, prec)
        proc.set_good_helicities(np.ones(proc.ncomb, dtype=np.uint8))
        # two calls in a row on different events: 40 events = 5 per CTA of the static scratch, then a ragged 13
        for nevt, seed in ((40, 11), (13, 12)):
            mom = inputs.momenta(process, nevt, seed=seed)
            d_mom = torch.from_numpy(mom).cuda()
            ref = proc.sigma_batch(d_mom).cpu().numpy()
            got = proc.sigma_batch_noalloc(d_mom).cpu().numpy()
            assert np.isfinite(got).all() and (got > 0).all()
            assert np.abs(got / ref - 1).max() < tol, (prec, nevt, np.abs(got / ref - 1).max())
        # and the existing path is untouched by the static one
        again = proc.sigma_batch(d_mom).cpu().numpy()
        assert np.array_equal(again, ref)
        # beyond the stated maximum: a clear error, nothing launched
        mom = inputs.momenta(process, max_evt + 1, seed=1)
        with pytest.raises(B.MGError, match="at most"):
            proc.sigma_batch_noalloc(torch.from_numpy(mom).cuda())
        proc.close()
    # a process whose kernels use no scratch memory has no such entry point
    proc = B.init_process("gg_ttxg", "fp64")
    proc.set_good_helicities(np.ones(proc.ncomb, dtype=np.uint8))
    with pytest.raises(B.MGError):
        proc.sigma_batch_noalloc(torch.from_numpy(inputs.momenta("gg_ttxg", 8)).cuda())
    proc.close()
    # without a helicity list the call refuses (the filter would synchronise and copy to the host)
    proc = B.init_process(process, "fp64")
    with pytest.raises(B.MGError, match="helicit"):
        proc.sigma_batch_noalloc(torch.from_numpy(inputs.momenta(process, 4)).cuda())
    proc.close()
