"""ppm_reduce_conserved_static (include/ppm.h): the conserved sums of SURVEY.md 8(c) C7 for callers that cannot allocate
device memory — the partial sums of the first pass live in a file-scope device array of the library, shared by every call.
Checked against the existing path, ppm_reduce_conserved, on calls in a row that leave different contents in that array.

In a file of its own that pytest collects last: the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  Passes alone in a fresh process (the first call resolves the array's address) and after the other tests."""
import numpy as np
import pytest
import torch

from paper_1810_13416_b200 import workloads as W

pytestmark = pytest.mark.gpu

# another first-pass block count only reorders fp64 additions of the same terms: a few ulp of the largest sum of magnitudes
REORDER_TOL = 1e-12


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1810_13416_b200.binding import PPM
    return PPM


def _static(g, out, nblocks=0):
    g.reduce_conserved_static(out, nblocks)
    torch.cuda.synchronize()
    return out.cpu().numpy().copy()


def test_static_scratch_sums_equal_the_allocating_path_on_calls_in_a_row():
    PPM = _gpu()
    from paper_1810_13416_b200.binding import STATIC_RED_BLOCKS
    out = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")     # the caller's output, allocated once
    w = W.make(1, n=32)
    g = PPM.from_workload(w)
    g.set_state(w.fields().cuda())
    # first call (in a fresh process: the one that looks the array's address up), default block count: bit for bit
    ref0 = g.reduce_conserved()
    got0 = _static(g, out)
    assert np.all(np.isfinite(got0)) and np.array_equal(got0, ref0), (got0, ref0)
    # second call right after it, on a changed state: the array still holds the first call's partial sums
    dt = g.cfl_dt(w.cfl)
    g.step(dt, 0)
    ref1 = g.reduce_conserved()
    got1 = _static(g, out)
    assert np.array_equal(got1, ref1), (got1, ref1)
    assert not np.array_equal(ref1, ref0)
    # the largest block count fills the whole array; a small count after it must not pick up anything it left behind
    scale = np.abs(ref1).max()
    for nb in (STATIC_RED_BLOCKS, 3, 1, 592):
        got = _static(g, out, nb)
        assert np.abs(got - ref1).max() <= REORDER_TOL * scale, (nb, got, ref1)
    assert np.array_equal(_static(g, out, 592), ref1)
    # another context (another grid, gravity with its base state, ragged extents) shares the same array
    w2 = W.make(2, n=18)
    g2 = PPM.from_workload(w2)
    g2.set_state(w2.fields().cuda())
    ref2 = g2.reduce_conserved()
    assert np.array_equal(_static(g2, out), ref2)
    assert np.array_equal(_static(g, out), ref1)            # and back: the first context's sums are unchanged
    assert np.array_equal(_static(g2, out), ref2)
    g2.close()
    g.close()


def test_static_scratch_rejects_what_does_not_fit_and_allocates_nothing():
    PPM = _gpu()
    from paper_1810_13416_b200.binding import PPMError, PPM_EINVAL, STATIC_RED_BLOCKS
    w = W.make(1, n=16)
    g = PPM.from_workload(w)
    g.set_state(w.fields().cuda())
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    ref = g.reduce_conserved()
    _static(g, out)                                          # address resolved, kernels loaded
    with pytest.raises(PPMError) as ei:
        g.reduce_conserved_static(out, STATIC_RED_BLOCKS + 1)
    assert ei.value.code == PPM_EINVAL and "static scratch array holds %d blocks" % STATIC_RED_BLOCKS in str(ei.value)
    with pytest.raises(PPMError) as ei:
        g.reduce_conserved_static(out, -1)
    assert ei.value.code == PPM_EINVAL
    with pytest.raises(ValueError):
        g.reduce_conserved_static(torch.zeros(6, dtype=torch.float64))           # a host tensor is not an output of this call
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)            # the refused calls wrote nothing
    # no device memory is taken or returned by the call (the driver's count of free bytes does not move)
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        g.reduce_conserved_static(out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert np.array_equal(out.cpu().numpy(), ref)
    g.close()
