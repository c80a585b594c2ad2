"""tnlm_srr_static (include/tnlm.h): the streak-reduction ratio of Eq. 10 through the entry point that
allocates nothing -- its scratch is a static device array inside libtnlm.so -- against the existing tnlm_srr path with a
caller workspace, and against the metrics oracle, on calls in a row that share that array.

This file is named so that pytest collects it last (the suite runs with `pytest -x`).  It must pass alone in a fresh
process (the first call on the device looks the array's address up) and after every other GPU test.
Tolerance: the one tests/test_metrics_gpu.py holds tnlm_srr to (atol 2e-6; the two paths run the same kernels, only the
order of the fp64 atomic adds differs)."""
import numpy as np
import pytest

from tnlm_inputs import random_stack

pytestmark = pytest.mark.gpu
ATOL = 2e-6


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1201_2450_b200 as T
    T.lib()
    return T


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def stacks(shape, seed, streak):
    """ground truth, a streaky 'FDK' stack and a half-cleaned 'enhanced' one"""
    star = random_stack(shape, seed)
    noise = random_stack(shape, seed + 1) - 0.5
    return star, star + streak * noise, star + 0.4 * streak * noise


def test_srr_static_matches_workspace_path_on_calls_in_a_row(T):
    import torch
    from oracle import tnlm_metrics as Q
    # the second call has fewer phases, another volume and much smaller TV sums than the first: sums left in the shared
    # array by the first call would show; the third repeats the first
    cases = [((5, 9, 33, 64), 11, 3.0), ((3, 4, 6, 130), 12, 0.01), ((5, 9, 33, 64), 11, 3.0)]
    for shape, seed, streak in cases:
        star, fdk, enh = stacks(shape, seed, streak)
        p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
        a, b, c = dev(fdk), dev(enh), dev(star)
        out = torch.full((shape[0],), float("nan"), dtype=torch.float64, device="cuda")
        got = T.tnlm_srr_static(p, a, b, c, out=out)
        assert got is out
        want = T.tnlm_srr(p, a, b, c)
        torch.cuda.synchronize()
        assert np.allclose(got.cpu().numpy(), want.cpu().numpy(), rtol=0, atol=ATOL)
        assert np.allclose(got.cpu().numpy(), Q.srr(fdk, enh, star), rtol=0, atol=ATOL)


def test_srr_static_back_to_back_on_one_stream_without_sync(T):
    """Two calls queued on one stream with no host synchronisation between them: the second clears and reuses the array
    after the first has read it (stream order), so both results stand."""
    import torch
    shape = (4, 6, 20, 48)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    s1, f1, e1 = (dev(x) for x in stacks(shape, 21, 2.0))
    s2, f2, e2 = (dev(x) for x in stacks(shape, 23, 0.05))
    o1 = torch.empty(4, dtype=torch.float64, device="cuda")
    o2 = torch.empty(4, dtype=torch.float64, device="cuda")
    T.tnlm_srr_static(p, f1, e1, s1, out=o1)
    T.tnlm_srr_static(p, f2, e2, s2, out=o2)
    torch.cuda.synchronize()
    assert np.allclose(o1.cpu().numpy(), T.tnlm_srr(p, f1, e1, s1).cpu().numpy(), rtol=0, atol=ATOL)
    assert np.allclose(o2.cpu().numpy(), T.tnlm_srr(p, f2, e2, s2).cpu().numpy(), rtol=0, atol=ATOL)


def test_srr_static_limit_and_device_memory(T):
    """The maximum is enforced with its own status code, the largest allowed size works, and a call leaves the device's
    free memory where it was (nothing is allocated behind the caller's back)."""
    import torch
    n_max = T.binding.SRR_STATIC_MAX_PHASES
    shape = (n_max + 1, 2, 3, 4)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    x = torch.zeros(shape, dtype=torch.float32, device="cuda")
    with pytest.raises(T.TnlmError) as ei:
        T.tnlm_srr_static(p, x, x, x)
    assert ei.value.code == -8 and "TNLM_SRR_STATIC_MAX_PHASES" in T.strerror(-8)

    shape = (n_max, 2, 5, 8)
    star, fdk, enh = stacks(shape, 31, 1.0)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    a, b, c = dev(fdk), dev(enh), dev(star)
    out = torch.empty(n_max, dtype=torch.float64, device="cuda")
    T.tnlm_srr_static(p, a, b, c, out=out)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    T.tnlm_srr_static(p, a, b, c, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert np.allclose(out.cpu().numpy(), T.tnlm_srr(p, a, b, c).cpu().numpy(), rtol=0, atol=ATOL)
