"""Parity of the metric kernels (tnlm_tv_diff, tnlm_srr, tnlm_cnr through the C ABI) with oracle/tnlm_metrics.py.
Tolerances (M4): the TV kernel forms each |grad h| in fp32 (differences of differences, two FMAs, an
approximate square root: a few ulp, <= ~1e-6 relative of the term in the worst case of cancelling operands that the
random stacks here do not reach) and accumulates non-negative terms in fp64, so TV and SRR are held to a relative
1e-6; the ROI sums are pure fp64 (only the summation order differs): 1e-9."""
import numpy as np
import pytest

from tnlm_inputs import CONFIGS, make_stack, random_stack

pytestmark = pytest.mark.gpu
REL = 1e-6


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


@pytest.mark.parametrize("shape", [(2, 1, 1, 1), (3, 5, 7, 9), (2, 9, 33, 64), (3, 4, 6, 130), (2, 17, 40, 31)])
def test_tv_and_srr_match_oracle(T, shape):
    from oracle import tnlm_metrics as Q
    a, b, c = random_stack(shape, 1), random_stack(shape, 2), random_stack(shape, 3)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    got = T.tnlm_tv_diff(p, dev(a), dev(b)).cpu().numpy()
    want = Q.tv_diff(a, b)
    assert np.allclose(got, want, rtol=REL, atol=1e-300), (got, want)
    got1 = T.tnlm_tv_diff(p, dev(a)).cpu().numpy()
    assert np.allclose(got1, Q.tv_diff(a), rtol=REL, atol=1e-300)
    if want.min() > 0:
        s = T.tnlm_srr(p, dev(a), dev(c), dev(b)).cpu().numpy()
        assert np.allclose(s, Q.srr(a, c, b), rtol=0, atol=2e-6)


def test_tv_special_cases(T):
    import torch
    shape = (2, 6, 8, 12)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    const = torch.full(shape, 3.25, device="cuda")
    assert (T.tnlm_tv_diff(p, const).cpu().numpy() == 0).all()
    a = dev(random_stack(shape, 5))
    assert (T.tnlm_tv_diff(p, a, a).cpu().numpy() == 0).all()
    s = T.tnlm_srr(p, dev(random_stack(shape, 6)), a, a).cpu().numpy()       # enhanced == ground truth
    assert np.allclose(s, 1.0)


def test_cnr_matches_oracle_and_rejects_bad_boxes(T):
    from oracle import tnlm_metrics as Q
    shape = (3, 12, 40, 50)
    s = random_stack(shape, 9)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 0.5)
    for phase, roi, bg in [(0, (2, 5, 3, 9, 4, 11), (6, 12, 20, 40, 30, 50)), (2, (0, 12, 0, 40, 0, 50), (0, 1, 0, 1, 0, 1)),
                           (1, (11, 12, 39, 40, 49, 50), (3, 4, 0, 40, 7, 9))]:
        got = T.tnlm_cnr(p, dev(s), phase, roi, bg).cpu().numpy()
        want = Q.cnr(s, phase, roi, bg)
        with np.errstate(divide="ignore"):
            assert np.allclose(got[:4], want[:4], rtol=1e-9, atol=1e-12), (got, want)
            if np.isfinite(want[4]):
                assert np.isclose(got[4], want[4], rtol=1e-8)
    for bad in [(0, 0, 0, 1, 0, 1), (0, 13, 0, 1, 0, 1), (-1, 2, 0, 1, 0, 1), (0, 1, 0, 1, 5, 51)]:
        with pytest.raises(T.TnlmError) as ei:
            T.tnlm_cnr(p, dev(s), 0, bad, (0, 1, 0, 1, 0, 1))
        assert ei.value.code == -2
    with pytest.raises(T.TnlmError):
        T.tnlm_cnr(p, dev(s), 3, (0, 1, 0, 1, 0, 1), (0, 1, 0, 1, 0, 1))


def test_enhancement_removes_streaks_on_the_thorax_phantom(T):
    """Direction of PAPER.md Table 1 (SRR 85-88 % on their data): positive SRR for every phase, and it is the
    oracle's number (full-size stack of the config-2 recipe, metrics and enhancement all on the GPU)."""
    from oracle import tnlm_metrics as Q
    cfg = CONFIGS["config2"]
    g = make_stack(cfg)
    star = make_stack(cfg, clean=True)
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    gd, sd = dev(g), dev(star)
    f = T.tnlm_enhance(p, gd, cfg.n_iter)
    s = T.tnlm_srr(p, gd, f, sd).cpu().numpy()
    assert (s > 0.3).all() and (s < 1.0).all(), s
    assert np.allclose(s, Q.srr(g, f.cpu().numpy(), star), rtol=0, atol=2e-6)
