"""qhp_pibar_noalloc (include/qhp.h): the PI-BAR estimator (Eq. 27-28) through the entry point
that allocates nothing (partial sums in a static device array of the library) against the existing qhp_pibar.
Collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

KB = 1.987204258640832e-3
BETA = 1.0 / (KB * 300.0)


def _series(nA, nB):
    import torch
    rng = np.random.default_rng(7 * nA + nB)
    wA, wB = rng.normal(0.8, 0.7, nA), rng.normal(-0.3, 0.5, nB)
    return torch.as_tensor(wA).cuda(), torch.as_tensor(wB).cuda()


def test_two_calls_in_a_row_match_the_allocating_path():
    import torch
    import paper_2212_03137_b200 as qhp
    # two problems of different size back to back: the second call finds the first one's partial sums in the
    # shared scratch array (more CTAs first, then fewer, then more again)
    cases = [_series(300_001, 299_999), _series(31, 1000), _series(4000, 2500)]
    outs = [torch.full((2,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    qhp.qhp_pibar_noalloc(*cases[0], BETA, outs[0])            # first call on the device: set-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (wA, wB), out in zip(cases, outs):                     # same stream: the calls do not overlap
        qhp.qhp_pibar_noalloc(wA, wB, BETA, out)
    qhp.qhp_pibar_noalloc(*cases[0], BETA, outs[0], max_iter=3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0               # no device memory was taken or returned
    dF3, it3 = outs[0].tolist()
    ref3, itr3 = qhp.qhp_pibar(*cases[0], BETA, max_iter=3)
    assert it3 == itr3 <= 3 and abs(dF3 - ref3) < 1e-11 * max(1.0, abs(ref3))
    for (wA, wB), out in list(zip(cases, outs))[1:]:
        ref, it_ref = qhp.qhp_pibar(wA, wB, BETA)
        dF, it = out.tolist()
        assert abs(dF - ref) < 1e-11 * max(1.0, abs(ref))      # the tolerance of tests/test_gpu_pibar.py
        assert int(it) == it_ref
    # and once more after the allocating path ran in between
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qhp.qhp_pibar_noalloc(*cases[0], BETA, out)
    torch.cuda.synchronize()
    ref, it_ref = qhp.qhp_pibar(*cases[0], BETA)
    assert abs(out[0].item() - ref) < 1e-11 * max(1.0, abs(ref)) and int(out[1].item()) == it_ref


def test_matches_the_oracle_and_rejects_what_does_not_fit():
    import torch
    import oracle as O
    import paper_2212_03137_b200 as qhp
    wA, wB = _series(4000, 2500)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qhp.qhp_pibar_noalloc(wA, wB, BETA, out)
    torch.cuda.synchronize()
    ref, _ = O.pibar(wA.cpu().numpy(), wB.cpu().numpy(), BETA)
    assert abs(out[0].item() - ref) < 1e-11 * max(1.0, abs(ref))
    big = torch.zeros(qhp.PIBAR_NOALLOC_MAX_N + 1, dtype=torch.float64, device="cuda")
    before = out.clone()
    with pytest.raises(qhp.QhpError, match="QHP_PIBAR_NOALLOC_MAX_N") as ei:
        qhp.qhp_pibar_noalloc(big, wB, BETA, out)
    assert ei.value.code == -1
    with pytest.raises(qhp.QhpError, match="QHP_PIBAR_NOALLOC_MAX_N"):
        qhp.qhp_pibar_noalloc(wA, big, BETA, out)
    with pytest.raises(qhp.QhpError):
        qhp.qhp_pibar_noalloc(wA, wB, -1.0, out)
    with pytest.raises(qhp.QhpError):
        qhp.qhp_pibar_noalloc(wA[:0], wB, BETA, out)
    torch.cuda.synchronize()
    assert torch.equal(out, before)                            # a rejected call launches nothing
    qhp.qhp_pibar_noalloc(big[:-1], wB, BETA, out)             # exactly the maximum is served
    torch.cuda.synchronize()
    ref, _ = qhp.qhp_pibar(big[:-1], wB, BETA)
    assert abs(out[0].item() - ref) < 1e-11 * max(1.0, abs(ref))
