"""GPU parity of the stand-alone primitives: Philox words (bit-exact), Box-Muller normals, the
shared-memory Stockham FFT.  All calls go through the C ABI (paper_2212_03137_b200.binding)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_philox_words_bit_exact_and_normals():
    import oracle as O
    import paper_2212_03137_b200 as qhp
    seed = 0x0123456789ABCDEF
    for (atom0, mode, tag, step, n) in [(0, 0, 3, 0, 257), (1000, 31, 3, 123456789012, 64), (215990, 0, 4, 3071, 10)]:
        words, z = qhp.qhp_philox_normals(seed, atom0, mode, tag, step, n)
        words = words.cpu().numpy().view(np.uint32)
        z = z.cpu().numpy()
        assert not np.isnan(z).any()        # NaN = the component-wise and 3-at-once device paths disagree
        for i in range(n):
            ref = O.philox4x32_10([atom0 + i, mode | (tag << 24), step & 0xFFFFFFFF, step >> 32],
                                  [seed & 0xFFFFFFFF, seed >> 32])
            assert np.array_equal(words[i], ref)                       # integer work: bit-exact
            zr = O.normals3(seed, atom0 + i, mode, tag, step)
            assert np.abs(z[i] - zr).max() < 4e-15 * max(1.0, np.abs(zr).max())


def test_philox_normal_moments():
    import paper_2212_03137_b200 as qhp
    _, z = qhp.qhp_philox_normals(42, 0, 5, 3, 7, 400000)
    z = z.cpu().numpy().ravel()
    n = z.size
    assert abs(z.mean()) < 5 / np.sqrt(n)
    assert abs(z.var() - 1) < 5 * np.sqrt(2 / n)
    assert abs((z ** 4).mean() - 3) < 5 * np.sqrt(96 / n)


@pytest.mark.parametrize("n", [8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192])
def test_fft_matches_dft(n):
    import torch
    import paper_2212_03137_b200 as qhp
    rng = np.random.default_rng(n)
    batch = 5
    x = rng.standard_normal((batch, n)) + 1j * rng.standard_normal((batch, n))
    ref = np.fft.fft(x, axis=1)
    if n <= 256:   # direct O(n^2) DFT as the definition
        k = np.arange(n)
        Wm = np.exp(-2j * np.pi * np.outer(k, k) / n)
        assert np.abs(x @ Wm.T - ref).max() < 1e-11 * np.abs(ref).max()
    d = torch.as_tensor(x).cuda()
    qhp.qhp_fft_c2c(d, -1)
    out = d.cpu().numpy()
    assert np.abs(out - ref).max() < 1e-12 * np.abs(ref).max()
    # Parseval and inverse
    assert abs((np.abs(out) ** 2).sum() / n - (np.abs(x) ** 2).sum()) < 1e-12 * (np.abs(x) ** 2).sum()
    qhp.qhp_fft_c2c(d, +1)
    assert np.abs(d.cpu().numpy() / n - x).max() < 1e-12 * np.abs(x).max()
