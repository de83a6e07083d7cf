"""Pins for O6 (Philox4x32-10 + Box-Muller normals)."""
import numpy as np

import oracle as O
from helpers import read_golden


def test_philox_known_answer_vectors():
    for row in read_golden("philox4x32_10_kat.txt"):
        v = [int(s, 16) for s in row]
        out = O.philox4x32_10(v[0:4], v[4:6])
        assert [int(o) for o in out] == v[6:10]


def test_counter_layout_and_box_muller():
    # counter = (atom, mode | tag<<24, step_lo, step_hi); key = (seed_lo, seed_hi)
    seed, atom, mode, tag, step = 0x1234567890ABCDEF, 77, 5, 3, (3 << 32) + 9
    w = O.philox4x32_10([atom, mode | (tag << 24), step & 0xFFFFFFFF, step >> 32],
                        [seed & 0xFFFFFFFF, seed >> 32]).astype(np.float64)
    u = (w + 0.5) / 2.0 ** 32
    z = O.normals3(seed, atom, mode, tag, step)
    ref = [np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]),
           np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
           np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3])]
    assert np.allclose(z, ref, rtol=0, atol=1e-14)


def test_normals_moments():
    z = np.array([O.normals3(42, a, 0, 4, s) for a in range(40) for s in range(500)]).ravel()
    n = z.size                                   # 60000
    assert abs(z.mean()) < 5 / np.sqrt(n)
    assert abs(z.var() - 1) < 5 * np.sqrt(2 / n)
    assert abs((z ** 4).mean() - 3) < 5 * np.sqrt(96 / n)
    # the three components of one call are uncorrelated
    zz = z.reshape(-1, 3)
    c = np.corrcoef(zz.T)
    assert np.abs(c - np.eye(3)).max() < 5 / np.sqrt(n / 3)
