"""Pins for the oracle's Philox4x32-10 and its uniform -> normal map (reading A11)."""
import numpy as np

from oracle import wl_oracle as o

# Known-answer vectors of Philox4x32-10 published with the Random123 library
# (Salmon, Moraes, Dror, Shaw, SC'11; file kat_vectors): counter, key -> output.
KAT = [
    ([0, 0, 0, 0], [0, 0],
     [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]),
    ([0xffffffff] * 4, [0xffffffff] * 2,
     [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]),
    ([0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344], [0xa4093822, 0x299f31d0],
     [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]),
]


def test_philox_known_answers():
    for ctr, key, want in KAT:
        assert o.philox4x32_10(ctr, key) == want


def test_philox_counter_and_key_sensitivity():
    base = o.philox4x32_10([1, 2, 3, 0], [7, 0])
    assert o.philox4x32_10([2, 2, 3, 0], [7, 0]) != base
    assert o.philox4x32_10([1, 2, 3, 0], [8, 0]) != base
    assert o.philox4x32_10([1, 2, 3, 0], [7, 0]) == base


def test_normal_pair_uses_counter_layout_and_box_muller():
    # Rebuild the pair from the raw Philox words with numpy: counter (point, loop_lo,
    # loop_hi, 0), key (seed_lo, seed_hi), 53-bit uniforms in (0,1], Box-Muller.
    seed, loop, point = (5 << 32) | 9, (3 << 32) | 11, 77
    w = o.philox4x32_10([point, loop & 0xffffffff, loop >> 32, 0], [seed & 0xffffffff, seed >> 32])
    u1 = (((w[1] << 32 | w[0]) >> 11) + 1) / 2.0 ** 53
    u2 = (((w[3] << 32 | w[2]) >> 11) + 1) / 2.0 ** 53
    r, th = np.sqrt(-2 * np.log(u1)), 2 * np.pi * u2
    nx, ny = o.normal_pair(seed, loop, point)
    assert abs(nx - r * np.cos(th)) < 1e-14 and abs(ny - r * np.sin(th)) < 1e-14


def test_normal_pair_moments():
    n = 40000
    z = np.array([o.normal_pair(123, l, 1) for l in range(n)])
    assert np.all(np.isfinite(z))
    se = 1 / np.sqrt(n)
    assert np.all(np.abs(z.mean(0)) < 5 * se)
    assert np.all(np.abs(z.var(0) - 1) < 5 * np.sqrt(2) * se)
    assert abs((z[:, 0] * z[:, 1]).mean()) < 5 * se
    assert np.all(np.abs((z ** 4).mean(0) - 3) < 5 * np.sqrt(96) * se)
