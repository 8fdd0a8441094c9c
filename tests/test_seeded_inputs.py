"""The shared seeded input generator (seeded_inputs/): recipe of SURVEY.md 8(d)."""
import ctypes

import numpy as np

import seeded_inputs as si


def test_splitmix64_known_vector():
    # first output of the reference splitmix64 stream seeded with 0 (published test vector)
    lib = ctypes.CDLL(si.build())
    lib.si_splitmix64.restype = ctypes.c_uint64
    lib.si_splitmix64.argtypes = [ctypes.c_uint64]
    assert lib.si_splitmix64(0) == 0xE220A8397B1DCDAF


def test_counter_based_offsets_and_determinism():
    sub = si.subseed(20241214, 3, si.WHICH_SWAP)
    g = si.gauss(sub, 1001)
    for off, n in ((0, 1), (1, 7), (500, 501), (999, 2)):
        np.testing.assert_array_equal(si.gauss(sub, n, offset=off), g[off:off + n])
    assert not np.array_equal(si.gauss(si.subseed(20241214, 4, si.WHICH_SWAP), 16), g[:16])
    assert not np.array_equal(si.gauss(si.subseed(20241214, 3, si.WHICH_A), 16), g[:16])


def test_box_muller_by_hand():
    # element 0/1 from the first two uniforms, retyped with python ints (recipe in gauss.c header)
    M = (1 << 64) - 1
    GOLD = 0x9E3779B97F4A7C15

    def mix(z):
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    sub = mix(((12345 ^ (2 << 8) ^ 1) + GOLD) & M)
    assert sub == si.subseed(12345, 2, 1)
    u = [((mix((sub + (k + 1) * GOLD) & M) >> 11) + 0.5) / 2.0 ** 53 for k in range(2)]
    r = np.sqrt(-2 * np.log(u[0]))
    z = si.gauss(sub, 2)
    np.testing.assert_allclose(z, [r * np.cos(2 * np.pi * u[1]), r * np.sin(2 * np.pi * u[1])], rtol=1e-14)


def test_moments():
    g = si.gauss(si.subseed(1, 0, 0), 1 << 20)
    assert abs(g.mean()) < 5e-3 and abs(g.std() - 1) < 5e-3
    assert abs(np.mean(g ** 4) - 3) < 0.05
    assert abs(np.corrcoef(g[:-1], g[1:])[0, 1]) < 5e-3
