"""Pins for the oracle's counter-based randomness (R-15).

Philox4x32-10 is pinned against an implementation that is not ours: cuRAND's HOST generator
(libcurand, runs on the CPU) -- `curandGenerate` with seed s and offset 4n returns block n of the
stream keyed by s.  Normals/uniforms are pinned by exact identities and sample moments.
"""
import ctypes as C
import math

import numpy as np
import pytest


def _curand_block(seed, n):
    cr = C.CDLL("libcurand.so.10")
    gen = C.c_void_p()
    assert cr.curandCreateGeneratorHost(C.byref(gen), 161) == 0      # CURAND_RNG_PSEUDO_PHILOX4_32_10
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    assert cr.curandSetGeneratorOffset(gen, C.c_ulonglong(4 * n)) == 0
    out = np.zeros(4, np.uint32)
    assert cr.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(4)) == 0
    cr.curandDestroyGenerator(gen)
    return out


@pytest.mark.parametrize("seed", [0, 1, 3005, 0x0123456789ABCDEF, 2**64 - 1])
@pytest.mark.parametrize("n", [0, 1, 2, 77, 65535, 65536, 65537, 2**32 + 5, 2**48 - 1, 2**48 + 3 * 65536 + 9,
                               2**60 + 12345678901])
def test_philox_matches_curand_host(orc, seed, n):
    hi = n >> 16
    ours = orc.philox([hi & 0xFFFFFFFF, hi >> 32, n & 0xFFFF, 0], [seed & 0xFFFFFFFF, seed >> 32])
    assert np.array_equal(ours, _curand_block(seed, n))


def test_philox_all_counter_words_matter(orc):
    base = orc.philox([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] += 1
        assert not np.array_equal(base, orc.philox(c, [5, 6]))
    assert not np.array_equal(base, orc.philox([1, 2, 3, 4], [5, 7]))


def test_uniform_is_word_of_block(orc):
    seed, c1, c2, c3 = 42, 7, 3, orc.tag(5, 2, 2)
    for n in (0, 1, 2, 3, 4, 9, 1023):
        w = orc.philox([n // 4, c1, c2, c3], [seed, 0])[n % 4]
        u = orc.uniform(seed, c1, c2, c3, n)
        assert u == ((int(w) >> 9) + 0.5) / 2**23
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u          # exact in fp32


def test_box_muller_identities(orc):
    seed, c1, c2, c3 = 9, 1, 1, orc.tag(5, 1, 2)
    for blk in range(50):
        z = [orc.normal(seed, c1, c2, c3, 4 * blk + l) for l in range(4)]
        u = [orc.uniform(seed, c1, c2, c3, 4 * blk + l) for l in range(4)]
        assert math.isclose(z[0] ** 2 + z[1] ** 2, -2 * math.log(u[0]), rel_tol=1e-12)
        assert math.isclose(z[2] ** 2 + z[3] ** 2, -2 * math.log(u[2]), rel_tol=1e-12)
        assert math.isclose(math.atan2(z[1], z[0]) % (2 * math.pi), 2 * math.pi * u[1], rel_tol=1e-9, abs_tol=1e-12)
        assert math.isclose(math.atan2(z[3], z[2]) % (2 * math.pi), 2 * math.pi * u[3], rel_tol=1e-9, abs_tol=1e-12)


def test_normal_moments(orc):
    n = 200_000
    z = np.array([orc.normal(123, 5, 2, orc.tag(5, 1, 2), i) for i in range(n)])
    assert abs(z.mean()) < 4 / math.sqrt(n)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((z ** 3).mean()) < 4 * math.sqrt(15 / n)
    assert abs((z ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 4 / math.sqrt(n)


def test_noise_is_keyed_structurally(orc):
    from paper_2606_26164_b200 import inputs
    wl = inputs.config(2, N=8)
    o = orc.Oracle(wl)
    a = o.noise(1, 3, 1, 2, 5)
    assert a == o.noise(1, 3, 1, 2, 5)
    others = [o.noise(2, 3, 1, 2, 5), o.noise(1, 4, 1, 2, 5), o.noise(1, 3, 6, 2, 5), o.noise(1, 3, 1, 3, 5),
              o.noise(1, 3, 1, 2, 6)]
    assert all(b != a for b in others)
    z = np.array([o.noise(1, i, 1, 1, s) for i in range(200) for s in range(50)]) / wl.obj.sigma_noise
    assert abs(z.mean()) < 0.04 and abs(z.std() - 1) < 0.03
    wl0 = inputs.config(1, N=8)
    assert orc.Oracle(wl0).noise(1, 0, 1, 1, 0) == 0.0
