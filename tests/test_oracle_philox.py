"""Pin P13: oracle Philox4x32-10 against cuRAND's host generator (a library routine) and
uniformity tests."""
import ctypes
import os

import numpy as np
import pytest

from oracle.philox import philox4x32_10, uniforms

_CURAND = "/usr/local/cuda/lib64/libcurand.so.10"


@pytest.mark.skipif(not os.path.exists(_CURAND), reason="libcurand not present")
@pytest.mark.parametrize("seed", [0, 1, 0x123456789ABCDEF, 0xFFFFFFFFFFFFFFFF, 0xDEADBEEFCAFEF00D])
def test_philox_matches_curand_host(seed):
    # cuRAND host PHILOX4_32_10, default ordering: output quad Q uses counter
    # (c0,c1) = Q // 65536 (64 bit), c2 = Q % 65536, c3 = 0, key = seed (found empirically, and
    # checked here for Q spanning c0, c1 and c2).
    lib = ctypes.CDLL(_CURAND)
    for Q0 in (0, 65536 * 3 - 8, (3 << 48) + 65536 * 9 + 11):
        gen = ctypes.c_void_p()
        assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(4 * Q0)) == 0
        out = np.zeros(64, dtype=np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(64)) == 0
        lib.curandDestroyGenerator(gen)
        q = [Q0 + i for i in range(16)]
        c01 = np.array([v // 65536 for v in q], dtype=np.uint64)
        c2 = np.array([v % 65536 for v in q], dtype=np.uint64)
        r = philox4x32_10(c01 & np.uint64(0xFFFFFFFF), c01 >> np.uint64(32), c2, 0 * c2,
                          seed & 0xFFFFFFFF, seed >> 32)
        mine = np.stack(r, axis=1).reshape(-1).astype(np.uint32)
        np.testing.assert_array_equal(mine, out)


def test_uniforms_layout_and_range():
    i = np.arange(1000, dtype=np.uint64) + np.uint64(1 << 33)
    u = uniforms(42, i, 3, 5)
    assert u.shape == (5, 1000) and (u >= 0).all() and (u < 1).all()
    # slot/stream layout: uniform e = slot e%2 of stream e//2; counter = (i_lo, i_hi, g, s)
    r = philox4x32_10(i & np.uint64(0xFFFFFFFF), i >> np.uint64(32), 0 * i + np.uint64(3), 0 * i + np.uint64(1), 42, 0)
    u2 = (((r[1] << np.uint64(32)) | r[0]) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    u3 = (((r[3] << np.uint64(32)) | r[2]) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    np.testing.assert_array_equal(u[2], u2)
    np.testing.assert_array_equal(u[3], u3)
    # different iteration / seed / stream decorrelate
    assert not np.array_equal(uniforms(42, i, 4, 1), uniforms(42, i, 3, 1))
    assert not np.array_equal(uniforms(43, i, 3, 1), uniforms(42, i, 3, 1))


def test_uniformity():
    u = uniforms(7, np.arange(1 << 18, dtype=np.uint64), 0, 4)
    for e in range(4):
        assert abs(u[e].mean() - 0.5) < 4 * (1 / 12 / (1 << 18)) ** 0.5
        assert abs(u[e].var() - 1 / 12) < 1e-3
        h = np.bincount((u[e] * 256).astype(int), minlength=256)
        chi2 = ((h - 1024.0) ** 2 / 1024.0).sum()
        assert 150 < chi2 < 380           # 255 dof
    assert abs(np.corrcoef(u[0], u[1])[0, 1]) < 0.01
