"""Pins for the oracle's RNG layer (O1-O3 of DESIGN.md section 3): Philox4x32-10 against
NVIDIA's own implementation, the keying convention, the hot start and the sweep direction."""
import ctypes

import numpy as np
import pytest

from oracle import xy_oracle as xo

TWO_PI = 6.283185307179586


def _shim_call(lib, ctr, key):
    c = np.ascontiguousarray(ctr, np.uint32)
    k = np.ascontiguousarray(key, np.uint32)
    out = np.zeros(4, np.uint32)
    lib.shim_curand_philox4x32_10(c.ctypes.data_as(ctypes.c_void_p), k.ctypes.data_as(ctypes.c_void_p),
                                  out.ctypes.data_as(ctypes.c_void_p))
    return out


def test_philox_matches_curand_header(curand_shim):
    """Independent implementation: cuRAND's curand_Philox4x32_10(uint4, uint2), host path."""
    rng = np.random.default_rng(2024)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xffffffff] * 4, [0xffffffff] * 2),
             ([1, 0, 0, 0], [0, 0]), ([0, 1, 0, 0], [0, 0]), ([0, 0, 1, 0], [0, 0]),
             ([0, 0, 0, 1], [0, 0]), ([0, 0, 0, 0], [1, 0]), ([0, 0, 0, 0], [0, 1])]
    for _ in range(20000):
        cases.append((rng.integers(0, 2 ** 32, 4, dtype=np.uint64), rng.integers(0, 2 ** 32, 2, dtype=np.uint64)))
    for ctr, key in cases:
        assert (xo.philox4x32_10(ctr, key) == _shim_call(curand_shim, ctr, key)).all()


def test_philox_matches_curand_host_generator():
    """Second independent route: libcurand's host generator CURAND_RNG_PSEUDO_PHILOX4_32_10.
    Its output order is out[4*(65536*c + s) + j] = Philox(ctr=(c,0,s,0), key=seed)[j]."""
    try:
        lib = ctypes.CDLL("libcurand.so")
    except OSError:
        try:
            lib = ctypes.CDLL("/usr/local/cuda/lib64/libcurand.so")
        except OSError:
            pytest.skip("libcurand not available")
    for seed in (0, 5, 0x123456789ABCDEF1):
        gen = ctypes.c_void_p()
        assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
        n = 4 * 65536 * 2
        out = np.zeros(n, np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(n)) == 0
        lib.curandDestroyGenerator(gen)
        key = [seed & 0xffffffff, seed >> 32]
        for c, s in ((0, 0), (0, 1), (0, 777), (0, 65535), (1, 0), (1, 4242)):
            mine = xo.philox4x32_10([c, 0, s, 0], key)
            base = 4 * (65536 * c + s)
            assert (out[base:base + 4] == mine).all(), (seed, c, s)


def test_philox_structure():
    """Each round is a bijection of the counter: distinct counters -> distinct outputs;
    every counter word and key word matters."""
    key = [0xDEADBEEF, 0x12345678]
    outs = {tuple(xo.philox4x32_10([c, 0, 0, 0], key)) for c in range(1 << 14)}
    assert len(outs) == 1 << 14
    base = tuple(xo.philox4x32_10([7, 7, 7, 7], key))
    for pos in range(4):
        ctr = [7, 7, 7, 7]
        ctr[pos] ^= 1
        assert tuple(xo.philox4x32_10(ctr, key)) != base
    for pos in range(2):
        k2 = list(key)
        k2[pos] ^= 1
        assert tuple(xo.philox4x32_10([7, 7, 7, 7], k2)) != base


def test_rng_keying_convention():
    """key = (seed lo, seed hi); counter = (idx lo, idx hi, (u32)t, tag)."""
    seed, idx, t = 0xA1B2C3D4E5F60718, 0x1_0000_0003, 123456
    for tag in range(4):
        want = xo.philox4x32_10([idx & 0xffffffff, idx >> 32, t, tag], [seed & 0xffffffff, seed >> 32])
        assert (xo.rng(seed, idx, t, tag) == want).all()
    assert len({tuple(xo.rng(seed, 5, 9, tag)) for tag in range(4)}) == 4


def test_uniform_exact_and_open_interval():
    assert xo.uniform(0) == 0.5 / 2 ** 32
    assert xo.uniform(0xffffffff) == (2 ** 32 - 0.5) / 2 ** 32 < 1.0
    assert xo.uniform(0x80000000) == 0.5 + 0.5 / 2 ** 32


def test_bond_uniform_pairing():
    """two Philox calls per quad of sites: call BOND holds the 16 leading bits of the quad's 8 uniforms,
    call BOND_LO the 16 trailing bits; site 4q+j takes word j (x: low halves, y: high halves)."""
    seed, t = 99, 17
    for i in (0, 1, 2, 3, 4, 4093, 4094, 4095, (1 << 32) + 6, (1 << 32) + 7):
        A = xo.rng(seed, i >> 2, t, xo.TAG_BOND)
        B = xo.rng(seed, i >> 2, t, xo.TAG_BOND_LO)
        ux, uy = xo.bond_uniforms_site(seed, t, i)
        j = i % 4
        wx = ((int(A[j]) & 0xffff) << 16) | (int(B[j]) & 0xffff)
        wy = (int(A[j]) & 0xffff0000) | (int(B[j]) >> 16)
        assert ux == (float(wx) + 0.5) / 2 ** 32 and uy == (float(wy) + 0.5) / 2 ** 32


def test_uniform_moments():
    """mean, variance and a 64-bin chi^2 of the bond uniforms over 2*10^5 draws."""
    seed = 3
    u = np.array([xo.bond_uniforms_site(seed, 0, i) for i in range(100000)]).ravel()
    n = u.size
    assert abs(u.mean() - 0.5) < 5 / np.sqrt(12 * n)
    assert abs(u.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    h, _ = np.histogram(u, bins=64, range=(0, 1))
    chi2 = ((h - n / 64) ** 2 / (n / 64)).sum()
    assert chi2 < 63 + 5 * np.sqrt(2 * 63)


def test_bond_uniforms_uncorrelated_within_quad():
    """the 8 uniforms of a quad come from two calls (leading / trailing halves): no correlation between
    the x and y uniform of a site, between neighbouring sites of a quad, or between quads."""
    seed, n = 5, 1 << 16
    u = np.array([xo.bond_uniforms_site(seed, 3, i) for i in range(n)]) - 0.5     # [n, 2]
    lim = 5.0 / 12.0 / np.sqrt(n)
    assert abs((u[:, 0] * u[:, 1]).mean()) < lim                                    # x vs y of a site
    for lag in (1, 2, 3, 4):
        assert abs((u[:-lag, 0] * u[lag:, 0]).mean()) < lim
        assert abs((u[:-lag, 1] * u[lag:, 1]).mean()) < lim
        assert abs((u[:-lag, 0] * u[lag:, 1]).mean()) < lim
    # leading and trailing halves of one uniform are independent: 16 x 16 coarse contingency
    w = np.floor((u[:, 0] + 0.5) * 2 ** 32).astype(np.uint64)
    hi, lo = (w >> 28) & 15, (w >> 12) & 15
    h = np.zeros((16, 16)); np.add.at(h, (hi.astype(int), lo.astype(int)), 1)
    chi2 = ((h - n / 256) ** 2 / (n / 256)).sum()
    assert chi2 < 255 + 5 * np.sqrt(2 * 255)


def test_hot_init():
    L, seed = 256, 1
    th = xo.init(L, seed, xo.INIT_HOT)
    N = L * L
    assert th.dtype == np.float32 and th.min() >= 0.0 and th.max() < TWO_PI
    # definition, re-derived from the raw words
    for i in (0, 1, 2, 12345, N - 1):
        w = xo.rng(seed, i, 0, xo.TAG_INIT)
        assert th[i] == np.float32(TWO_PI * ((int(w[0]) >> 8) / 2 ** 24))
    h, _ = np.histogram(th, bins=64, range=(0, TWO_PI))
    chi2 = ((h - N / 64) ** 2 / (N / 64)).sum()
    assert chi2 < 63 + 5 * np.sqrt(2 * 63)
    o = xo.observe(th, L)
    assert abs(o.E / N) < 4 / np.sqrt(N)          # 2N links, var 1/2 each -> sd = 1/sqrt(N)
    assert (xo.init(L, seed, xo.INIT_HOT) == th).all()
    assert (xo.init(L, seed + 1, xo.INIT_HOT) != th).mean() > 0.99


def test_cold_init():
    th = xo.init(64, 5, xo.INIT_COLD)
    assert (th == 0).all() and not np.signbit(th).any()
    o = xo.observe(th, 64)
    assert o.E == -2.0 * 64 * 64 and o.Mx == 64 * 64 and o.My == 0.0 and o.Sx == 0.0


def test_phi():
    seed = 11
    ph = np.array([xo.phi(seed, t) for t in range(20000)])
    assert ph.min() >= 0 and ph.max() < TWO_PI
    assert len(np.unique(ph)) > 19990
    h, _ = np.histogram(ph, bins=32, range=(0, TWO_PI))
    chi2 = ((h - ph.size / 32) ** 2 / (ph.size / 32)).sum()
    assert chi2 < 31 + 5 * np.sqrt(2 * 31)
    w = xo.rng(seed, 0, 77, xo.TAG_DIR)
    assert xo.phi(seed, 77) == TWO_PI * (int(w[0]) / 2 ** 32)
    assert xo.phi(seed, 77) == xo.phi(seed, 77) != xo.phi(seed + 1, 77)
