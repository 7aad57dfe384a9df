"""Pins of the oracle's structure-factor sums and second-moment correlation length
(Eq. 8-9; O9 / reading G21)."""
import math

import numpy as np
import pytest

import xy_inputs
from oracle import xy_oracle as xo
from golden_io import table1

TWO_PI = 2.0 * math.pi


def test_fourier_vs_numpy_fft():
    """sum_r s(r) e^{ikr} at k = (2pi/L, 0) and (0, 2pi/L) is one bin of numpy's FFT of the spin field."""
    L = 48
    th = xy_inputs.random_angles(L, 3)
    F = xo.fourier(th, L)
    t = th.astype(np.float64).reshape(L, L)                 # [y, x]
    for field, f_x, f_y in ((np.cos(t), F[0:2], F[4:6]), (np.sin(t), F[2:4], F[6:8])):
        ft = np.fft.fft2(field)                             # sum f e^{-i(ky y + kx x)}
        zx, zy = np.conj(ft[0, 1]), np.conj(ft[1, 0])       # e^{+ikx}: conjugate of a real field's bin
        assert abs(f_x[0] - zx.real) < 1e-9 and abs(f_x[1] - zx.imag) < 1e-9
        assert abs(f_y[0] - zy.real) < 1e-9 and abs(f_y[1] - zy.imag) < 1e-9


def test_fourier_closed_forms():
    L = 32
    N = L * L
    x = np.tile(np.arange(L), L)
    y = np.repeat(np.arange(L), L)
    # plane wave along x: theta = 2 pi x / L  ->  (N/2, 0, 0, N/2) along x, nothing along y
    F = xo.fourier((TWO_PI * x / L).astype(np.float32), L)
    assert np.allclose(F[:4], [N / 2, 0, 0, N / 2], atol=1e-4) and np.allclose(F[4:], 0, atol=1e-4)
    assert abs(xo.sk(F[:4], L) - N / 2) < 1e-3
    # plane wave along y: the transposed statement (a swapped x / y in the oracle fails here)
    F = xo.fourier((TWO_PI * y / L).astype(np.float32), L)
    assert np.allclose(F[4:], [N / 2, 0, 0, N / 2], atol=1e-4) and np.allclose(F[:4], 0, atol=1e-4)
    # opposite chirality flips the sign of the sin-sin term only
    F = xo.fourier(((TWO_PI * (L - x) / L) % TWO_PI).astype(np.float32), L)
    assert np.allclose(F[:4], [N / 2, 0, 0, -N / 2], atol=1e-4)
    # uniform field: sum_x e^{ikx} = 0
    F = xo.fourier(np.full(N, 1.25, np.float32), L)
    assert np.allclose(F, 0, atol=1e-9)


def test_xi2nd_inverts_ornstein_zernike():
    """Eq. 8 is built so that chi(k) = chi0 / (1 + xi^2 4 sin^2(k/2)) at k = 2pi/L returns xi exactly."""
    for L in (64, 1024):
        for xi in (3.0, 0.75 * L):
            chi0 = 17.0
            chik = chi0 / (1.0 + xi * xi * 4.0 * math.sin(math.pi / L) ** 2)
            assert xo.xi2nd(chi0, chik, L) == pytest.approx(xi, rel=1e-12)


def test_xi2nd_over_L_paper_table1_row_64():
    """PAPER.md:82 (Table I, L = 64): xi_2nd/L = 0.7464(11) at beta_KT(64) = 1.09167."""
    row = table1()[64]
    beta, want, err = row["beta"], row["xi"], row["xi_err"]
    L, seed = 64, 4
    N = L * L
    th = xo.init(L, seed, xo.INIT_HOT)
    xo.run(th, L, seed, 0, beta, 2000, series=False)        # thermalise
    chi0, chik, n, t = 0.0, 0.0, 12000, 2000
    for _ in range(n):
        o = xo.run(th, L, seed, t, beta, 1, series=True)[-1]
        t += 1
        F = xo.fourier(th, L)
        chi0 += (o["Mx"] ** 2 + o["My"] ** 2) / N
        chik += 0.5 * (xo.sk(F[:4], L) + xo.sk(F[4:], L))
    got = xo.xi2nd(chi0 / n, chik / n, L) / L
    # beta_KT(64) itself carries +-0.00025 -> d(xi/L) ~ 0.002; statistical error of 12000 sweeps ~ 0.004
    assert abs(got - want) < 5 * err + 0.012, (got, want)
