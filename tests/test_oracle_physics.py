"""Physics pins for the whole oracle sweep: limits with closed forms and the paper's own numbers."""
import math

import numpy as np

from golden_io import constants, table1
from oracle import xy_oracle as xo


def _binned_err(x, nb=40):
    m = x.size // nb
    b = x[: m * nb].reshape(nb, m).mean(axis=1)
    return b.std(ddof=1) / math.sqrt(nb)


def test_beta_zero_exact():
    """beta = 0: no bonds, every site its own cluster, ~half the sites reflected, E/N ~ 0."""
    L, N = 64, 4096
    th = xo.init(L, 2, xo.INIT_HOT)
    before = th.copy()
    b, lab, o = xo.sweep(th, L, seed=2, t=0, beta=0.0)
    assert b.sum() == 0 and (lab == np.arange(N)).all() and o.n_clusters == N
    nflip = (th != before).sum()
    assert abs(nflip - N / 2) < 4.5 * math.sqrt(N / 4)
    ser = xo.run(th, L, 2, 1, 0.0, 300)
    assert np.abs(ser["E"] / N).max() < 5 / math.sqrt(N)


def test_high_temperature_energy():
    """small beta: <cos> per link = beta/2 + O(beta^3), two links per site: E/N = -beta."""
    L, N, beta = 32, 1024, 0.05
    th = xo.init(L, 4, xo.INIT_HOT)
    xo.run(th, L, 4, 0, beta, 200, series=False)
    ser = xo.run(th, L, 4, 200, beta, 20000)
    e = ser["E"] / N
    assert abs(e.mean() + beta) < 4.5 * _binned_err(e) + 2 * beta ** 3


def test_low_temperature_spin_wave():
    """T = 0.05 from a cold start: harmonic equipartition E/N = -2 + (T/2)(1 - 1/N) (N-1 modes),
    anharmonic corrections O(T^2); helicity modulus Y_x = 1 - T/4 + O(T^2)."""
    L, N, beta = 32, 1024, 20.0
    T = 1 / beta
    th = xo.init(L, 6, xo.INIT_COLD)
    xo.run(th, L, 6, 0, beta, 2000, series=False)
    ser = xo.run(th, L, 6, 2000, beta, 15000)
    e = ser["E"] / N
    want = -2 + T / 2 * (1 - 1 / N)
    assert abs(e.mean() - want) < 4.5 * _binned_err(e) + T * T / 8
    for c, s in (("Cx", "Sx"), ("Cy", "Sy")):
        Y = (ser[c] / N).mean() - beta * N * ((ser[s] / N) ** 2).mean()
        assert abs(Y - (1 - T / 4)) < 0.01


def test_paper_table1_L64():
    """Table I row L=64: at beta_KT(64) = 1.09167 the paper has <m^2> = 0.34924(29)
    and, by construction of its PCC run, beta*Y = 0.636508."""
    row = table1()[64]
    crit = constants()["betaY_critical"]
    L, N, beta = 64, 4096, row["beta"]
    th = xo.init(L, 8, xo.INIT_HOT)
    xo.run(th, L, 8, 0, beta, 1500, series=False)
    ser = xo.run(th, L, 8, 1500, beta, 20000)
    m2 = (ser["Mx"] ** 2 + ser["My"] ** 2) / N ** 2
    err = _binned_err(m2)
    assert abs(m2.mean() - row["m2"]) < 4.5 * math.hypot(err, row["m2_err"]), (m2.mean(), err)
    # helicity modulus in x and y (jackknife over bins for the error)
    for c, s in (("Cx", "Sx"), ("Cy", "Sy")):
        e = ser[c] / N
        s2 = (ser[s] / N) ** 2
        bY = beta * (e.mean() - beta * N * s2.mean())
        nb = 40
        m = e.size // nb
        eb = e[: m * nb].reshape(nb, m).mean(axis=1)
        sb = s2[: m * nb].reshape(nb, m).mean(axis=1)
        jk = beta * (((eb.sum() - eb) / (nb - 1)) - beta * N * ((sb.sum() - sb) / (nb - 1)))
        jerr = math.sqrt((nb - 1) / nb * ((jk - jk.mean()) ** 2).sum())
        assert abs(bY - crit) < 4.5 * jerr + 0.002, (bY, jerr)


def test_helicity_brackets_the_jump():
    """beta*Y is well below 2/pi in the disordered phase and well above it at low T."""
    L, N = 32, 1024
    out = {}
    for beta in (0.8, 1.5):
        th = xo.init(L, 10, xo.INIT_HOT)
        xo.run(th, L, 10, 0, beta, 500, series=False)
        ser = xo.run(th, L, 10, 500, beta, 4000)
        out[beta] = beta * ((ser["Cx"] / N).mean() - beta * N * ((ser["Sx"] / N) ** 2).mean())
    assert out[0.8] < 0.45 < 2 / math.pi < 0.9 < out[1.5]


def test_determinism_and_chaining():
    L = 32
    a = xo.init(L, 5, xo.INIT_HOT)
    b = a.copy()
    xo.run(a, L, 5, 0, 1.1, 20, series=False)
    for t in range(20):
        xo.sweep(b, L, 5, t, 1.1)
    assert (a == b).all()
    c = xo.init(L, 5, xo.INIT_HOT)
    xo.run(c, L, 5, 0, 1.1, 12, series=False)
    xo.run(c, L, 5, 12, 1.1, 8, series=False)          # resume from (theta, t)
    assert (a == c).all()
