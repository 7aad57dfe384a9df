"""The whole sweep is a correct Markov kernel for exp(-beta H), H of Eq. 3:
exact detailed balance on the 2x2 torus, and the Ising limit on 4x4 against exact enumeration."""
import itertools
import math

import numpy as np
import pytest

from oracle import xy_oracle as xo

TWO_PI = 6.283185307179586
PI = 3.141592653589793


def _clock_setup(q):
    """angles on the q-gon; directions phi_m = pi m/q - pi/2 map the q-gon to itself:
    theta' = 2 phi + pi - theta = 2 pi (m - k)/q."""
    ang = np.array([np.float32(TWO_PI * k / q) for k in range(q)], np.float32)
    phis = [PI * m / q - PI / 2 for m in range(q)]
    return ang, phis


def _nearest_state(theta, q):
    return int(round(float(theta) * q / TWO_PI)) % q


def _transition_matrix(q, beta):
    L, N = 2, 4
    ang, phis = _clock_setup(q)
    nstates = q ** N
    states = np.array(list(itertools.product(range(q), repeat=N)), np.int64)   # [s, site]
    powers = q ** np.arange(N - 1, -1, -1)
    idx = np.arange(N)
    x, y = idx % L, idx // L
    nbr = np.stack([y * L + (x + 1) % L, ((y + 1) % L) * L + x], axis=1)
    # everything below comes from the oracle's pure functions
    ptab = np.zeros((q, q, q))                       # [m, ki, kj] bond probability
    rtab = np.zeros((q, q), np.int64)                # [m, k] reflected state
    for m, ph in enumerate(phis):
        A = xo.reflect_const(ph)
        for ki in range(q):
            t2 = xo.reflect(ang[ki], A)
            rtab[m, ki] = _nearest_state(t2, q)
            assert abs(((float(t2) - TWO_PI * rtab[m, ki] / q + PI) % TWO_PI) - PI) < 1e-6
            for kj in range(q):
                p = xo.bond_prob(beta, xo.sigma(ang[ki], ph), xo.sigma(ang[kj], ph))
                ptab[m, ki, kj] = min(max(p, 0.0), 1.0)      # "u < p" with u uniform on (0,1)
    labels = {}
    for bs in range(1 << (2 * N)):
        b = np.array([(bs >> (2 * i)) & 3 for i in range(N)], np.uint8)
        labels[bs] = xo.label(b, L)[0]
    P = np.zeros((nstates, nstates))
    for m in range(q):
        pb = np.stack([ptab[m, states[:, i], states[:, nbr[i, d]]] for i in range(N) for d in range(2)], axis=1)
        for bs in range(1 << (2 * N)):
            on = np.array([(bs >> k) & 1 for k in range(2 * N)], bool)
            w = np.prod(np.where(on, pb, 1.0 - pb), axis=1)
            if not (w > 0).any():
                continue
            lab = labels[bs]
            roots = np.unique(lab)
            for flips in itertools.product((0, 1), repeat=roots.size):
                fl = dict(zip(roots.tolist(), flips))
                new = states.copy()
                for i in range(N):
                    if fl[int(lab[i])]:
                        new[:, i] = rtab[m, states[:, i]]
                np.add.at(P, (np.arange(nstates), new @ powers), w / q / 2 ** roots.size)
    # Boltzmann weights, H = -sum over the 8 links of the 2x2 torus (each pair double-bonded)
    th = TWO_PI * states / q
    H = np.zeros(nstates)
    for i in range(N):
        for d in range(2):
            H -= np.cos(th[:, i] - th[:, nbr[i, d]])
    pi = np.exp(-beta * H)
    pi /= pi.sum()
    return P, pi, states, powers


@pytest.mark.parametrize("q,beta", [(4, 0.7), (4, 1.12), (6, 1.12)])
def test_detailed_balance_2x2(q, beta):
    P, pi, _, _ = _transition_matrix(q, beta)
    assert np.abs(P.sum(axis=1) - 1).max() < 1e-12
    flow = pi[:, None] * P
    # fp32 angles make the q-gon inexact at the 1e-7 level; a wrong formula breaks this at O(0.1)
    assert np.abs(flow - flow.T).max() < 2e-7
    assert np.abs(pi @ P - pi).max() < 2e-7
    assert (np.linalg.matrix_power(P, 64) > 0).all()       # ergodic on the q-gon states


def test_sweep_composition_matches_transition_row():
    """xyo_sweep itself (bonds -> label -> flip with the RNG) samples the row of P."""
    q, beta = 4, 1.12
    P, _, states, powers = _transition_matrix(q, beta)
    ang, phis = _clock_setup(q)
    for a in (5, 77, 200):
        counts = np.zeros(P.shape[0])
        n_per = 6000
        for m, ph in enumerate(phis):
            for rep in range(n_per):
                th = ang[states[a]].copy()
                xo.sweep(th, 2, seed=1000 + a, t=m * n_per + rep, beta=beta, fix_phi=ph)
                new = np.array([_nearest_state(v, q) for v in th])
                counts[new @ powers] += 1
        n = n_per * q
        exp = P[a] * n
        assert (counts[exp == 0] == 0).all()
        big = exp >= 5
        chi2 = ((counts[big] - exp[big]) ** 2 / exp[big]).sum()
        dof = big.sum() - 1
        assert chi2 < dof + 5 * math.sqrt(2 * dof) + 5, (a, chi2, dof)


def _ising_exact(Lq, beta):
    N = Lq * Lq
    s = ((np.arange(1 << N)[:, None] >> np.arange(N)) & 1) * 2 - 1
    s = s.reshape(-1, Lq, Lq)
    E = -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2)) - (s * np.roll(s, -1, axis=1)).sum(axis=(1, 2))
    M = s.sum(axis=(1, 2))
    w = np.exp(-beta * (E - E.min()))
    Z = w.sum()
    e1 = (w * E).sum() / Z
    e2 = (w * E * E).sum() / Z
    m2 = (w * M * M).sum() / Z
    return e1 / N, m2 / N ** 2, beta ** 2 * (e2 - e1 ** 2) / N


def _binned_err(x, nb=50):
    m = x.size // nb
    b = x[: m * nb].reshape(nb, m).mean(axis=1)
    return b.std(ddof=1) / math.sqrt(nb)


@pytest.mark.parametrize("beta", [0.2, 0.4407, 0.7])
def test_ising_limit_4x4(beta):
    """angles in {0, pi}, r fixed along x: sigma = +-1, p = 1 - exp(-2 beta) on parallel pairs:
    the 2D Ising SW algorithm.  <E>/N, <M^2>/N^2, specific heat vs all 2^16 states."""
    L, N, n = 4, 16, 150000
    th = (np.random.default_rng(3).integers(0, 2, N) * PI).astype(np.float32)
    xo.run(th, L, seed=77, t0=0, beta=beta, n=2000, fix_phi=0.0, series=False)
    ser = xo.run(th, L, seed=77, t0=2000, beta=beta, n=n, fix_phi=0.0)
    assert (np.abs(np.cos(th.astype(np.float64))) > 0.999999).all()     # still Ising states
    e = ser["E"] / N
    m2 = (ser["Mx"] / N) ** 2
    assert np.abs(ser["My"]).max() < 1e-3 and np.abs(ser["Sx"]).max() < 1e-3
    e_ex, m2_ex, c_ex = _ising_exact(L, beta)
    assert abs(e.mean() - e_ex) < 4.5 * _binned_err(e) + 1e-6
    assert abs(m2.mean() - m2_ex) < 4.5 * _binned_err(m2) + 1e-6
    e2 = (ser["E"] - ser["E"].mean()) ** 2 * beta ** 2 / N
    assert abs(e2.mean() - c_ex) < 5 * _binned_err(e2) + 1e-3 * c_ex
