"""Pins of the q-state Potts oracle (readings P1-P5, oracle/xy_oracle.c).

H = -sum_<ij> delta(s_i, s_j).  What the mathematics fixes, independent of the oracle's own code:
exact Boltzmann distribution of the 2x2 torus (q = 3: 81 states) against the frequencies of the
oracle's sweep and its exact one-step transition matrix; the q = 2 model on 4x4 against the
enumeration of all 2^16 states; the bond rule's closed forms; uniformity of the fresh spins; the
energy at the self-dual point beta_c = ln(1 + sqrt q), where e = -(1 + 1/sqrt q) per site.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import xy_oracle as xo


def _energy(s, L):
    a = s.reshape(L, L)
    return -int((a == np.roll(a, -1, axis=1)).sum() + (a == np.roll(a, -1, axis=0)).sum())


def test_init_and_observe_against_numpy():
    L, q = 48, 5
    s = xo.potts_init(L, q, seed=9, kind=xo.INIT_HOT)
    assert s.max() < q and np.bincount(s, minlength=q).min() > L * L / q * 0.8
    # hot start restated: floor(q * w0 / 2^32) of the INIT call of the site
    for i in (0, 1, 777, L * L - 1):
        assert s[i] == (int(xo.rng(9, i, 0, xo.TAG_INIT)[0]) * q) >> 32
    o = xo.potts_observe(s, L)
    a = s.reshape(L, L)
    assert o.ex == (a == np.roll(a, -1, axis=1)).sum() and o.ey == (a == np.roll(a, -1, axis=0)).sum()
    assert o.E == _energy(s, L) and list(o.count)[:q] == np.bincount(s, minlength=q).tolist()
    assert (xo.potts_init(L, q, 9, xo.INIT_COLD) == 0).all()


def test_bond_rule_closed_forms():
    L, beta = 64, 0.8
    p = xo.potts_bond_prob(beta)
    assert abs(p - (1.0 - math.exp(-beta))) < 1e-15
    cold = np.zeros(L * L, np.uint8)
    b, nx, ny = xo.potts_bonds(cold, L, beta, seed=4, t=3)
    n = L * L
    for cnt, bit in ((nx, 1), (ny, 2)):
        assert cnt == ((b & bit) != 0).sum()
        assert abs(cnt - n * p) < 5 * math.sqrt(n * p * (1 - p))          # binomial density
    # a bond is exactly "equal spins and u < p" with the site's own uniforms
    s = xo.potts_init(L, 3, seed=4, kind=xo.INIT_HOT)
    b, _, _ = xo.potts_bonds(s, L, beta, seed=4, t=3)
    a = s.reshape(L, L)
    eqx = (a == np.roll(a, -1, axis=1)).ravel()
    eqy = (a == np.roll(a, -1, axis=0)).ravel()
    assert not (b[~eqx] & 1).any() and not (b[~eqy] & 2).any()
    import ctypes as C
    ux, uy = C.c_double(), C.c_double()
    for i in range(0, L * L, 97):
        xo._bond_u_site(4, 3, i, C.byref(ux), C.byref(uy))
        assert bool(b[i] & 1) == bool(eqx[i] and ux.value < p)
        assert bool(b[i] & 2) == bool(eqy[i] and uy.value < p)
    # beta = 0: no bonds at all; huge beta: every satisfied link is a bond
    assert not xo.potts_bonds(s, L, 0.0, 4, 3)[0].any()
    b, _, _ = xo.potts_bonds(s, L, 50.0, 4, 3)
    assert ((b & 1) != 0).sum() == eqx.sum() and ((b & 2) != 0).sum() == eqy.sum()
    # a 3-colouring with no equal neighbours has no bond whatever beta is
    x, y = np.meshgrid(np.arange(63), np.arange(63))
    chk = ((x + y) % 3).astype(np.uint8).ravel()
    assert not xo.potts_bonds(chk, 63, 50.0, 1, 0)[0].any()


def test_fresh_spins_uniform_constant_on_clusters():
    q, t, seed = 5, 11, 3
    draws = np.array([xo.potts_new_spin(seed, rho, t, q) for rho in range(40000)])
    exp = draws.size / q
    chi2 = ((np.bincount(draws, minlength=q) - exp) ** 2 / exp).sum()
    assert draws.max() < q and chi2 < (q - 1) + 5 * math.sqrt(2 * (q - 1)) + 5
    # restated from the definition: word rho & 3 of the POTTS call of rho >> 2
    for rho in (0, 5, 1023, 2 ** 33 + 7):
        w = xo.rng(seed, rho >> 2, t, xo.TAG_POTTS)
        assert xo.potts_new_spin(seed, rho, t, q) == (int(w[rho & 3]) * q) >> 32
    # consecutive labels are independent: lag-1 pairs fill the q x q table evenly
    pairs = np.bincount(draws[:-1] * q + draws[1:], minlength=q * q)
    e2 = (draws.size - 1) / q ** 2
    assert ((pairs - e2) ** 2 / e2).sum() < (q * q - 1) + 5 * math.sqrt(2 * (q * q - 1)) + 5
    L = 32
    s = xo.potts_init(L, q, seed, xo.INIT_HOT)
    b, lab, o = xo.potts_sweep(s, L, q, seed, t, 1.2)
    for rho in np.unique(lab)[:200]:
        assert (s[lab == rho] == xo.potts_new_spin(seed, int(rho), t, q)).all()
    assert o.n_clusters == np.unique(lab).size and o.E == _energy(s, L)


def _exact_2x2(q, beta):
    """Boltzmann weights and the exact one-step SW transition matrix of the 2x2 torus (double bonds),
    from the definition: bonds on equal pairs with probability p, fresh uniform spin per cluster."""
    L, N = 2, 4
    p = 1.0 - math.exp(-beta)
    states = np.array(list(itertools.product(range(q), repeat=N)), np.int64)
    powers = q ** np.arange(N - 1, -1, -1)
    idx = np.arange(N)
    x, y = idx % L, idx // L
    nbr = np.stack([y * L + (x + 1) % L, ((y + 1) % L) * L + x], axis=1)
    H = np.zeros(len(states))
    for i in range(N):
        for d in range(2):
            H -= states[:, i] == states[:, nbr[i, d]]
    pi = np.exp(-beta * H)
    pi /= pi.sum()
    P = np.zeros((len(states), len(states)))
    for a, st in enumerate(states):
        links = [(i, nbr[i, d]) for i in range(N) for d in range(2)]
        for bs in range(1 << len(links)):
            w = 1.0
            par = list(range(N))

            def find(u):
                while par[u] != u:
                    u = par[u]
                return u
            for k, (i, j) in enumerate(links):
                on = (bs >> k) & 1
                if st[i] == st[j]:
                    w *= p if on else 1.0 - p
                elif on:
                    w = 0.0
                if on and w:
                    ri, rj = find(i), find(j)
                    if ri != rj:
                        par[max(ri, rj)] = min(ri, rj)
            if w == 0.0:
                continue
            roots = sorted({find(i) for i in range(N)})
            for new in itertools.product(range(q), repeat=len(roots)):
                m = dict(zip(roots, new))
                ns = np.array([m[find(i)] for i in range(N)])
                P[a, ns @ powers] += w / q ** len(roots)
    return P, pi, states, powers


def test_exact_kernel_2x2_is_reversible_for_boltzmann():
    P, pi, _, _ = _exact_2x2(3, 0.9)
    assert np.abs(P.sum(axis=1) - 1).max() < 1e-12
    flow = pi[:, None] * P
    assert np.abs(flow - flow.T).max() < 1e-14 and np.abs(pi @ P - pi).max() < 1e-14


def test_sweep_samples_transition_row_and_boltzmann_2x2():
    q, beta, L = 3, 0.9, 2
    P, pi, states, powers = _exact_2x2(q, beta)
    for a in (0, 17, 50):                                   # rows of P
        counts = np.zeros(len(states))
        n = 20000
        for rep in range(n):
            s = states[a].astype(np.uint8).copy()
            xo.potts_sweep(s, L, q, seed=500 + a, t=rep, beta=beta)
            counts[s.astype(np.int64) @ powers] += 1
        exp = P[a] * n
        assert (counts[exp == 0] == 0).all()
        big = exp >= 5
        chi2 = ((counts[big] - exp[big]) ** 2 / exp[big]).sum()
        dof = big.sum() - 1
        assert chi2 < dof + 5 * math.sqrt(2 * dof) + 5, (a, chi2, dof)
    # the chain's long-run frequencies are the Boltzmann weights
    s = np.zeros(4, np.uint8)
    counts = np.zeros(len(states))
    n = 120000
    for t in range(n):
        xo.potts_sweep(s, L, q, seed=8, t=t, beta=beta)
        counts[s.astype(np.int64) @ powers] += 1
    # SW decorrelates in ~1 sweep on 2x2: chi-square with a modest allowance for autocorrelation
    exp = pi * n
    chi2 = ((counts - exp) ** 2 / exp).sum()
    dof = len(states) - 1
    assert chi2 < 1.5 * (dof + 5 * math.sqrt(2 * dof)), (chi2, dof)


def _potts2_exact_4x4(beta):
    N = 16
    s = ((np.arange(1 << N)[:, None] >> np.arange(N)) & 1).reshape(-1, 4, 4)
    E = -((s == np.roll(s, -1, axis=2)).sum(axis=(1, 2)) + (s == np.roll(s, -1, axis=1)).sum(axis=(1, 2)))
    n0 = (s == 0).sum(axis=(1, 2))
    w = np.exp(-beta * (E - E.min()))
    Z = w.sum()
    return (w * E).sum() / Z / N, (w * (2.0 * n0 / N - 1) ** 2).sum() / Z


@pytest.mark.parametrize("beta", [0.4, 0.8814, 1.4])
def test_q2_4x4_against_enumeration(beta):
    """q = 2 is the Ising model at K = beta / 2: <E>/N and <m^2> over all 2^16 states."""
    L, N, n = 4, 16, 60000
    s = xo.potts_init(L, 2, seed=2, kind=xo.INIT_HOT)
    e = np.empty(n)
    m2 = np.empty(n)
    for t in range(n + 1000):
        _, _, o = xo.potts_sweep(s, L, 2, seed=2, t=t, beta=beta)
        if t >= 1000:
            e[t - 1000] = o.E / N
            m2[t - 1000] = (2.0 * o.count[0] / N - 1) ** 2
    e_ex, m2_ex = _potts2_exact_4x4(beta)

    def err(x, nb=40):
        b = x[: x.size // nb * nb].reshape(nb, -1).mean(axis=1)
        return b.std(ddof=1) / math.sqrt(nb)
    assert abs(e.mean() - e_ex) < 4.5 * err(e) + 1e-6, (e.mean(), e_ex)
    assert abs(m2.mean() - m2_ex) < 4.5 * err(m2) + 1e-6, (m2.mean(), m2_ex)


def test_q3_energy_at_self_dual_point():
    """beta_c = ln(1 + sqrt q); e(beta_c) = -(1 + 1/sqrt q) per site in the infinite lattice (duality);
    finite-size shifts at L = 48 are below 2 %."""
    q, L = 3, 48
    beta_c = math.log(1 + math.sqrt(q))
    s = xo.potts_init(L, q, seed=6, kind=xo.INIT_HOT)
    es = []
    for t in range(700):
        _, _, o = xo.potts_sweep(s, L, q, seed=6, t=t, beta=beta_c)
        if t >= 200:
            es.append(o.E / (L * L))
    e_c = -(1 + 1 / math.sqrt(q))
    assert abs(np.mean(es) - e_c) < 0.03 * abs(e_c), (np.mean(es), e_c)
    # and the two limits: beta = 0 redraws every site (e = -2/q), large beta orders (e -> -2)
    s = xo.potts_init(L, q, 6, xo.INIT_HOT)
    _, _, o = xo.potts_sweep(s, L, q, 6, 0, 0.0)
    assert o.n_clusters == L * L and abs(o.E / (L * L) + 2 / q) < 0.06
    s = xo.potts_init(L, q, 6, xo.INIT_COLD)
    for t in range(20):
        _, _, o = xo.potts_sweep(s, L, q, 6, t, 6.0)
    assert o.E / (L * L) < -1.98
