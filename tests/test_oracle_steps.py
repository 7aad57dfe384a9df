"""Pins for the single steps of the oracle: bond rule (O4), labels (O5), flip (O6), observables (O7)."""
import math
from collections import deque

import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import xy_inputs
from oracle import xy_oracle as xo

TWO_PI = 6.283185307179586
PI = 3.141592653589793


# ------------------------------------------------------------------ bonds (O4)
def test_bond_prob_closed_form_values():
    """p = 1 - exp(-2 beta sigma_i sigma_j), against mpmath-free exact arithmetic via math.exp."""
    for beta, si, sj in ((1.12, 1.0, 1.0), (0.5, 0.3, 0.9), (2.0, -0.4, -0.7), (1.0, 1e-9, 1e-9)):
        want = 1.0 - math.exp(-2.0 * beta * si * sj)
        got = xo.bond_prob(beta, si, sj)
        assert abs(got - want) <= 1e-15 + 1e-12 * abs(want)
    assert xo.bond_prob(1.0, 0.5, -0.5) < 0          # antiparallel -> p < 0 -> never active
    assert xo.bond_prob(0.0, 1.0, 1.0) == 0.0
    assert xo.bond_prob(1e9, 1.0, 1.0) == 1.0


def test_sigma_is_projection_on_r():
    rng = np.random.default_rng(0)
    for _ in range(200):
        th = np.float32(rng.uniform(0, TWO_PI))
        ph = rng.uniform(0, TWO_PI)
        want = math.cos(float(th)) * math.cos(ph) + math.sin(float(th)) * math.sin(ph)   # s . r
        assert abs(xo.sigma(th, ph) - want) < 1e-15


@pytest.mark.parametrize("beta,phi", [(1.12, 0.0), (0.7, 0.9), (1.3, 2.5)])
def test_bond_density_cold_lattice(beta, phi):
    """cold lattice, fixed phi: every sigma_i sigma_j = cos^2 phi, so the bond density is
    1 - exp(-2 beta cos^2 phi) within binomial error over 2N trials."""
    L = 128
    th = np.zeros(L * L, np.float32)
    b = xo.bonds(th, L, beta, phi, seed=42, t=3)
    p = 1.0 - math.exp(-2.0 * beta * math.cos(phi) ** 2)
    n = 2 * L * L
    k = int((b & 1).sum() + (b >> 1).sum())
    assert abs(k - n * p) < 4.5 * math.sqrt(n * p * (1 - p))
    # x and y separately
    for kk in ((b & 1).sum(), (b >> 1).sum()):
        assert abs(kk - n / 2 * p) < 4.5 * math.sqrt(n / 2 * p * (1 - p))


def test_bond_special_cases_exact():
    L = 32
    N = L * L
    cold = np.zeros(N, np.float32)
    assert xo.bonds(cold, L, 1.12, PI / 2, 1, 0).sum() == 0          # sigma ~ 6e-17: p ~ 1e-32 < min U
    assert xo.bonds(cold, L, 0.0, 0.3, 1, 0).sum() == 0              # beta = 0
    assert (xo.bonds(cold, L, 1e9, 0.0, 1, 0) == 3).all()            # beta huge: all 2N bonds
    y, x = np.mgrid[0:L, 0:L]
    checker = (((x + y) % 2) * PI).astype(np.float32).ravel()         # antiparallel neighbours
    assert xo.bonds(checker, L, 5.0, 0.0, 1, 0).sum() == 0
    stripes = ((x % 2) * PI).astype(np.float32).ravel()               # parallel along y only
    b = xo.bonds(stripes, L, 1e9, 0.0, 1, 0)
    assert (b == 2).all()


def test_bond_neighbour_convention_and_wrap():
    """bit0 couples (x,y)-(x+1 mod L,y); bit1 couples (x,y)-(x,y+1 mod L); site i = y*L+x."""
    L = 8
    N = L * L
    ux = np.full(N, 0.5)
    uy = np.full(N, 0.5)
    beta = 1e9                                    # active iff sigma_i sigma_j > 0
    th = np.zeros(N, np.float32)
    th[3 * L + 7] = np.float32(PI)                # site (x=7, y=3) antiparallel to all
    b = xo.bonds_from_u(th, L, beta, 0.0, ux, uy)
    want = np.full(N, 3, np.uint8)
    want[3 * L + 7] = 0                           # its own +x (wraps to x=0) and +y bonds
    want[3 * L + 6] &= ~np.uint8(1)               # left neighbour's x bond
    want[2 * L + 7] &= ~np.uint8(2)               # upper neighbour's y bond
    assert (b == want).all()
    th = np.zeros(N, np.float32)
    th[7 * L + 2] = np.float32(PI)                # bottom row: +y wraps to row 0
    b = xo.bonds_from_u(th, L, beta, 0.0, ux, uy)
    assert b[7 * L + 2] == 0 and b[6 * L + 2] == 1 and b[7 * L + 1] == 2 and b[0 * L + 2] == 3


def test_bond_decision_is_u_less_than_p_with_margins():
    L = 16
    th = xy_inputs.random_angles(L, 3)
    rng = np.random.default_rng(1)
    ux, uy = rng.random(L * L), rng.random(L * L)
    b, mx, my = xo.bonds_from_u(th, L, 1.12, 0.77, ux, uy, margins=True)
    assert ((b & 1) == (mx < 0)).all() and ((b >> 1) == (my < 0)).all()
    b2, mx2, my2 = xo.bonds(th, L, 1.12, 0.77, 5, 9, margins=True)
    for i in (0, 17, 255):
        assert xo.bond_margin(th, L, 1.12, 0.77, 5, 9, i, 0) == mx2[i]
        assert xo.bond_margin(th, L, 1.12, 0.77, 5, 9, i, 1) == my2[i]
    # the rng form equals the injected form fed with the rng's uniforms
    u = np.array([xo.bond_uniforms_site(5, 9, i) for i in range(L * L)])
    assert (xo.bonds_from_u(th, L, 1.12, 0.77, u[:, 0].copy(), u[:, 1].copy()) == b2).all()


# ------------------------------------------------------------------ labels (O5)
def _edges(b, L):
    idx = np.arange(L * L)
    x, y = idx % L, idx // L
    r = y * L + (x + 1) % L
    d = ((y + 1) % L) * L + x
    ex = (b & 1).astype(bool)
    ey = ((b >> 1) & 1).astype(bool)
    return np.concatenate([idx[ex], idx[ey]]), np.concatenate([r[ex], d[ey]])


def _labels_scipy(b, L):
    N = L * L
    src, dst = _edges(b, L)
    g = coo_matrix((np.ones(src.size, np.int8), (src, dst)), shape=(N, N))
    _, comp = connected_components(g, directed=False)
    mins = np.full(comp.max() + 1, N, np.int64)
    np.minimum.at(mins, comp, np.arange(N))
    return mins[comp]


def _labels_bfs(b, L):
    N = L * L
    adj = [[] for _ in range(N)]
    src, dst = _edges(b, L)
    for s, d in zip(src.tolist(), dst.tolist()):
        adj[s].append(d)
        adj[d].append(s)
    lab = [-1] * N
    for s in range(N):               # ascending: the seed of each flood fill is the minimum index
        if lab[s] >= 0:
            continue
        lab[s] = s
        q = deque([s])
        while q:
            u = q.popleft()
            for v in adj[u]:
                if lab[v] < 0:
                    lab[v] = s
                    q.append(v)
    return np.array(lab, np.int64)


def _check_invariants(b, lab, ncl, L):
    N = L * L
    idx = np.arange(N)
    assert (lab <= idx).all() and (lab[lab] == lab).all()
    src, dst = _edges(b, L)
    assert (lab[src] == lab[dst]).all()
    assert ncl == (lab == idx).sum()
    assert ncl >= N - src.size


@pytest.mark.parametrize("L", [2, 3, 4, 5, 8, 16])
def test_labels_vs_bfs_and_scipy_random(L):
    reps = 200 if L <= 8 else 60
    for dens in (0.1, 0.3, 0.5, 0.7, 0.9):
        for rep in range(reps):
            b = xy_inputs.random_bonds(L, dens, seed=1000 * L + rep)
            lab, ncl = xo.label(b, L)
            assert (lab == _labels_scipy(b, L)).all()
            if rep < 20:
                assert (lab == _labels_bfs(b, L)).all()
            _check_invariants(b, lab, ncl, L)


@pytest.mark.parametrize("L", [2, 3, 4, 8, 16, 64])
@pytest.mark.parametrize("kind", xy_inputs.BOND_PATTERNS)
def test_labels_patterns(L, kind):
    if kind == "checker_islands" and L % 2:
        pytest.skip("needs even L")
    b = xy_inputs.pattern_bonds(L, kind)
    lab, ncl = xo.label(b, L)
    assert (lab == _labels_scipy(b, L)).all()
    _check_invariants(b, lab, ncl, L)
    if kind in ("all_on", "serpentine", "comb"):
        assert ncl == 1 and (lab == 0).all()
    if kind == "all_off":
        assert ncl == L * L
    if kind == "h_stripes":
        assert ncl == L and (lab == (np.arange(L * L) // L) * L).all()
    if kind == "wrap_only":
        assert lab[L - 1] == 0 and lab[(L - 1) * L] == 0


def test_labels_exhaustive_small():
    """every one of the 2^(2N) bond sets for L = 2 (2^8) and L = 3 (2^18), against a vectorised
    min-label propagation written here."""
    for L in (2, 3):
        N = L * L
        nb = 2 * N
        sets = np.arange(1 << nb, dtype=np.int64)
        bits = ((sets[:, None] >> np.arange(nb)) & 1).astype(bool)     # bit 2i: x bond of i, 2i+1: y bond
        idx = np.arange(N)
        x, y = idx % L, idx // L
        nbr = np.stack([y * L + (x + 1) % L, ((y + 1) % L) * L + x], axis=1)   # [i, dir]
        lab = np.tile(idx, (sets.size, 1))
        for _ in range(N + 1):
            before = lab.copy()
            for i in range(N):
                for d in range(2):
                    j = nbr[i, d]
                    on = bits[:, 2 * i + d]
                    m = np.minimum(lab[:, i], lab[:, j])
                    lab[:, i] = np.where(on, m, lab[:, i])
                    lab[:, j] = np.where(on, m, lab[:, j])
            if (lab == before).all():
                break
        stride = 1 if L == 2 else 1
        for s in range(0, sets.size, stride):
            b = (bits[s, 0::2].astype(np.uint8) | (bits[s, 1::2].astype(np.uint8) << 1))
            got, _ = xo.label(b, L)
            assert (got == lab[s]).all(), (L, s)


# ------------------------------------------------------------------ flip (O6)
def test_reflection_identities():
    rng = np.random.default_rng(7)
    for _ in range(2000):
        ph = rng.uniform(0, TWO_PI)
        th = np.float32(rng.uniform(0, TWO_PI))
        A = xo.reflect_const(ph)
        assert 0.0 <= A < TWO_PI
        t2 = xo.reflect(th, A)
        assert 0.0 <= t2 <= np.float32(TWO_PI)
        # s -> s - 2 (s.r) r : component along r changes sign, component across r is kept
        assert abs(math.cos(t2 - ph) + math.cos(float(th) - ph)) < 1e-6
        assert abs(math.sin(t2 - ph) - math.sin(float(th) - ph)) < 1e-6
        sx, sy = math.cos(float(th)), math.sin(float(th))
        rx, ry = math.cos(ph), math.sin(ph)
        dot = sx * rx + sy * ry
        assert abs(math.cos(t2) - (sx - 2 * dot * rx)) < 1e-6
        assert abs(math.sin(t2) - (sy - 2 * dot * ry)) < 1e-6
        # involution up to fp32 rounding (compare mod 2pi)
        t3 = xo.reflect(t2, A)
        d = abs(float(t3) - float(th))
        assert min(d, TWO_PI - d) < 1e-6


def test_flip_sites_touches_only_flagged():
    th = xy_inputs.random_angles(16, 2)
    flag = (np.arange(256) % 3 == 0).astype(np.uint8)
    out = xo.flip_sites(th.copy(), 1.234, flag)
    assert (out[flag == 0] == th[flag == 0]).all()
    A = xo.reflect_const(1.234)
    assert all(out[i] == xo.reflect(th[i], A) for i in np.nonzero(flag)[0])


def test_flip_is_per_cluster_and_fair():
    L, seed, t, beta = 64, 21, 4, 1.12
    th = xy_inputs.smooth_angles(L, 5)
    ph = xo.phi(seed, t)
    b = xo.bonds(th, L, beta, ph, seed, t)
    lab, ncl = xo.label(b, L)
    sig_before = np.array([xo.sigma(v, ph) for v in th])
    # all sites of a cluster share sign(sigma)
    roots = np.unique(lab)
    for r in roots[:200]:
        s = np.sign(sig_before[lab == r])
        assert (s == s[0]).all() or (lab == r).sum() == 1
    th2 = th.copy()
    nflip = xo.flip(th2, L, lab, ph, seed, t)
    changed = th2 != th
    coin = np.array([xo.flip_coin(seed, r, t) for r in roots])
    flipped_roots = set(roots[coin == 1].tolist())
    want = np.array([l in flipped_roots for l in lab.tolist()])
    sig_after = np.array([xo.sigma(v, ph) for v in th2])
    assert np.allclose(sig_after[want], -sig_before[want], atol=1e-6)
    assert (th2[~want] == th[~want]).all()
    assert nflip == want.sum() and (changed <= want).all()
    # fair coin over many clusters
    coins = np.array([xo.flip_coin(seed, r, tt) for r in range(2000) for tt in range(10)])
    assert abs(coins.mean() - 0.5) < 4 * 0.5 / math.sqrt(coins.size)
    # one Philox call serves 128 consecutive labels: coin = bit (rho mod 128) of its 128-bit output
    for rho in (0, 1, 31, 32, 127, 128, 1234, 2**32 - 1, 2**32 + 77):
        w = xo.rng(seed, rho >> 7, t, xo.TAG_FLIP)
        assert xo.flip_coin(seed, rho, t) == (int(w[(rho >> 5) & 3]) >> (rho & 31)) & 1
    # neighbouring labels (same Philox call) are uncorrelated
    c = np.array([xo.flip_coin(seed, r, t) for r in range(1 << 14)], dtype=np.float64) - 0.5
    for lag in (1, 2, 32, 64, 127, 128):
        corr = 4.0 * (c[:-lag] * c[lag:]).mean()
        assert abs(corr) < 4.0 / math.sqrt(c.size - lag)


# ------------------------------------------------------------------ observables (O7)
def test_observe_vs_fsum():
    L = 24
    th = xy_inputs.random_angles(L, 9)
    o = xo.observe(th, L)
    t = th.astype(np.float64).reshape(L, L)
    tr = np.roll(t, -1, axis=1)       # right neighbour (x+1)
    td = np.roll(t, -1, axis=0)       # down neighbour (y+1)
    want = dict(Mx=math.fsum(np.cos(t).ravel()), My=math.fsum(np.sin(t).ravel()),
                Cx=math.fsum(np.cos(t - tr).ravel()), Sx=math.fsum(np.sin(t - tr).ravel()),
                Cy=math.fsum(np.cos(t - td).ravel()), Sy=math.fsum(np.sin(t - td).ravel()))
    for k, v in want.items():
        assert abs(getattr(o, k) - v) < 1e-11, k
    assert o.E == -(o.Cx + o.Cy)


def test_observe_direction_convention():
    """a uniform twist along x only shows up in Cx/Sx, along y only in Cy/Sy."""
    L = 16
    y, x = np.mgrid[0:L, 0:L]
    k = TWO_PI / L
    o = xo.observe((k * x).astype(np.float32).ravel(), L)
    N = L * L
    assert abs(o.Cx - N * math.cos(k)) < 1e-4 and abs(o.Sx + N * math.sin(k)) < 1e-4   # theta_i - theta_R = -k
    assert abs(o.Cy - N) < 1e-9 and abs(o.Sy) < 1e-9
    o = xo.observe((k * y).astype(np.float32).ravel(), L)
    assert abs(o.Cy - N * math.cos(k)) < 1e-4 and abs(o.Sy + N * math.sin(k)) < 1e-4
    assert abs(o.Cx - N) < 1e-9 and abs(o.Sx) < 1e-9
