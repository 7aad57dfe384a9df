"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

config 4 (L = 16384, cold start seed 13, beta = 1.11996): one sweep of a thermalising state, compared with
the oracle on everything the oracle can do at this size in about a minute: bond decisions of sampled
sites one by one (whole rows and columns including the periodic wrap and tile borders, plus random
sites), the FULL label array (the oracle's sequential union-find on the GPU's bond array), the FULL
flip (the oracle's coin and reflection on the GPU's labels), the counts, and the observables against
an independent numpy evaluation in fp64 (1e-9 N).

config 5 (L = 65536, hot start seed 17): the first rows of the lattice (labels are minimum indices, so
the labels of a prefix of rows point into that prefix): sampled bond decisions, and the properties
that fix a labeling at any size (every active bond joins equal labels, label <= index, roots are fixed
points), plus the flip of the prefix."""
import numpy as np
import pytest

from oracle import xy_oracle as xo

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def xy():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_6116_b200 as m
    return m


def check_bond_sites(sites, L, th, bonds, seed, t, beta, ph):
    """bond decisions of the given sites, one by one from the oracle's definition"""
    bad = 0
    for i in sites:
        i = int(i)
        y, x = divmod(i, L)
        ir = y * L + (x + 1) % L
        idn = ((y + 1) % L) * L + x
        if idn >= th.size or ir >= th.size:
            continue                                  # neighbour outside the fetched prefix
        ux, uy = xo.bond_uniforms_site(seed, t, i)
        si = xo.sigma(float(th[i]), ph)
        px = xo.bond_prob(beta, si, xo.sigma(float(th[ir]), ph))
        py = xo.bond_prob(beta, si, xo.sigma(float(th[idn]), ph))
        want = (1 if ux < px else 0) | (2 if uy < py else 0)
        if want != int(bonds[i]):
            # a decision may differ only where the fp64 margin is below 1e-12 (expected: never)
            assert min(abs(ux - px), abs(uy - py)) < 1e-12, (i, want, int(bonds[i]), ux - px, uy - py)
            bad += 1
    return bad


def test_cfg4_full_size_sweep(xy):
    L, seed, beta = 16384, 13, 1.11996
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_COLD)
    st.sw_sweeps(beta, 2)
    t = st.get_sweep()
    th0 = st.get_angles()
    st.sw_sweeps(beta, 1)
    bonds, labels, th1, rec = st.get_bonds(), st.get_labels(), st.get_angles(), st.measure()
    st.destroy()
    ph = xo.phi(seed, t)

    # bonds: sampled rows / columns / random sites, one by one
    rng = np.random.default_rng(5)
    rows = [0, 31, 32, 8191, L - 1]
    cols = [0, 127, 128, L - 1]
    sites = np.concatenate([np.arange(r * L, (r + 1) * L) for r in rows]
                           + [np.arange(c, N, L)[::4] for c in cols]
                           + [rng.integers(0, N, 20000)])
    assert check_bond_sites(sites, L, th0, bonds, seed, t, beta, ph) == 0
    nbx, nby = int((bonds & 1).sum()), int(((bonds >> 1) & 1).sum())
    assert (rec.n_bonds_x, rec.n_bonds_y) == (nbx, nby)

    # labels: the whole array against the oracle's union-find on the same bonds
    lab_ref, ncl = xo.label(bonds, L)
    assert np.array_equal(labels, lab_ref)
    assert rec.n_clusters == ncl
    del lab_ref

    # flip: the whole array, bit for bit
    th_ref = th0.copy()
    xo.flip(th_ref, L, labels, ph, seed, t)
    assert np.array_equal(th1.view(np.uint32), th_ref.view(np.uint32))
    del th_ref, labels, bonds, th0

    # observables of the state after the sweep: independent fp64 evaluation (numpy pairwise sums)
    a = th1.astype(np.float64).reshape(L, L)
    del th1
    assert abs(rec.Mx - np.cos(a).sum()) <= 1e-9 * N and abs(rec.My - np.sin(a).sum()) <= 1e-9 * N
    d = a - np.roll(a, -1, axis=1)
    cx, sx = np.cos(d).sum(), np.sin(d).sum()
    d = a - np.roll(a, -1, axis=0)
    cy, sy = np.cos(d).sum(), np.sin(d).sum()
    for got, want in ((rec.Cx, cx), (rec.Sx, sx), (rec.Cy, cy), (rec.Sy, sy), (rec.E, -(cx + cy))):
        assert abs(got - want) <= 1e-9 * N, (got, want)
    assert rec.sweep == t + 1 and rec.beta == beta


@pytest.mark.parametrize("flags", [0, 1])              # 1: labels held as 64-bit words (north_star: int64 from L = 65536)
def test_cfg5_prefix_rows(xy, flags):
    L, seed, beta, R = 65536, 17, 1.11996, 96
    n = R * L
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=flags)
    st.sw_sweeps(beta, 1)
    t = st.get_sweep()
    th0 = st.get_angles(n=n)
    st.sw_sweeps(beta, 1)
    bonds, labels, th1 = st.get_bonds(n), st.get_labels(n), st.get_angles(n=n)
    st.destroy()
    ph = xo.phi(seed, t)
    rng = np.random.default_rng(6)
    sites = np.concatenate([np.arange(0, L), np.arange(31 * L, 33 * L), rng.integers(0, (R - 1) * L, 20000)])
    assert check_bond_sites(sites, L, th0, bonds, seed, t, beta, ph) == 0

    lab = labels.reshape(R, L)
    b = bonds.reshape(R, L)
    idx = np.arange(n, dtype=np.int64).reshape(R, L)
    assert (lab <= idx).all() and (lab >= 0).all()                     # minimum index: never above the site's own
    assert np.array_equal(labels[labels], labels)                       # roots are fixed points (and lie in the prefix)
    bx, by = (b & 1).astype(bool), ((b >> 1) & 1).astype(bool)
    assert (lab[bx] == np.roll(lab, -1, axis=1)[bx]).all()              # every active x bond joins equal labels (wrap included)
    assert (lab[:-1][by[:-1]] == lab[1:][by[:-1]]).all()                # every active y bond inside the prefix
    # clusters that lie inside the prefix without touching its last row are exact components: compare the
    # partition with the oracle's labeling of the prefix taken as an open strip (periodic in x only)
    strip = bonds.copy().reshape(R, L)
    strip[R - 1, :] &= 1                                                 # cut the y bonds that leave the prefix
    # the oracle labels L x L lattices; embed the strip's first W columns as a W x W open window
    W = 64
    win = np.zeros((W, W), np.uint8)
    win[:, :] = strip[:W, :W]
    win[:, W - 1] &= 2
    win[W - 1, :] &= 1
    lab_w, _ = xo.label(win.reshape(-1), W)
    lab_w = lab_w.reshape(W, W)
    g = lab[:W, :W]
    # two window sites the oracle joins inside the window must carry equal GPU labels
    for r in np.unique(lab_w):
        m = lab_w == r
        assert np.unique(g[m]).size == 1

    # flip of the prefix: the oracle's coin on the GPU's labels; unflipped sites untouched, flipped ones
    # (a sample) reflected to the bit
    A = xo.reflect_const(ph)
    roots = np.unique(labels)
    coins = np.fromiter((xo.flip_coin(seed, int(r), t) for r in roots), dtype=np.uint8, count=roots.size)
    site_coin = coins[np.searchsorted(roots, labels)].astype(bool)
    assert np.array_equal(th1[~site_coin].view(np.uint32), th0[~site_coin].view(np.uint32))
    flipped = np.nonzero(site_coin)[0]
    samp = flipped[:: max(1, flipped.size // 100000)]
    want = np.array([xo.reflect(float(th0[i]), A) for i in samp], dtype=np.float32)
    assert np.array_equal(th1[samp].view(np.uint32), want.view(np.uint32))
