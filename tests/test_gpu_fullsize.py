"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

config 4 (L = 16384, cold start seed 13, beta = 1.11996): one sweep compared with the oracle on everything
the oracle can do at this size in a minute or two, at t = 1, 2 (thermalising, near-ordered), 100, and at t = 500
and 1500 (the equilibrium-shaped state bench.py times: bond density 0.47, fractal clusters, the longest merge
chains): the bonds (at t = 500 ALL 5.4e8 decisions from the oracle's fp64 definition; at the other sweeps sampled
rows, columns and random sites one by one), the FULL label array (the oracle's sequential union-find on the bond array), the
FULL flip (the oracle's coin and reflection), the counts, and the observables against an independent numpy
evaluation in fp64 (1e-9 N).

config 5 (L = 65536, hot start seed 17), both label widths (north_star: int64 labels at this size): the
whole-lattice invariants of the labeling counted on the device (xy_debug_check_labels: label <= index, roots
are fixed points, every active bond joins equal labels, root count = cluster count), and bands of rows
fetched with the _range getters - the first rows, the last rows (y wrap to row 0), the rows around site
index 2^31, a tile-row boundary far from the origin: sampled bond decisions one by one, label invariants on
the band, and the flip (the oracle's coin of every label in the band, reflection to the bit).

L = 32768: full one-sweep parity (all bonds, all labels, all angles) - the largest size the oracle labels
in full on the GPU box's host memory."""
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


@pytest.mark.parametrize("t0", [1, 2, 100, 500, 1500])
def test_cfg4_full_size_sweep(xy, t0):
    L, seed, beta = 16384, 13, 1.11996
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_COLD)
    st.sw_sweeps(beta, t0)
    t = st.get_sweep()
    th0 = st.get_angles()
    st.sw_sweeps(beta, 1)
    bonds, labels, th1, rec = st.get_bonds(), st.get_labels(), st.get_angles(), st.measure()
    inv = st.debug_check_labels()
    st.destroy()
    ph = xo.phi(seed, t)
    assert (inv["label_above_index"], inv["root_not_fixed"], inv["x_bond_split"], inv["y_bond_split"]) == (0, 0, 0, 0)
    assert inv["n_roots"] == rec.n_clusters

    if t0 == 500:
        # every decision of the sweep from the oracle's definition
        b_ref = xo.bonds(th0, L, beta, ph, seed, t)
        if not np.array_equal(bonds, b_ref):
            bad = np.nonzero(bonds != b_ref)[0]
            assert check_bond_sites(bad[:1000], L, th0, bonds, seed, t, beta, ph) == 0 and bad.size <= 1000
        del b_ref
    else:
        rng = np.random.default_rng(5)
        rows = [0, 31, 32, 8191, L - 1]
        cols = [0, 127, 128, L - 1]
        sites = np.concatenate([np.arange(r * L, (r + 1) * L) for r in rows]
                               + [np.arange(c, N, L)[::4] for c in cols]
                               + [rng.integers(0, N, 20000)])
        assert check_bond_sites(sites, L, th0, bonds, seed, t, beta, ph) == 0
    nbx, nby = int((bonds & 1).sum()), int(((bonds >> 1) & 1).sum())
    assert (rec.n_bonds_x, rec.n_bonds_y) == (nbx, nby)
    if t0 >= 500:
        assert 0.40 < (nbx + nby) / (2 * N) < 0.55          # the equilibrium-shaped workload of bench.py

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


def check_band(st, L, seed, t, beta, ph, r0, R, th_prev_get, rng):
    """rows r0 .. r0+R-1 of the state after sweep t (angles before the sweep come from th_prev_get): sampled bond
    decisions, label invariants inside the band, the flip of the band"""
    first, n = r0 * L, R * L
    th0x = th_prev_get(first, n)                       # the band's rows plus the row below them
    th0 = th0x[:n]
    bonds, labels, th1 = st.get_bonds(n, first=first), st.get_labels(n, first=first), st.get_angles(n=n, first=first)
    # bond decisions: whole rows at the band's start, a tile-row border inside it, random sites; the neighbours of
    # the sampled sites must lie inside the band (the last row's y bonds need the row after the band)
    def sample(sites):
        bad = 0
        for i in sites:
            i = int(i)
            y, x = divmod(i, L)
            ir, idn = y * L + (x + 1) % L, (y + 1) * L + x
            ux, uy = xo.bond_uniforms_site(seed, t, first + i)
            si = xo.sigma(float(th0[i]), ph)
            px = xo.bond_prob(beta, si, xo.sigma(float(th0x[ir]), ph))
            py = xo.bond_prob(beta, si, xo.sigma(float(th0x[idn]), ph))
            want = (1 if ux < px else 0) | (2 if uy < py else 0)
            if want != int(bonds[i]):
                assert min(abs(ux - px), abs(uy - py)) < 1e-12, (first + i, want, int(bonds[i]))
                bad += 1
        return bad
    mid = (R // 2) * L
    sites = np.concatenate([np.arange(0, L, 3), np.arange(mid - L, mid + L, 5), rng.integers(0, (R - 1) * L, 8000)])
    assert sample(sites) == 0
    lab = labels.reshape(R, L)
    b = bonds.reshape(R, L)
    idx = first + np.arange(n, dtype=np.int64).reshape(R, L)
    assert (lab <= idx).all() and (lab >= 0).all()
    bx, by = (b & 1).astype(bool), ((b >> 1) & 1).astype(bool)
    assert (lab[bx] == np.roll(lab, -1, axis=1)[bx]).all()              # active x bonds (wrap in x included)
    assert (lab[:-1][by[:-1]] == lab[1:][by[:-1]]).all()                # active y bonds inside the band
    # flip: the oracle's coin of every label in the band; unflipped sites untouched, flipped ones reflected to the bit
    A = xo.reflect_const(ph)
    roots = np.unique(labels)
    coins = np.fromiter((xo.flip_coin(seed, int(r), t) for r in roots), dtype=np.uint8, count=roots.size)
    site_coin = coins[np.searchsorted(roots, labels)].astype(bool)
    assert np.array_equal(th1[~site_coin].view(np.uint32), th0[~site_coin].view(np.uint32))
    flipped = np.nonzero(site_coin)[0]
    samp = flipped[:: max(1, flipped.size // 50000)]
    want = np.array([xo.reflect(float(th0[i]), A) for i in samp], dtype=np.float32)
    assert np.array_equal(th1[samp].view(np.uint32), want.view(np.uint32))
    return lab, b


@pytest.mark.parametrize("flags", [1, 0])              # 1: labels held as 64-bit words (north_star: int64 from L = 65536)
def test_cfg5_bands_and_invariants(xy, flags):
    import torch
    L, seed, beta, R = 65536, 17, 1.11996, 64
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=flags)
    st.sw_sweeps(beta, 1)
    t = st.get_sweep()
    # the angles before the sweep under test stay on the device (17 GB): a torch copy of the theta region read back
    # through a second state is not available, so keep the bands we need
    bands = {"first": 0, "last": L - R, "2^31": 32768 - R // 2, "tile row 1250": 40000 - R // 2}
    prev = {k: st.get_angles(n=(R + 1) * L if r0 + R < L else R * L, first=r0 * L) for k, r0 in bands.items()}
    row0 = st.get_angles(n=L, first=0)
    st.sw_sweeps(beta, 1)
    rec = st.measure()
    inv = st.debug_check_labels()
    assert (inv["label_above_index"], inv["root_not_fixed"], inv["x_bond_split"], inv["y_bond_split"]) == (0, 0, 0, 0), inv
    assert inv["n_roots"] == rec.n_clusters
    assert 0.2 < rec.n_clusters / N < 0.6
    ph = xo.phi(seed, t)
    rng = np.random.default_rng(6)
    for name, r0 in bands.items():
        th_prev = prev[name]
        if r0 + R == L:                                   # the last band's y neighbours are row 0
            th_prev = np.concatenate([th_prev, row0])
        lab, b = check_band(st, L, seed, t, beta, ph, r0, R, lambda first, n, a=th_prev: a, rng)
        if name == "first":
            # labels are minimum indices: the labels of the first rows point into them, so roots are checkable here
            flat = lab.reshape(-1)
            assert np.array_equal(flat[flat], flat)
        if name == "last":
            # y wrap: an active y bond in row L-1 joins the label of row 0 below it
            lab0 = st.get_labels(L, first=0)
            by_last = ((b[R - 1] >> 1) & 1).astype(bool)
            assert by_last.any() and (lab[R - 1][by_last] == lab0[by_last]).all()
        if name == "2^31":
            assert (lab >= 0).all() and lab.max() >= 2 ** 31          # indices beyond 2^31 survive the label width
    st.destroy()
    torch.cuda.empty_cache()


def test_L32768_full_parity(xy):
    """one sweep from the hot start at L = 32768 (1.07e9 sites; u32 labels): ALL bonds from the oracle's definition,
    the FULL label array, the FULL flip.  About 25 GB of host memory."""
    L, seed, beta = 32768, 17, 1.11996
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_HOT)
    st.sw_sweeps(beta, 1)
    t = st.get_sweep()
    th0 = st.get_angles()
    st.sw_sweeps(beta, 1)
    bonds, rec = st.get_bonds(), st.measure()
    ph = xo.phi(seed, t)
    b_ref = xo.bonds(th0, L, beta, ph, seed, t)
    if not np.array_equal(bonds, b_ref):
        bad = np.nonzero(bonds != b_ref)[0]
        assert check_bond_sites(bad[:1000], L, th0, bonds, seed, t, beta, ph) == 0 and bad.size <= 1000
    del b_ref
    lab_ref, ncl = xo.label(bonds, L)
    labels = st.get_labels()
    assert np.array_equal(labels, lab_ref)
    assert rec.n_clusters == ncl
    del lab_ref
    xo.flip(th0, L, labels, ph, seed, t)
    del labels
    th1 = st.get_angles()
    st.destroy()
    assert np.array_equal(th1.view(np.uint32), th0.view(np.uint32))
