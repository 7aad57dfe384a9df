"""GPU parity of the q-state Potts sweep against the oracle, through the C-ABI:
spins, bonds, labels and all counts are integers, so everything is compared for equality."""
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


def _same_obs(g, o, q):
    assert (g.E, g.ex, g.ey) == (o.E, o.ex, o.ey)
    assert list(g.count)[:q] == list(o.count)[:q] and sum(list(g.count)[q:]) == 0
    assert (g.n_bonds_x, g.n_bonds_y, g.n_clusters) == (o.n_bonds_x, o.n_bonds_y, o.n_clusters)


@pytest.mark.parametrize("L,q,init,beta", [(64, 2, "hot", 0.8814), (128, 3, "hot", 1.005), (192, 3, "cold", 1.005),
                                           (256, 5, "hot", 1.2), (320, 16, "hot", 1.6), (384, 2, "cold", 0.5)])
def test_chained_sweeps_equal_the_oracle(xy, L, q, init, beta):
    kind = xy.INIT_HOT if init == "hot" else xy.INIT_COLD
    seed = 100 + L + q
    st = xy.PottsState(L, q, seed, kind)
    ref = xo.potts_init(L, q, seed, xo.INIT_HOT if init == "hot" else xo.INIT_COLD)
    assert (st.get_spins() == ref).all()
    g0 = st.measure()
    o0 = xo.potts_observe(ref, L)
    assert (g0.E, g0.ex, g0.ey, list(g0.count)[:q]) == (o0.E, o0.ex, o0.ey, list(o0.count)[:q])
    assert (g0.n_bonds_x, g0.n_clusters) == (0, 0)
    for t in range(12):
        st.sweeps(beta, 1)
        b, lab, o = xo.potts_sweep(ref, L, q, seed, t, beta)
        assert (st.get_bonds() == b).all(), f"bonds differ at sweep {t}"
        assert (st.get_labels() == lab).all(), f"labels differ at sweep {t}"
        assert (st.get_spins() == ref).all(), f"spins differ at sweep {t}"
        _same_obs(st.measure(), o, q)
        _same_obs(st.measure(), o, q)                     # a second measure returns the same record
    st.destroy()


def test_chain_of_n_equals_n_single_sweeps_and_resume(xy):
    L, q, seed, beta = 256, 3, 5, 1.005
    a = xy.PottsState(L, q, seed, xy.INIT_HOT)
    b = xy.PottsState(L, q, seed, xy.INIT_HOT)
    a.sweeps(beta, 40)
    for _ in range(25):
        b.sweeps(beta, 1)
    saved, T = b.get_spins(), b.get_sweep()
    b.destroy()
    c = xy.PottsState(L, q, seed + 99, xy.INIT_COLD)          # resume: spins + counter are the whole state
    c.set_spins(saved)
    c.destroy()
    c = xy.PottsState(L, q, seed, xy.INIT_COLD)
    c.set_spins(saved)
    c.set_sweep(T)
    c.sweeps(beta, 15)
    assert (a.get_spins() == c.get_spins()).all() and a.get_sweep() == c.get_sweep() == 40
    ref = xo.potts_init(L, q, seed, xo.INIT_HOT)
    for t in range(40):
        _, _, o = xo.potts_sweep(ref, L, q, seed, t, beta)
    assert (a.get_spins() == ref).all()
    _same_obs(a.measure(), o, q)
    a.destroy(); c.destroy()


@pytest.mark.parametrize("beta", [0.0, 1e-7, 3.0, 40.0, 1e9])
def test_threshold_extremes(xy, beta):
    """p = 0 (T = 0), p tiny (T >> 16 = 0: every decision with leading bits 0 needs the trailing ones), p near 1
    and p = 1 exactly (T = 2^32: the threshold does not fit 32 bits)."""
    L, q, seed = 128, 3, 77
    st = xy.PottsState(L, q, seed, xy.INIT_COLD)
    ref = xo.potts_init(L, q, seed, xo.INIT_COLD)
    for t in range(3):
        st.sweeps(beta, 1)
        b, lab, o = xo.potts_sweep(ref, L, q, seed, t, beta)
        assert (st.get_bonds() == b).all() and (st.get_labels() == lab).all() and (st.get_spins() == ref).all()
        _same_obs(st.measure(), o, q)
    st.destroy()


def test_trailing_bits_path_is_exercised(xy):
    """beta chosen so that T >> 16 is a value the 16 leading bits hit often enough at L = 1024: with 2^21
    decisions on equal pairs about 32 take the second Philox call; bonds must still equal the oracle's."""
    L, q, seed, beta = 1024, 2, 3, 0.7
    st = xy.PottsState(L, q, seed, xy.INIT_COLD)
    ref = xo.potts_init(L, q, seed, xo.INIT_COLD)
    st.sweeps(beta, 1)
    b, lab, o = xo.potts_sweep(ref, L, q, seed, 0, beta)
    assert (st.get_bonds() == b).all() and (st.get_labels() == lab).all() and (st.get_spins() == ref).all()
    # how many decisions of this sweep needed the trailing bits (restated from the definition of the uniforms)
    p = xo.potts_bond_prob(beta)
    import math
    T = math.ceil(p * 2.0 ** 32 - 0.5)
    n_open = 0
    for qd in range(L * L // 4):
        w = xo.rng(seed, qd, 0, xo.TAG_BOND)
        n_open += sum(int((int(x) & 0xffff) == T >> 16) + int((int(x) >> 16) == T >> 16) for x in w)
    assert n_open >= 5, n_open                            # ~32 expected: the second call was really needed
    _same_obs(st.measure(), o, q)
    st.destroy()


def test_error_codes(xy):
    with pytest.raises(xy.XYError):
        xy.PottsState(64, 1, 1)
    with pytest.raises(xy.XYError):
        xy.PottsState(64, 17, 1)
    with pytest.raises(xy.XYError):
        xy.PottsState(100, 3, 1)
    st = xy.PottsState(64, 3, 1, xy.INIT_COLD)
    with pytest.raises(xy.XYError):
        st.get_bonds()
    with pytest.raises(xy.XYError):
        st.sweeps(-1.0, 1)
    bad = np.zeros(64 * 64, np.uint8)
    bad[5] = 3
    with pytest.raises(xy.XYError):
        st.set_spins(bad)
    assert (st.get_spins() == 0).all()                    # rejected input left the state alone
    st.destroy()


def test_full_size_potts_sweep_invariants(xy):
    """L = 8192, q = 3 at the self-dual point, in the launch configuration the bench times: 30 sweeps, then the
    properties that hold at any size, checked on the host from the getters: bonds only on equal pairs, labels
    constant on bonds and pointing at roots with label <= index, spins constant on clusters, counts consistent."""
    L, q, seed, beta = 8192, 3, 12, 1.0050525
    st = xy.PottsState(L, q, seed, xy.INIT_HOT)
    st.sweeps(beta, 30)
    before = st.get_spins().reshape(L, L)
    st.sweeps(beta, 1)
    b = st.get_bonds().reshape(L, L)
    lab = st.get_labels().reshape(L, L)
    after = st.get_spins().reshape(L, L)
    bx, by = (b & 1) != 0, (b & 2) != 0
    assert (before == np.roll(before, -1, axis=1))[bx].all() and (before == np.roll(before, -1, axis=0))[by].all()
    assert (lab == np.roll(lab, -1, axis=1))[bx].all() and (lab == np.roll(lab, -1, axis=0))[by].all()
    flat = lab.ravel()
    idx = np.arange(L * L)
    assert (flat <= idx).all() and (flat[flat] == flat).all()
    assert (after.ravel() == after.ravel()[flat]).all()               # one spin per cluster
    roots = np.flatnonzero(flat == idx)
    sample = roots[:: max(1, roots.size // 500)]
    for rho in sample:                                                # and it is the oracle's draw for that label
        assert after.ravel()[rho] == xo.potts_new_spin(seed, int(rho), 30, q)
    o = st.measure()
    assert o.n_clusters == roots.size and o.n_bonds_x == bx.sum() and o.n_bonds_y == by.sum()
    assert o.ex == (after == np.roll(after, -1, axis=1)).sum() and list(o.count)[:q] == np.bincount(after.ravel(), minlength=q).tolist()
    st.destroy()
