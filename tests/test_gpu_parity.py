"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Contract (BASELINE.json north_star):
  bonds, labels  bit-exact (a bond may differ only where the oracle's |u - p| < 1e-12; counted,
                 expected 0)
  angles         <= 1e-6 rad (expected: 0 ulp, the reflection is specified to the rounding)
  observables    |gpu - oracle| <= 1e-9 * N for the signed sums, 1e-9 relative for E, Cx, Cy
  counts         equal
"""
import math

import numpy as np
import pytest

import xy_inputs
from oracle import xy_oracle as xo

pytestmark = pytest.mark.gpu

TWO_PI = 6.283185307179586


@pytest.fixture(scope="module")
def xy():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_6116_b200 as m
    return m


def ulp_diff(a, b):
    ia = a.view(np.int32).astype(np.int64)
    ib = b.view(np.int32).astype(np.int64)
    return np.abs(ia - ib)


def check_obs(g, o, N, where=""):
    """g: dict-like GPU record, o: oracle Obs"""
    for k in ("Mx", "My", "Sx", "Sy", "Cx", "Cy", "E"):
        gv, ov = float(g[k]), float(getattr(o, k))
        assert abs(gv - ov) <= 1e-9 * N, (where, k, gv, ov)
    for k in ("Cx", "Cy", "E"):
        gv, ov = float(g[k]), float(getattr(o, k))
        if abs(ov) > 0.05 * N:
            assert abs(gv - ov) <= 1e-9 * abs(ov), (where, k, gv, ov)
    for k in ("n_bonds_x", "n_bonds_y", "n_clusters", "sweep"):
        assert int(g[k]) == int(getattr(o, k)), (where, k, int(g[k]), int(getattr(o, k)))


def one_sweep_parity(xy, st, theta_before, L, seed, t, beta, fix_phi=None, where=""):
    """oracle sweeps theta_before (a copy) once; compare everything with the GPU state."""
    ref = theta_before.copy()
    b_ref, lab_ref, o_ref = xo.sweep(ref, L, seed, t, beta, fix_phi=fix_phi)
    b_gpu = st.get_bonds()
    n_mismatch = 0
    if not (b_gpu == b_ref).all():
        ph = xo.phi(seed, t) if fix_phi is None else fix_phi
        for i in np.nonzero(b_gpu != b_ref)[0]:
            for d in (0, 1):
                if ((b_gpu[i] ^ b_ref[i]) >> d) & 1:
                    m = xo.bond_margin(theta_before, L, beta, ph, seed, t, int(i), d)
                    assert abs(m) < 1e-12, (where, "bond mismatch with margin", int(i), d, m)
                    n_mismatch += 1
    assert n_mismatch == 0, (where, "bond mismatches inside the 1e-12 margin", n_mismatch)
    lab_gpu = st.get_labels()
    assert (lab_gpu == lab_ref).all(), (where, "labels", int((lab_gpu != lab_ref).sum()))
    th_gpu = st.get_angles()
    ulps = ulp_diff(th_gpu, ref)
    assert ulps.max() == 0, (where, "angles max ulp", int(ulps.max()))
    g = st.measure().as_dict()
    check_obs(g, o_ref, L * L, where)
    assert g["beta"] == beta
    return ref


# ----------------------------------------------------------------------------------------------
def test_philox_three_way(xy):
    """the CUDA path's Philox == NVIDIA cuRAND's device function == the oracle's."""
    rng = np.random.default_rng(5)
    n = 200000
    ctr = rng.integers(0, 2 ** 32, (n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, (n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[:8] = [[0, 0, 0, 0], [1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1],
               [0xffffffff] * 4, [0, 0, 0, 3], [5, 0, 9, 2]]
    mine = xy.debug_philox(ctr, key)
    theirs = xy.debug_curand_philox(ctr, key)
    assert (mine == theirs).all()
    for i in list(range(16)) + list(range(1000, n, 997)):
        assert (xo.philox4x32_10(ctr[i], key[i]) == mine[i]).all()


@pytest.mark.parametrize("L", [64, 128, 192, 320])
def test_init_parity(xy, L):
    for seed in (1, 0xFEDCBA9876543210):
        st = xy.XYState(L, seed, xy.INIT_HOT)
        assert (st.get_angles() == xo.init(L, seed, xo.INIT_HOT)).all()
        o = st.measure()
        ref = xo.observe(xo.init(L, seed, xo.INIT_HOT), L)
        assert o.sweep == 0 and math.isnan(o.beta) and o.n_clusters == 0
        for k in ("Mx", "My", "Cx", "Sx", "Cy", "Sy", "E"):
            assert abs(getattr(o, k) - getattr(ref, k)) <= 1e-9 * L * L
        st.destroy()
    st = xy.XYState(L, 3, xy.INIT_COLD)
    th = st.get_angles()
    assert (th == 0).all() and not np.signbit(th).any()
    o = st.measure()
    assert o.E == -2.0 * L * L and o.Mx == L * L and o.My == 0 and o.Sx == 0
    st.destroy()


CASES = [
    # L, input, beta      (L = 64, 192, 320: 64-wide tiles; 128, 256, 384, 1024: 128-wide tiles;
    #                      192/320/384 give tile counts that are not powers of two)
    (64, "hot", 1.12), (64, "cold", 1.12), (64, "smooth", 0.9), (64, "vortex", 1.5),
    (128, "hot", 1.12), (128, "cold", 1.3), (128, "smooth", 1.12),
    (192, "hot", 1.0), (192, "vortex", 1.12), (192, "cold", 0.9),
    (256, "smooth", 1.12), (256, "random", 0.5), (320, "smooth", 1.2),
    (384, "vortex", 1.12), (384, "cold", 1.12),
    (1024, "hot", 1.12), (1024, "cold", 1.12), (1024, "smooth", 1.11996),
]


def make_input(kind, L, seed):
    if kind == "hot":
        return None, xy_inputs.INIT_CODE["hot"]
    if kind == "cold":
        return None, xy_inputs.INIT_CODE["cold"]
    if kind == "smooth":
        return xy_inputs.smooth_angles(L, seed), 0
    if kind == "vortex":
        return xy_inputs.vortex_pair_angles(L, seed), 0
    if kind == "random":
        return xy_inputs.random_angles(L, seed), 0
    raise ValueError(kind)


@pytest.mark.parametrize("L,kind,beta", CASES)
@pytest.mark.parametrize("flags", [0, 1])
def test_sweep_parity(xy, L, kind, beta, flags):
    """three chained sweeps from each input, full state compared after every sweep."""
    if flags and L > 384:
        pytest.skip("64-bit labels are covered at the smaller sizes")
    seed = 1000 + L
    theta, init = make_input(kind, L, seed)
    st = xy.XYState(L, seed, init, flags=flags)
    if theta is not None:
        st.set_angles(theta)
        cur = theta.copy()
    else:
        cur = xo.init(L, seed, init)
    assert (st.get_angles() == cur).all()
    for t in range(3):
        st.sw_sweeps(beta, 1)
        cur = one_sweep_parity(xy, st, cur, L, seed, t, beta, where=f"L={L} {kind} t={t}")
    st.destroy()


def test_config1_chained_1000_sweeps(xy):
    """BASELINE config 1: L=64, hot start seed 1, beta=1.12, 1000 sweeps, all chained, observables
    of every sweep from the device ring against the oracle's series."""
    cfg = xy_inputs.CONFIGS[0]
    L, seed, beta, n = cfg["L"], cfg["seed"], cfg["beta"], cfg["sweeps"]
    st = xy.XYState(L, seed, xy.INIT_HOT)
    ref = xo.init(L, seed, xo.INIT_HOT)
    ser_ref = xo.run(ref, L, seed, 0, beta, n)
    st.sw_sweeps(beta, n)
    ser = st.get_series(1, n)
    assert (st.get_angles() == ref).all()
    N = L * L
    for k in range(n):
        for f in ("Mx", "My", "Sx", "Sy", "Cx", "Cy", "E"):
            assert abs(ser[f][k] - ser_ref[f][k]) <= 1e-9 * N, (k, f)
        for f in ("n_bonds_x", "n_bonds_y", "n_clusters", "sweep"):
            assert ser[f][k] == ser_ref[f][k], (k, f)
        assert ser["beta"][k] == beta
    # the physics the config asks to record
    m2 = (ser["Mx"] ** 2 + ser["My"] ** 2) / N ** 2
    assert 0.2 < m2[200:].mean() < 0.5
    assert st.get_fallback_count() < 2 * N * n * 1e-4
    st.destroy()


def test_chaining_and_resume(xy):
    L, seed, beta = 128, 9, 1.1
    a = xy.XYState(L, seed, xy.INIT_HOT)
    a.sw_sweeps(beta, 12)
    ta = a.get_angles()
    b = xy.XYState(L, seed, xy.INIT_HOT)
    for _ in range(12):
        b.sw_sweeps(beta, 1)
    assert (b.get_angles() == ta).all()
    oa, ob = a.measure(), b.measure()
    assert oa.as_dict() == ob.as_dict()
    # resume from (theta, t) in a fresh state
    c = xy.XYState(L, seed, xy.INIT_HOT)
    c.sw_sweeps(beta, 5)
    snap, t = c.get_angles(), c.get_sweep()
    d = xy.XYState(L, seed, xy.INIT_COLD)
    d.set_angles(snap)
    d.set_sweep(t)
    d.sw_sweeps(beta, 7)
    assert (d.get_angles() == ta).all()
    # run twice: identical, including the observables bit for bit
    e = xy.XYState(L, seed, xy.INIT_HOT)
    e.sw_sweeps(beta, 12)
    assert (e.get_angles() == ta).all() and e.measure().as_dict() == oa.as_dict()
    sa, se = a.get_series(0, 13), e.get_series(0, 13)
    assert sa.tobytes() == se.tobytes()
    for s in (a, b, c, d, e):
        s.destroy()


def test_series_measure_semantics(xy):
    L, seed, beta = 64, 4, 1.0
    st = xy.XYState(L, seed, xy.INIT_HOT)
    ref = xo.init(L, seed, xo.INIT_HOT)
    o0 = st.measure()
    assert o0.sweep == 0 and o0.n_bonds_x == 0
    st.sw_sweeps(beta, 3)
    r1 = st.measure()                      # lazily computed record T=3
    st.sw_sweeps(beta, 2)
    ser = st.get_series(0, 6)              # records 0..5, the last again lazily
    ser_ref = xo.run(ref, L, seed, 0, beta, 5)
    assert list(ser["sweep"]) == [0, 1, 2, 3, 4, 5]
    for k in range(5):
        for f in ("E", "Mx", "Sx", "Cy"):
            assert abs(ser[f][k + 1] - ser_ref[f][k]) <= 1e-9 * L * L
        assert ser["n_clusters"][k + 1] == ser_ref["n_clusters"][k]
    assert r1.E == ser["E"][3] and r1.n_clusters == ser["n_clusters"][3]
    with pytest.raises(xy.XYError):
        st.get_series(3, 10)
    st.destroy()


@pytest.mark.parametrize("L", [64, 128, 192, 256])
@pytest.mark.parametrize("flags", [0, 1])
def test_labels_on_injected_bonds(xy, L, flags):
    """the labeling kernels alone (tile-local union-find + boundary merge + flatten) on adversarial
    and random bond sets."""
    st = xy.XYState(L, 1, xy.INIT_COLD, flags=flags)
    sets = [xy_inputs.pattern_bonds(L, k) for k in xy_inputs.BOND_PATTERNS]
    sets += [xy_inputs.random_bonds(L, d, 50 + i) for i, d in enumerate((0.05, 0.3, 0.45, 0.5, 0.55, 0.7, 0.95))]
    for k, b in enumerate(sets):
        st.label_bonds(b)
        got = st.get_labels()
        want, _ = xo.label(b, L)
        assert (got == want).all(), (L, k, int((got != want).sum()))
    st.destroy()


def test_ising_limit_fixed_phi(xy):
    """angles in {0, pi}, r fixed along x (xy_debug_fix_phi): parity over 50 chained sweeps."""
    L, seed, beta = 64, 6, 0.44
    th = xy_inputs.clock_angles(L, 2, 3)
    st = xy.XYState(L, seed, xy.INIT_COLD)
    st.set_angles(th)
    st.debug_fix_phi(True, 0.0)
    ref = th.copy()
    for t in range(50):
        st.sw_sweeps(beta, 1)
        if t % 10 == 0:
            ref = one_sweep_parity(xy, st, ref, L, seed, t, beta, fix_phi=0.0, where=f"ising t={t}")
        else:
            xo.sweep(ref, L, seed, t, beta, fix_phi=0.0)
    assert (st.get_angles() == ref).all()
    st.destroy()


def test_beta_extremes(xy):
    L, seed = 128, 2
    st = xy.XYState(L, seed, xy.INIT_HOT)
    th0 = st.get_angles()
    st.sw_sweeps(0.0, 1)
    one_sweep_parity(xy, st, th0, L, seed, 0, 0.0, where="beta=0")
    assert st.get_bonds().sum() == 0 and st.measure().n_clusters == L * L
    st2 = xy.XYState(L, seed, xy.INIT_COLD)
    st2.debug_fix_phi(True, 0.0)
    st2.sw_sweeps(1e9, 1)
    assert (st2.get_bonds() == 3).all() and (st2.get_labels() == 0).all()
    one_sweep_parity(xy, st2, np.zeros(L * L, np.float32), L, seed, 0, 1e9, fix_phi=0.0, where="beta=1e9")
    st.destroy()
    st2.destroy()


def test_pcc_trace_parity(xy):
    """config 3's schedule (beta0 1.05, dbeta0 1e-3 halved down to 1e-6, target 2/pi, window 20,
    dirs 1) chained at L=64 and L=128: beta traces must be bit-equal to the oracle's."""
    cfg = xy_inputs.CONFIGS[2]
    for L, n, halve in ((64, 3000, 300), (128, 600, 100)):
        for dirs in (1, 2):
            sg = xy.PccSchedule(n_sweeps=n, discard=40, window=cfg["window"], dirs=dirs, dbeta0=cfg["dbeta0"],
                                halve_every=halve, dbeta_min=cfg["dbeta_min"], target=cfg["target"])
            so = xo.PccSchedule(n_sweeps=n, discard=40, window=cfg["window"], dirs=dirs, dbeta0=cfg["dbeta0"],
                                halve_every=halve, dbeta_min=cfg["dbeta_min"], target=cfg["target"])
            st = xy.XYState(L, cfg["seed"], xy.INIT_HOT)
            out = st.pcc_run(cfg["beta0"], sg)
            ref_theta = xo.init(L, cfg["seed"], xo.INIT_HOT)
            ref = xo.pcc_run(ref_theta, L, cfg["seed"], 0, cfg["beta0"], so, trace_cap=n)
            assert out["n_decisions"] == ref["n_decisions"] == (n - 40) // cfg["window"]
            assert (out["trace_beta"] == ref["trace_beta"]).all(), (L, dirs)
            assert np.abs(out["trace_bY"] - ref["trace_bY"]).max() < 1e-9
            assert np.abs(ref["trace_bY"] - cfg["target"]).min() > 1e-10     # no decision was a coin toss
            assert out["beta_final"] == ref["beta_final"] and out["dbeta_final"] == ref["dbeta_final"]
            assert out["beta_mean"] == ref["beta_mean"]
            assert (st.get_angles() == ref_theta).all()
            assert st.get_sweep() == n
            st.destroy()


def test_errors(xy):
    for L in (0, 32, 100, 65600):
        with pytest.raises(xy.XYError) as e:
            xy.XYState(L, 1)
        assert e.value.code == -2
    st = xy.XYState(64, 1)
    for beta in (-1.0, float("nan"), float("inf")):
        with pytest.raises(xy.XYError) as e:
            st.sw_sweeps(beta, 1)
        assert e.value.code == -1
    with pytest.raises(xy.XYError) as e:
        st.get_labels()
    assert e.value.code == -5
    bad = np.full(64 * 64, 7.0, np.float32)
    with pytest.raises(xy.XYError):
        st.set_angles(bad)
    st.set_angles(np.zeros(64 * 64, np.float32))
    st.set_sweep(2 ** 32 - 1)
    with pytest.raises(xy.XYError) as e:
        st.sw_sweeps(1.0, 2)
    assert e.value.code == -5
    st.destroy()
    # caller-owned workspace that is too small
    import torch
    import ctypes as C
    from paper_1210_6116_b200 import binding
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    assert binding._lib.xy_create_ex(C.byref(h), 64, 1, 0, 0, ws.data_ptr(), 1024) == -1
    # library-owned allocation works too
    st = xy.XYState(64, 1, torch_workspace=False)
    st.sw_sweeps(1.0, 2)
    assert st.measure().sweep == 2
    st.destroy()


def test_pcc_continue_and_checkpoint(xy):
    """xy_pcc_run(2 M) == xy_pcc_run(M) + xy_pcc_continue(M), also through a checkpoint into a fresh state (angles, sweep
    counter, controller state); the device-side sums of <m^2> equal the per-sweep series of the fed sweeps."""
    L, seed, M = 128, 9, 240
    mk = lambda n, disc: xy.PccSchedule(n_sweeps=n, discard=disc, window=20, dirs=1, dbeta0=1e-3, halve_every=100,
                                        dbeta_min=1e-6, target=2 / np.pi)
    a = xy.XYState(L, seed, xy.INIT_HOT)
    ra = a.pcc_run(1.05, mk(2 * M + 10, 10))
    b = xy.XYState(L, seed, xy.INIT_HOT)
    r1 = b.pcc_run(1.05, mk(M + 10, 10))
    r2 = b.pcc_continue(mk(M, 0))
    assert r2["beta_final"] == ra["beta_final"] and r2["dbeta_final"] == ra["dbeta_final"]
    assert (np.concatenate([r1["trace_beta"], r2["trace_beta"]]) == ra["trace_beta"]).all()
    assert (np.concatenate([r1["trace_bY"], r2["trace_bY"]]) == ra["trace_bY"]).all()
    assert (a.get_angles() == b.get_angles()).all()
    # checkpoint after the first part, restore into another state
    c = xy.XYState(L, seed, xy.INIT_HOT)
    c.pcc_run(1.05, mk(M + 10, 10))
    ck = (c.get_angles(), c.get_sweep(), c.pcc_get_state())
    d = xy.XYState(L, seed, xy.INIT_COLD)                 # the seed belongs to the checkpoint: same RNG stream
    d.set_angles(ck[0]); d.set_sweep(ck[1]); d.pcc_set_state(ck[2])
    r3 = d.pcc_continue(mk(M, 0))
    assert r3["beta_final"] == ra["beta_final"] and (r3["trace_beta"] == r2["trace_beta"]).all()
    assert (d.get_angles() == a.get_angles()).all()
    sa, sd = a.pcc_get_state(), d.pcc_get_state()
    assert (sa.k, sa.n_decisions, sa.n_acc) == (sd.k, sd.n_decisions, sd.n_acc) == (2 * M, 2 * M // 20, 2 * M)
    assert sa.sum_m2 == sd.sum_m2 and sa.beta == sd.beta
    # the fed sweeps are the states T = 11 ... 2 M + 10 of run a
    ser = a.get_series(11, 2 * M)
    m2 = ((ser["Mx"] ** 2 + ser["My"] ** 2) / float(L * L) ** 2).sum()
    assert abs(sa.sum_m2 - m2) <= 1e-12 * m2
    for s in (a, b, c, d):
        s.destroy()
