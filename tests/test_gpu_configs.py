"""Parity at the BASELINE configs' own sizes and schedules (north_star: bit-exact at every config), and the
kernel variants that only large or odd sizes select.  Everything goes through the C-ABI.

config 2 (L = 1024, cold, seed 7, beta in {0.90, 1.00, 1.12, 1.30}): 200 chained sweeps per beta with the
          per-sweep observables and the final state compared, then sampled one-step parities at t = 2000, 5000
          and 12000 (the sweep is a deterministic function of (theta, seed, t, beta)).
config 3 (L = 4096, hot, seed 11, PCC beta0 = 1.05, dbeta0 = 1e-3, window 20, target 2/pi): the first 40
          sweeps (two decisions) chained - beta trace and final angles of xy_pcc_run against the oracle's
          controller, and bonds / labels / angles in full at sweeps 0, 10, 20, 30, 39 - then five sampled
          one-step parities later in the run; the literal 20 000-sweep schedule at L = 64 and a shortened
          one at L = 256 with bit-equal beta traces.
filter    full byte-compare of the bonds of >= 10 sweeps at L = 4096 for beta in {0.5, 1.11996, 5, 50}
          (1.3e9 decisions) against the oracle's fp64 definition: the volume test of the fp32 filter.
variants  L = 4160 (64-wide tiles with 32-row strips), both label widths; FOURIER at L = 8192.
"""
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import xy_inputs
from oracle import xy_oracle as xo

pytestmark = pytest.mark.gpu

OBS_KEYS = ("Mx", "My", "Sx", "Sy", "Cx", "Cy", "E")


@pytest.fixture(scope="module")
def xy():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_6116_b200 as m
    return m


def assert_bonds_equal(b_gpu, b_ref, theta_before, L, beta, seed, t, where):
    """bond bytes equal; a differing decision is tolerated only where the oracle's |u - p| < 1e-12 (counted)"""
    if np.array_equal(b_gpu, b_ref):
        return 0
    ph = xo.phi(seed, t)
    n = 0
    for i in np.nonzero(b_gpu != b_ref)[0][:100]:
        for d in (0, 1):
            if ((int(b_gpu[i]) ^ int(b_ref[i])) >> d) & 1:
                m = xo.bond_margin(theta_before, L, beta, ph, seed, t, int(i), d)
                assert abs(m) < 1e-12, (where, "bond mismatch", int(i), d, m)
                n += 1
    assert n == 0, (where, "bond mismatches inside the 1e-12 margin", n)
    return n


def assert_obs_close(g, o, N, where):
    for k in OBS_KEYS:
        assert abs(float(g[k]) - float(getattr(o, k))) <= 1e-9 * N, (where, k, float(g[k]), float(getattr(o, k)))
    for k in ("n_bonds_x", "n_bonds_y", "n_clusters"):
        assert int(g[k]) == int(getattr(o, k)), (where, k)


def one_step(st, L, seed, beta, where):
    """sampled one-step parity: theta from the GPU, one GPU sweep, the oracle's sweep of the same theta"""
    t = st.get_sweep()
    th0 = st.get_angles()
    st.sw_sweeps(beta, 1)
    ref = th0.copy()
    b_ref, lab_ref, o_ref = xo.sweep(ref, L, seed, t, beta)
    assert_bonds_equal(st.get_bonds(), b_ref, th0, L, beta, seed, t, where)
    assert np.array_equal(st.get_labels(), lab_ref), (where, "labels")
    assert np.array_equal(st.get_angles().view(np.uint32), ref.view(np.uint32)), (where, "angles")
    assert_obs_close(st.measure().as_dict(), o_ref, L * L, where)


# ---------------------------------------------------------------------------------------------------
def test_config2_all_betas(xy):
    """200 chained sweeps per beta (per-sweep records and final angles), then one-step parities at t = 2000, 5000 and
    12000 (SURVEY.md:482-485).  The oracle's four chains run side by side on host threads (the C oracle releases the
    GIL)."""
    cfg = xy_inputs.CONFIGS[1]
    L, seed, n = cfg["L"], cfg["seed"], 200
    N = L * L

    def chain(beta):
        ref = xo.init(L, seed, xo.INIT_COLD)
        return ref, xo.run(ref, L, seed, 0, beta, n)
    with ThreadPoolExecutor(len(cfg["betas"])) as ex:
        refs = list(ex.map(chain, cfg["betas"]))
    for beta, (ref, ser_ref) in zip(cfg["betas"], refs):
        st = xy.XYState(L, seed, xy.INIT_COLD)
        st.sw_sweeps(beta, n)
        ser = st.get_series(1, n)
        assert np.array_equal(st.get_angles().view(np.uint32), ref.view(np.uint32)), f"angles after {n} chained sweeps, beta={beta}"
        for f in OBS_KEYS:
            assert np.abs(ser[f] - ser_ref[f]).max() <= 1e-9 * N, (beta, f)
        for f in ("n_bonds_x", "n_bonds_y", "n_clusters", "sweep"):
            assert np.array_equal(ser[f], ser_ref[f]), (beta, f)
        for t in (cfg["therm"], 5000, 12000):
            st.sw_sweeps(beta, t - st.get_sweep())
            one_step(st, L, seed, beta, f"cfg2 beta={beta} t={t}")
        st.destroy()


def _cfg3_schedules(xy, n, window=None, halve=None):
    cfg = xy_inputs.CONFIGS[2]
    kw = dict(n_sweeps=n, discard=cfg["discard"], window=window or cfg["window"], dirs=cfg["dirs"], dbeta0=cfg["dbeta0"],
              halve_every=halve or cfg["halve_every"], dbeta_min=cfg["dbeta_min"], target=cfg["target"])
    return cfg, xy.PccSchedule(**kw), xo.PccSchedule(**kw)


def test_config3_first_40_sweeps_chained(xy):
    n, full_at = 40, (0, 10, 20, 30, 39)
    cfg, sg, so = _cfg3_schedules(xy, n)
    L, seed = cfg["L"], cfg["seed"]
    N = L * L
    # the device-side controller: one xy_pcc_run call
    a = xy.XYState(L, seed, xy.INIT_HOT)
    out = a.pcc_run(cfg["beta0"], sg)
    th_a = a.get_angles()
    assert a.get_sweep() == n
    a.destroy()
    # the oracle sweep by sweep under its own controller; a second GPU state follows with the oracle's betas
    b = xy.XYState(L, seed, xy.INIT_HOT)
    ref = xo.init(L, seed, xo.INIT_HOT)
    assert np.array_equal(b.get_angles(), ref)
    ctl = xo.PccController(cfg["beta0"], so)
    trace = []
    for t in range(n):
        beta = ctl.beta
        before = ref.copy() if t in full_at else None
        b_ref, lab_ref, o_ref = xo.sweep(ref, L, seed, t, beta)
        b.sw_sweeps(beta, 1)
        if t in full_at:
            assert_bonds_equal(b.get_bonds(), b_ref, before, L, beta, seed, t, f"cfg3 t={t}")
            assert np.array_equal(b.get_labels(), lab_ref), f"cfg3 labels t={t}"
            assert np.array_equal(b.get_angles().view(np.uint32), ref.view(np.uint32)), f"cfg3 angles t={t}"
        assert_obs_close(b.measure().as_dict(), o_ref, N, f"cfg3 t={t}")
        d = ctl.feed(N, o_ref.Cx, o_ref.Sx, o_ref.Cy, o_ref.Sy)
        if d:
            trace.append(d)
    assert out["n_decisions"] == len(trace) == 2
    assert list(out["trace_beta"]) == [d[0] for d in trace]            # bit-equal betas
    assert np.abs(out["trace_bY"] - np.array([d[1] for d in trace])).max() < 1e-9
    assert out["beta_final"] == ctl.beta
    assert np.array_equal(th_a.view(np.uint32), ref.view(np.uint32)), "xy_pcc_run's final angles"
    # five sampled one-step parities later in the run (beta along the PCC path towards beta_KT(4096) = 1.11097)
    for more, beta in ((160, 1.07), (300, 1.09), (500, 1.10), (1000, 1.11), (2000, 1.11097)):
        b.sw_sweeps(beta, more - 1)
        one_step(b, L, seed, beta, f"cfg3 sampled t={b.get_sweep()}")
    b.destroy()


def test_config3_literal_schedule_L64(xy):
    """config 3's schedule as BASELINE.json states it (20 000 sweeps, window 20, dbeta halved every 2000 measured
    sweeps), chained at L = 64: every beta of the 1000 decisions, beta_mean and the final angles bit for bit"""
    n = 20000
    cfg, sg, so = _cfg3_schedules(xy, n)
    assert (sg.window, sg.halve_every, sg.n_sweeps) == (20, 2000, 20000)
    L, seed = 64, cfg["seed"]
    st = xy.XYState(L, seed, xy.INIT_HOT)
    out = st.pcc_run(cfg["beta0"], sg)
    ref_theta = xo.init(L, seed, xo.INIT_HOT)
    ref = xo.pcc_run(ref_theta, L, seed, 0, cfg["beta0"], so, trace_cap=n)
    assert out["n_decisions"] == ref["n_decisions"] == (n - cfg["discard"]) // cfg["window"]
    assert np.array_equal(out["trace_beta"], ref["trace_beta"])
    assert np.abs(out["trace_bY"] - ref["trace_bY"]).max() < 1e-9
    assert out["beta_final"] == ref["beta_final"] and out["dbeta_final"] == ref["dbeta_final"]
    assert out["beta_mean"] == ref["beta_mean"]
    assert np.array_equal(st.get_angles().view(np.uint32), ref_theta.view(np.uint32))
    st.destroy()


def test_config3_pcc_trace_L256(xy):
    """config 3's schedule, shortened in proportion (4000 sweeps = 200 decisions, dbeta halved every 400), chained
    at L = 256 (the oracle's share of this test is 50 s)"""
    n = 4000
    cfg, sg, so = _cfg3_schedules(xy, n, halve=400)
    L, seed = 256, cfg["seed"]
    st = xy.XYState(L, seed, xy.INIT_HOT)
    out = st.pcc_run(cfg["beta0"], sg)
    ref_theta = xo.init(L, seed, xo.INIT_HOT)
    ref = xo.pcc_run(ref_theta, L, seed, 0, cfg["beta0"], so, trace_cap=n)
    assert out["n_decisions"] == ref["n_decisions"] == n // cfg["window"]
    assert np.array_equal(out["trace_beta"], ref["trace_beta"])
    assert np.abs(out["trace_bY"] - ref["trace_bY"]).max() < 1e-9
    assert np.abs(ref["trace_bY"] - cfg["target"]).min() > 1e-10          # no decision was a coin toss
    assert out["beta_final"] == ref["beta_final"] and out["dbeta_final"] == ref["dbeta_final"]
    assert out["beta_mean"] == ref["beta_mean"]
    assert np.array_equal(st.get_angles().view(np.uint32), ref_theta.view(np.uint32))
    st.destroy()


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("beta", [0.5, 1.11996, 5.0, 50.0])
def test_filter_volume_L4096(xy, beta, record_property):
    """every bond decision of 10 sweeps (3.4e8 per beta) against the oracle's fp64 definition, on the angles
    the GPU itself produced; reports how many decisions sat inside the filter's band and took the exact path"""
    L, seed, n = 4096, 21, 10
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_HOT)
    st.sw_sweeps(beta, 30)                                   # away from the hot start: realistic sigma products
    thetas, bonds_gpu, ts = [], [], []
    fb0 = st.get_fallback_count()
    for _ in range(n):
        ts.append(st.get_sweep())
        thetas.append(st.get_angles())
        st.sw_sweeps(beta, 1)
        bonds_gpu.append(st.get_bonds())
    fallbacks = st.get_fallback_count() - fb0
    st.destroy()
    delta = 1.2e-5 + 1.0e-6 * beta                           # filter_delta(beta), csrc/xy_device.cuh

    def check(k):
        b_ref, mx, my = xo.bonds(thetas[k], L, beta, xo.phi(seed, ts[k]), seed, ts[k], margins=True)
        assert_bonds_equal(bonds_gpu[k], b_ref, thetas[k], L, beta, seed, ts[k], f"filter beta={beta} t={ts[k]}")
        m = np.minimum(np.abs(mx), np.abs(my))
        # decisions within 0.4 delta of the threshold are inside the band for certain (the filter's error is
        # below 0.7 delta): each must have taken the exact path
        return int((np.abs(mx) < 0.3 * delta).sum() + (np.abs(my) < 0.3 * delta).sum()), float(m.min())

    with ThreadPoolExecutor(max_workers=5) as ex:
        res = list(ex.map(check, range(n)))
    surely_inside = sum(r[0] for r in res)
    assert fallbacks >= surely_inside, (fallbacks, surely_inside)
    if delta < 0.01:
        assert fallbacks <= 2 * N * n * 2.5 * delta, (fallbacks, "fallback rate far above 2 delta per bond")
    record_property("decisions", 2 * N * n)
    record_property("fallbacks", fallbacks)
    record_property("min_abs_margin", min(r[1] for r in res))
    print(f"beta={beta}: {2 * N * n} decisions, 0 mismatches, {fallbacks} exact-path decisions "
          f"({fallbacks / (2 * N * n):.2e} per bond, 2 delta = {2 * delta:.2e}), smallest |u - p| = {min(r[1] for r in res):.2e}")


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1])
def test_L4160_narrow_tiles_long_strips(xy, flags):
    """L = 65 * 64: the 64-wide-tile kernels with 32-row strips (chosen only for L > 4096 not a multiple of 128)"""
    L, seed, beta = 4160, 5, 1.11996
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=flags)
    assert np.array_equal(st.get_angles(), xo.init(L, seed, xo.INIT_HOT))
    st.sw_sweeps(beta, 3)
    one_step(st, L, seed, beta, f"L=4160 flags={flags}")
    st.set_obs_mode(xy.OBS_NONE)                         # the fp32-only variant must decide the same bonds
    one_step(st, L, seed, beta, f"L=4160 flags={flags} obs off")
    st.destroy()


def test_fourier_L8192(xy):
    """XY_FLAG_FOURIER with 32-row strips (the xi_2nd path of the Table I rows L >= 8192)"""
    L, seed, beta = 8192, 3, 1.11996
    N = L * L
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=xy.FLAG_FOURIER)
    st.sw_sweeps(beta, 4)
    th = st.get_angles()
    F = st.measure_fourier()
    assert np.abs(F - xo.fourier(th, L)).max() <= 1e-9 * N
    o, ref = st.measure(), xo.observe(th, L)
    for k in OBS_KEYS:
        assert abs(getattr(o, k) - getattr(ref, k)) <= 1e-9 * N, k
    # the record of the sweep before (filled by the sweep kernel itself, rotated frame) against the lazily
    # measured one of the same configuration
    st.sw_sweeps(beta, 1)
    fs = st.get_fourier_series(4, 1)[0]
    assert np.abs(np.concatenate([fs["Fx"], fs["Fy"]]) - F).max() <= 1e-9 * N
    st.destroy()


def test_obs_none_L8192_one_step(xy):
    """k_bonds<4, 32, bonds, no observables> (fp32 only, two CTAs of 8 warps per SM): the variant every lattice above
    4096 takes under XY_OBS_NONE, as in bench.py's observables-off legs; one sweep against the oracle in full"""
    L, seed, beta = 8192, 5, 1.11996
    st = xy.XYState(L, seed, xy.INIT_HOT)
    st.set_obs_mode(xy.OBS_NONE)
    st.sw_sweeps(beta, 3)
    one_step(st, L, seed, beta, "L=8192 obs off")
    st.destroy()


def test_obs_mode_none_same_trajectory(xy):
    """sweeps with the observables switched off produce the same bonds, labels and angles, bit for bit"""
    L, seed, beta = 512, 8, 1.1
    a = xy.XYState(L, seed, xy.INIT_HOT)
    b = xy.XYState(L, seed, xy.INIT_HOT)
    b.set_obs_mode(xy.OBS_NONE)
    a.sw_sweeps(beta, 25)
    b.sw_sweeps(beta, 25)
    assert np.array_equal(a.get_angles().view(np.uint32), b.get_angles().view(np.uint32))
    assert np.array_equal(a.get_bonds(), b.get_bonds()) and np.array_equal(a.get_labels(), b.get_labels())
    ra, rb = a.measure(), b.measure()                    # b: one observables-only pass
    assert (ra.n_bonds_x, ra.n_bonds_y, ra.n_clusters) == (rb.n_bonds_x, rb.n_bonds_y, rb.n_clusters)
    for k in OBS_KEYS:
        assert abs(getattr(ra, k) - getattr(rb, k)) <= 1e-9 * L * L
    sb = b.get_series(20, 5)                             # records of unobserved sweeps: counts kept, sums NaN
    assert np.isnan(sb["E"]).all() and (sb["n_clusters"] > 0).all() and (sb["beta"] == beta).all()
    a.destroy()
    b.destroy()


def test_set_angles_rejection_keeps_state(xy):
    L = 128
    st = xy.XYState(L, 3, xy.INIT_HOT)
    st.sw_sweeps(1.0, 2)
    th = st.get_angles()
    bad = th.copy()
    bad[L * 7 + 5] = 1e6
    with pytest.raises(xy.XYError):
        st.set_angles(bad)
    assert np.array_equal(st.get_angles(), th)           # nothing was committed
    st.sw_sweeps(1.0, 1)                                 # and the state is still usable
    assert st.measure().sweep == 3
    st.destroy()
