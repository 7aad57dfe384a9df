"""Pins for the PCC driver (O8): the rule of PAPER.md:62 on an injected observable, the halving
schedule, and the paper's beta_KT(64) on the real model."""
import math

import numpy as np

from golden_io import constants, table1
from oracle import xy_oracle as xo


def _sched(**kw):
    d = dict(n_sweeps=0, discard=0, window=1, dirs=1, dbeta0=1e-3, halve_every=0, dbeta_min=0.0,
             target=constants()["betaY_critical"])
    d.update(kw)
    return xo.PccSchedule(**d)


def test_rule_direction_and_convergence_on_injected_observable():
    """inject Cx so that beta*Y = g(beta) = 0.5*beta exactly (Sx = 0): beta must converge to
    g^-1(target) = 2*target, rising when beta*Y < target, falling otherwise."""
    s = _sched(window=4, dbeta0=1e-2, halve_every=400, dbeta_min=1e-5)
    N = 1024.0
    target = s.target
    c = xo.PccController(0.9, s)
    betas = []
    for k in range(8000):
        b = c.beta
        r = c.feed(N, Cx=0.5 * N, Sx=0.0)            # e = 0.5 -> Y = 0.5 -> beta*Y = 0.5*beta
        if r is not None:
            assert r[0] == b and abs(r[1] - 0.5 * b) < 1e-15
            step = c.beta - b
            assert (step > 0) == (r[1] < target)
            betas.append(b)
    assert abs(c.beta - 2 * target) < 2e-5
    assert abs(c.beta_mean() - 2 * target) < 2e-5
    assert c.dbeta == 1e-5


def test_halving_schedule_exact():
    s = _sched(window=5, dbeta0=1e-3, halve_every=20, dbeta_min=1e-4)
    c = xo.PccController(1.0, s)
    want = 1e-3
    for k in range(1, 201):
        c.feed(100.0, Cx=50.0, Sx=3.0)
        if k % 20 == 0:
            want = max(want / 2, 1e-4)
        assert c.dbeta == want
    assert c.c.n_decisions == 40


def test_window_average_and_s2_term():
    """Y = <e> - beta N <s^2> over the window (Eq. 4), dirs 1 and 2."""
    N = 400.0
    rng = np.random.default_rng(0)
    cx, sx, cy, sy = (rng.normal(200, 5, 7), rng.normal(0, 8, 7), rng.normal(190, 5, 7), rng.normal(0, 8, 7))
    for dirs in (1, 2):
        s = _sched(window=7, dirs=dirs)
        c = xo.PccController(1.1, s)
        r = None
        for k in range(7):
            r = c.feed(N, cx[k], sx[k], cy[k], sy[k])
        if dirs == 1:
            e = (cx / N).mean()
            s2 = ((sx / N) ** 2).mean()
        else:
            e = ((cx + cy) / (2 * N)).mean()
            s2 = ((sx ** 2 + sy ** 2) / (2 * N * N)).mean()
        want = 1.1 * (e - 1.1 * N * s2)
        assert r is not None and abs(r[1] - want) < 1e-13


def test_discard_and_trace_on_real_model():
    L = 16
    s = _sched(n_sweeps=60, discard=20, window=10, dbeta0=1e-2)
    th = xo.init(L, 3, xo.INIT_HOT)
    out = xo.pcc_run(th, L, 3, 0, 1.0, s, trace_cap=16)
    assert out["n_decisions"] == 4 and out["trace_len"] == 4
    assert out["trace_beta"][0] == 1.0
    # replay by hand with single sweeps and the controller
    th2 = xo.init(L, 3, xo.INIT_HOT)
    c = xo.PccController(1.0, s)
    tr = []
    for t in range(60):
        _, _, o = xo.sweep(th2, L, 3, t, c.beta)
        if t >= 20:
            r = c.feed(L * L, o.Cx, o.Sx, o.Cy, o.Sy)
            if r:
                tr.append(r)
    assert (th == th2).all()
    assert [r[0] for r in tr] == list(out["trace_beta"]) and [r[1] for r in tr] == list(out["trace_bY"])
    assert out["beta_final"] == c.beta


def test_pcc_finds_paper_beta_kt_L64():
    """paper protocol, shortened: L=64 must settle near beta_KT(64) = 1.09167(25).
    window 100 instead of 1000 biases the crossing by < 1e-3 (median vs mean of the window
    estimate); tolerance covers that and the walk's own spread."""
    row = table1()[64]
    L = 64
    s = _sched(n_sweeps=16000, discard=500, window=100, dbeta0=2e-3, halve_every=4000, dbeta_min=5e-4)
    th = xo.init(L, 12, xo.INIT_HOT)
    out = xo.pcc_run(th, L, 12, 0, 1.06, s, trace_cap=200)
    tb = out["trace_beta"]
    assert out["n_decisions"] == 155
    assert abs(tb[40:].mean() - row["beta"]) < 8e-3, tb[40:].mean()
    assert out["dbeta_final"] == 5e-4
