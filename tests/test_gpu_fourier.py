"""GPU parity of the structure-factor sums at k = 2 pi / L (XY_FLAG_FOURIER; Eq. 8-9)
against the oracle's plain definition: |gpu - oracle| <= 1e-9 N per sum, on injected configurations and
along a chain of sweeps; the hot-path results of a FOURIER state are bit-identical to a plain state's."""
import numpy as np
import pytest

import xy_inputs
from oracle import xy_oracle as xo

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def xy():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_6116_b200 as m
    return m


def check_fourier(F_gpu, theta, L, where=""):
    F_ref = xo.fourier(theta, L)
    N = L * L
    for k in range(8):
        assert abs(F_gpu[k] - F_ref[k]) <= 1e-9 * N, (where, k, F_gpu[k], F_ref[k])


@pytest.mark.parametrize("L", [64, 128, 192, 384, 1024])
@pytest.mark.parametrize("kind", ["random", "smooth", "wave_x", "wave_y"])
def test_fourier_injected(xy, L, kind):
    N = L * L
    if kind == "random":
        th = xy_inputs.random_angles(L, 7)
    elif kind == "smooth":
        th = xy_inputs.smooth_angles(L, 3)
    else:
        x = np.tile(np.arange(L), L)
        y = np.repeat(np.arange(L), L)
        th = (2.0 * np.pi * (x if kind == "wave_x" else y) / L).astype(np.float32)
    st = xy.XYState(L, 1, xy.INIT_COLD, flags=xy.FLAG_FOURIER)
    st.set_angles(th)
    F = st.measure_fourier()
    check_fourier(F, th, L, kind)
    if kind.startswith("wave"):                   # closed form: (N/2, 0, 0, N/2) along the wave, 0 across
        on, off = (F[:4], F[4:]) if kind == "wave_x" else (F[4:], F[:4])
        assert np.allclose(on, [N / 2, 0, 0, N / 2], atol=1e-3 * L) and np.allclose(off, 0, atol=1e-3 * L)
    st.destroy()


@pytest.mark.parametrize("L,flags", [(64, 0), (256, 0), (192, 1)])
def test_fourier_series_along_sweeps(xy, L, flags):
    seed, beta, n = 11, 1.1, 6
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=flags | xy.FLAG_FOURIER)
    plain = xy.XYState(L, seed, xy.INIT_HOT, flags=flags)
    ref = xo.init(L, seed, xo.INIT_HOT)
    thetas = [ref.copy()]
    for t in range(n):
        xo.sweep(ref, L, seed, t, beta)
        thetas.append(ref.copy())
    st.sw_sweeps(beta, n)
    plain.sw_sweeps(beta, n)
    assert (st.get_angles() == ref).all() and (plain.get_angles() == ref).all()
    ser = st.get_fourier_series(0, n + 1)
    assert list(ser["sweep"]) == list(range(n + 1))
    for t in range(n + 1):
        check_fourier(np.concatenate([ser["Fx"][t], ser["Fy"][t]]), thetas[t], L, f"T={t}")
    assert (st.measure_fourier() == np.concatenate([ser["Fx"][n], ser["Fy"][n]])).all()
    # the FOURIER variant's other sums follow another (fixed) order: same tolerance against the oracle
    o_ref = xo.observe(ref, L)
    g = st.measure()
    for k in ("Mx", "My", "Cx", "Sx", "Cy", "Sy", "E"):
        assert abs(getattr(g, k) - getattr(o_ref, k)) <= 1e-9 * L * L, k
    gp = plain.measure()
    assert (g.n_bonds_x, g.n_bonds_y, g.n_clusters) == (gp.n_bonds_x, gp.n_bonds_y, gp.n_clusters)
    st.destroy()
    plain.destroy()


def test_fourier_records_of_sweeps_without_observables_read_nan(xy):
    """XY_OBS_NONE sweeps of a FOURIER state: their structure-factor records carry the sweep number and NaN sums (never
    a stale record of an older sweep), the records around them are the oracle's, the chain itself is unchanged"""
    L, seed, beta = 128, 9, 1.1
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=xy.FLAG_FOURIER)
    ref = xo.init(L, seed, xo.INIT_HOT)
    thetas = [ref.copy()]
    for t in range(7):
        xo.sweep(ref, L, seed, t, beta)
        thetas.append(ref.copy())
    st.sw_sweeps(beta, 3)                              # records 0..2 filled by the sweeps, 3 still open
    st.set_obs_mode(xy.OBS_NONE)
    st.sw_sweeps(beta, 2)                              # sweeps 3, 4: no sums; records 3 (incoming state of sweep 3) and 4 never filled
    st.set_obs_mode(xy.OBS_ALL)
    st.sw_sweeps(beta, 2)                              # sweeps 5, 6 fill records 5, 6; record 7 on demand
    assert (st.get_angles() == ref).all()
    ser = st.get_fourier_series(0, 8)
    assert list(ser["sweep"]) == list(range(8))
    for t in range(8):
        F = np.concatenate([ser["Fx"][t], ser["Fy"][t]])
        if t in (3, 4):
            assert np.isnan(F).all(), (t, F)
        else:
            check_fourier(F, thetas[t], L, f"T={t}")
    obs = st.get_series(0, 8)
    assert np.isnan(obs["E"][3]) and np.isnan(obs["E"][4]) and not np.isnan(obs["E"][[0, 1, 2, 5, 6, 7]]).any()
    st.destroy()


def test_fourier_needs_flag(xy):
    st = xy.XYState(64, 1, xy.INIT_COLD)
    with pytest.raises(xy.XYError):
        st.measure_fourier()
    with pytest.raises(xy.XYError):
        st.get_fourier_series(0, 1)
    st.destroy()


def test_xi2nd_from_gpu_series_matches_oracle_chain(xy):
    """xi_2nd/L from a short GPU series equals the oracle's from the same chain (same configurations)."""
    L, seed, beta, n = 64, 4, 1.09167, 200
    st = xy.XYState(L, seed, xy.INIT_HOT, flags=xy.FLAG_FOURIER)
    st.sw_sweeps(beta, n)
    ser, obs = st.get_fourier_series(1, n), st.get_series(1, n)
    ref = xo.init(L, seed, xo.INIT_HOT)
    c0g = ckg = c0r = ckr = 0.0
    for t in range(n):
        o = xo.run(ref, L, seed, t, beta, 1, series=True)[-1]
        F = xo.fourier(ref, L)
        c0r += (o["Mx"] ** 2 + o["My"] ** 2) / (L * L)
        ckr += 0.5 * (xo.sk(F[:4], L) + xo.sk(F[4:], L))
        c0g += (obs["Mx"][t] ** 2 + obs["My"][t] ** 2) / (L * L)
        ckg += 0.5 * (xo.sk(ser["Fx"][t], L) + xo.sk(ser["Fy"][t], L))
    assert xo.xi2nd(c0g / n, ckg / n, L) == pytest.approx(xo.xi2nd(c0r / n, ckr / n, L), rel=1e-9)
    st.destroy()
