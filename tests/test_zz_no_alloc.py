"""xy_observe_static against xy_measure.

Who needs this call: a program that may not let a library allocate GPU memory -- all of it already belongs to the
program's own pool or caching allocator, or a cudaMalloc would stall the streams it keeps busy.  For such a caller
the kernel's scratch (per-CTA partial sums, a ticket counter, the sine / cosine table) is a fixed array inside the
library instead of a cudaMalloc'ed workspace.  Every call on a GPU reuses that one array and finds the previous call's
contents in it, so the test makes TWO calls in a row, on two different configurations and two lattice sizes, and
wants each to agree with the ordinary path (a state's xy_measure on the same angles) within the tolerance the other
GPU tests use for the sums, 1e-9 N.

This file sorts last on purpose (pytest -x stops at the first failure, and nothing should hide behind this one); it
has to pass both on its own in a fresh process -- the first call then does the per-device set-up -- and after all
other tests have used the GPU.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SUMS = ("E", "Mx", "My", "Cx", "Sx", "Cy", "Sy")


@pytest.fixture(scope="module")
def xy():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_6116_b200 as m
    return m


def reference(xy, L, seed, n_sweeps):
    """angles after a few sweeps from a hot start and the sums xy_measure reports for them (the existing path)"""
    st = xy.XYState(L, seed, xy.INIT_HOT)
    st.sw_sweeps(1.1, n_sweeps)
    theta = st.get_angles()
    obs = st.measure().as_dict()
    st.destroy()
    return theta, obs


def test_two_calls_in_a_row_match_xy_measure(xy):
    import torch
    # 512: 128-wide strips of 8 rows; 192: 64-wide strips (L not a multiple of 128); two different configurations,
    # so a sum left over from the first call cannot pass for the second
    cases = [(512, 11, 3), (192, 12, 1)]
    refs = [reference(xy, *c) for c in cases]
    dev = [torch.from_numpy(th).cuda() for th, _ in refs]
    outs = [torch.full((96,), 0xAB, dtype=torch.uint8, device="cuda") for _ in cases]    # poisoned: the call must fill it
    torch.cuda.synchronize()
    for (L, _, _), th, out in zip(cases, dev, outs):      # back to back on one stream, no synchronise in between
        assert xy.observe_static(th, L, out) is out
    torch.cuda.synchronize()
    for (L, _, _), (_, want), out, th, (th_host, _) in zip(cases, refs, outs, dev, refs):
        got = out.cpu().numpy().view(xy.OBS_DTYPE)[0]
        N = L * L
        for k in SUMS:
            assert abs(float(got[k]) - want[k]) <= 1e-9 * N, (L, k, float(got[k]), want[k])
        assert abs(float(got["E"])) > 0.1 * N                 # a real configuration, not zeros
        assert int(got["sweep"]) == 0 and float(got["beta"]) == 0.0
        assert (int(got["n_bonds_x"]), int(got["n_bonds_y"]), int(got["n_clusters"])) == (0, 0, 0)
        assert (th.cpu().numpy() == th_host).all()           # the input is not modified

    # the same array a third time: the first configuration again, after the second used the scratch
    out = xy.observe_static(dev[0], cases[0][0])
    torch.cuda.synchronize()
    got = out.cpu().numpy().view(xy.OBS_DTYPE)[0]
    for k in SUMS:
        assert abs(float(got[k]) - refs[0][1][k]) <= 1e-9 * cases[0][0] ** 2, k


def test_sizes_beyond_the_limit_are_rejected(xy):
    import torch
    th = torch.zeros(64 * 64, dtype=torch.float32, device="cuda")
    out = torch.zeros(96, dtype=torch.uint8, device="cuda")
    from paper_1210_6116_b200 import binding as b
    for bad in (65536 + 64, 100, 0):
        rc = b._lib.xy_observe_static(th.data_ptr(), bad, out.data_ptr(), None)
        assert rc == -2, (bad, rc)
        assert b"unsupported" in b._lib.xy_last_error()
    host = np.zeros(64 * 64, np.float32)
    assert b._lib.xy_observe_static(host.ctypes.data, 64, out.data_ptr(), None) == -1    # a host pointer is refused
    assert b._lib.xy_observe_static(None, 64, out.data_ptr(), None) == -1
    # and the call still works afterwards: cold lattice, E = -2 N exactly
    xy.observe_static(th, 64, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy().view(xy.OBS_DTYPE)[0]
    assert float(got["E"]) == -2.0 * 64 * 64 and float(got["Mx"]) == 64.0 * 64 and float(got["My"]) == 0.0
