"""Row-slab sharded sweep on ONE GPU: G slab states of one process, driven by the same
ShardedLattice.sweep the NCCL path uses (ranks are threads, host-side rendezvous only), against the oracle's sweep of
the whole lattice: angles, bonds and canonical labels bit for bit, counts equal, sums to 1e-9 N."""
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


def _run(xy, L, G, seed, init, beta, sweeps, flags=0, check_every=1, obs_none=False):
    from paper_1210_6116_b200 import shard
    kind = xy.INIT_HOT if init == "hot" else xy.INIT_COLD
    ref = xo.init(L, seed, xo.INIT_HOT if init == "hot" else xo.INIT_COLD)
    N = L * L

    def body(rank, comm):
        rows, y_off = shard.slab_rows(L, G, rank)
        slab = xy.SlabState(L, rows, y_off, seed, kind, flags)
        if obs_none:
            slab.set_obs_mode(xy.OBS_NONE)           # chained sweeps without the sums; measure still works
        return shard.ShardedLattice(slab, comm)

    lats = shard.run_threads(G, body)
    got = np.concatenate([lat.slab.get_angles() for lat in lats])
    assert (got == ref).all(), "initial state differs"
    for t in range(sweeps):
        shard.run_threads(G, lambda r, comm: lats[r].sweep(beta))
        b, lab, o = xo.sweep(ref, L, seed, t, beta)
        if t % check_every and t + 1 != sweeps:
            continue
        assert (np.concatenate([lat.slab.get_bonds() for lat in lats]) == b).all(), f"bonds differ at sweep {t}"
        assert (np.concatenate([lat.slab.get_labels() for lat in lats]) == lab).all(), f"labels differ at sweep {t}"
        assert (np.concatenate([lat.slab.get_angles() for lat in lats]) == ref).all(), f"angles differ at sweep {t}"
        res = shard.run_threads(G, lambda r, comm: lats[r].measure())
        for g in res:                                       # every rank holds the same global record
            for k in ("E", "Mx", "My", "Cx", "Sx", "Cy", "Sy"):
                assert abs(g[k] - getattr(o, k)) <= 1e-9 * N, (k, g[k], getattr(o, k))
            assert (g["n_bonds_x"], g["n_bonds_y"], g["n_clusters"]) == (o.n_bonds_x, o.n_bonds_y, o.n_clusters)
            assert g["sweep"] == t + 1
    for lat in lats:
        lat.slab.destroy()


@pytest.mark.parametrize("L,G,init,beta", [(128, 1, "hot", 1.12), (128, 2, "hot", 1.12), (256, 4, "hot", 1.12),
                                           (256, 2, "cold", 1.12), (256, 8, "hot", 0.7), (384, 3, "hot", 1.5),
                                           (192, 2, "hot", 1.12), (512, 4, "cold", 1.11996)])
def test_sharded_sweeps_equal_the_whole_lattice_oracle(xy, L, G, init, beta):
    _run(xy, L, G, seed=40 + L + G, init=init, beta=beta, sweeps=6)


def test_sharded_chain_large_clusters(xy):
    """cold start at low temperature: one cluster spans every slab for many sweeps (every cut root is overridden)"""
    _run(xy, 256, 4, seed=5, init="cold", beta=3.0, sweeps=8)


def test_sharded_beta_zero_and_huge(xy):
    _run(xy, 128, 2, seed=6, init="hot", beta=0.0, sweeps=2)
    _run(xy, 128, 4, seed=6, init="cold", beta=1e9, sweeps=2)


def test_sharded_longer_chain_L1024(xy):
    _run(xy, 1024, 4, seed=7, init="cold", beta=1.11996, sweeps=40, check_every=10)


def test_sharded_without_observables(xy):
    """the k_bonds variant without the fp64 sums (xy_set_obs_mode) on slabs, both tile widths"""
    _run(xy, 256, 2, seed=8, init="hot", beta=1.12, sweeps=5, obs_none=True, check_every=2)
    _run(xy, 192, 2, seed=8, init="hot", beta=1.12, sweeps=3, obs_none=True)


@pytest.mark.parametrize("L,G,init,obs_none", [(8192, 2, "hot", False), (8192, 8, "cold", True), (16384, 4, "hot", False)])
def test_sharded_large_lattices_take_the_32_row_strip_kernels(xy, L, G, init, obs_none):
    """L > 4096 selects k_bonds<4, 32, ..., kSlab> (long strips: halo row instead of the y wrap, bond bytes addressed
    from a base moved back by the slab's offset, whole-lattice Philox counters) and k_flip<4, 32, u32, kSlab> over
    thousands of tile rows per slab: the regime the paper shards in.  Chained sweeps, everything
    compared with the whole-lattice oracle (one sweep at L = 16384: an oracle sweep there takes a minute)."""
    _run(xy, L, G, seed=900 + G, init=init, beta=1.11996, sweeps=2 if L <= 8192 else 1, obs_none=obs_none)


def test_unequal_slabs(xy):
    """slabs of 32, 32 and 64 rows: nranks = 3 is not L / rows for any of them, so every rank's stitch table is the
    separately allocated one (the table inside the workspace is sized for equal slabs); three chained sweeps against
    the whole-lattice oracle"""
    from paper_1210_6116_b200 import shard
    L, seed, beta = 128, 77, 1.12
    rows, y_off = [32, 32, 64], [0, 32, 64]
    ref = xo.init(L, seed, xo.INIT_HOT)
    lats = shard.run_threads(3, lambda r, comm: shard.ShardedLattice(xy.SlabState(L, rows[r], y_off[r], seed, xy.INIT_HOT), comm))
    for t in range(3):
        shard.run_threads(3, lambda r, comm: lats[r].sweep(beta))
        b, lab, o = xo.sweep(ref, L, seed, t, beta)
        assert (np.concatenate([lat.slab.get_bonds() for lat in lats]) == b).all(), t
        assert (np.concatenate([lat.slab.get_labels() for lat in lats]) == lab).all(), t
        assert (np.concatenate([lat.slab.get_angles() for lat in lats]) == ref).all(), t
    for lat in lats:
        lat.slab.destroy()


def test_hot_slab_is_complete_before_any_exchange(xy):
    """a hot slab's halo row holds the initial values of the row below it from creation: the partial sums of freshly
    created slabs (no ShardedLattice, no exchange) add up to the observables of the whole hot lattice"""
    L, G, seed = 256, 4, 21
    o = xo.observe(xo.init(L, seed, xo.INIT_HOT), L)
    slabs = [xy.SlabState(L, L // G, r * (L // G), seed, xy.INIT_HOT) for r in range(G)]
    part = [s.measure() for s in slabs]
    for k in ("E", "Mx", "My", "Cx", "Sx", "Cy", "Sy"):
        assert abs(sum(getattr(p, k) for p in part) - getattr(o, k)) <= 1e-9 * L * L, k
    for s in slabs:
        s.destroy()


def test_slab_flip_with_a_foreign_record_is_reported_not_written(xy):
    """rank 0's slab handed the gathered records as if it were rank 1: its edge sites lie outside the slab; the stitch
    skips them (no out-of-bounds write) and the next blocking call says so; set_angles is refused between the phases"""
    import torch
    L, G = 128, 2
    slabs = [xy.SlabState(L, L // G, r * (L // G), 3, xy.INIT_HOT) for r in range(G)]
    for s in slabs:
        s.slab_label(1.12)
    with pytest.raises(xy.XYError) as e:
        slabs[0].set_angles(np.zeros(slabs[0].N, np.float32))
    assert e.value.code == -5
    gathered = torch.cat([s.edges for s in slabs])
    slabs[0].slab_flip(gathered, G, 1)                 # wrong rank
    with pytest.raises(xy.XYError) as e:
        slabs[0].measure()
    assert e.value.code == -1 and "outside the slab" in str(e.value)
    slabs[1].slab_flip(gathered, G, 1)                 # the right one: no complaint
    slabs[1].measure()
    slabs[1].get_labels()
    for s in slabs:
        s.destroy()


def test_slab_errors(xy):
    with pytest.raises(xy.XYError):
        xy.SlabState(128, 48, 0, 1)                 # rows not a multiple of 32
    with pytest.raises(xy.XYError):
        xy.SlabState(128, 64, 96, 1)                # beyond the lattice
    with pytest.raises(xy.XYError):
        xy.SlabState(128, 64, 0, 1, flags=xy.FLAG_LABELS64)
    s = xy.SlabState(128, 64, 64, 1)
    with pytest.raises(xy.XYError):
        s.sw_sweeps(1.0, 1)                         # a slab sweeps in two phases
    with pytest.raises(xy.XYError):
        import torch
        s.slab_flip(torch.zeros(2 * s.edges.numel(), dtype=torch.uint8, device="cuda"), 2, 0)   # no label phase yet
    s.destroy()


@pytest.mark.parametrize("L,G", [(128, 2), (256, 4), (256, 1)])
def test_sharded_pcc_equals_the_oracle_controller(xy, L, G):
    """the PCC driver on G slabs: beta trace equal to the oracle's whole-lattice run, final angles bit for bit"""
    from paper_1210_6116_b200 import shard
    seed, n, window = 17, 240, 20
    sg = xy.PccSchedule(n_sweeps=n, discard=20, window=window, dirs=1, dbeta0=1e-3, halve_every=100, dbeta_min=1e-6,
                        target=2 / np.pi)
    so = xo.PccSchedule(n_sweeps=n, discard=20, window=window, dirs=1, dbeta0=1e-3, halve_every=100, dbeta_min=1e-6,
                        target=2 / np.pi)
    ref_theta = xo.init(L, seed, xo.INIT_HOT)
    ref = xo.pcc_run(ref_theta, L, seed, 0, 1.05, so, trace_cap=n)

    def body(rank, comm):
        rows, y_off = shard.slab_rows(L, G, rank)
        slab = xy.SlabState(L, rows, y_off, seed, xy.INIT_HOT)
        slab.set_obs_mode(xy.OBS_NONE)               # the sums come from xy_slab_obs_partial, once per sweep
        return shard.ShardedLattice(slab, comm)
    lats = shard.run_threads(G, body)
    traces = [[] for _ in range(G)]

    def run(rank, comm):
        return lats[rank].pcc_run(1.05, sg, on_decision=lambda st: traces[rank].append(st.beta))
    finals = shard.run_threads(G, run)
    assert np.abs(ref["trace_bY"] - 2 / np.pi).min() > 1e-10          # no decision was a coin toss
    # the controller's beta AFTER decision k is the beta the next window runs at
    want_after = np.append(ref["trace_beta"][1:], ref["beta_final"])
    for r in range(G):
        assert finals[r].n_decisions == ref["n_decisions"] == (n - 20) // window
        assert finals[r].beta == ref["beta_final"] and finals[r].dbeta == ref["dbeta_final"]
        assert np.array_equal(np.array(traces[r]), want_after)
    got = np.concatenate([lat.slab.get_angles() for lat in lats])
    assert np.array_equal(got.view(np.uint32), ref_theta.view(np.uint32))
    for lat in lats:
        lat.slab.destroy()


@pytest.mark.parametrize("L,G", [(128, 2), (256, 4), (192, 3), (512, 8)])
def test_stitch_on_injected_bond_patterns(xy, L, G):
    """the label phase + stitch on adversarial bond sets (a serpentine that crosses every cut L/2 times, combs, stripes,
    wrap-only bonds, random densities): canonical labels of the G slabs equal the oracle's labels of the whole lattice"""
    import xy_inputs
    from paper_1210_6116_b200 import shard
    rng = np.random.default_rng(L + G)
    sets = [(k, xy_inputs.pattern_bonds(L, k)) for k in xy_inputs.BOND_PATTERNS]
    v_serp = np.zeros((L, L), np.uint8)                   # a snake running along the columns: crosses every cut L times
    v_serp[: L - 1, :] |= 2
    for x in range(L - 1):
        v_serp[L - 1 if x % 2 == 0 else 0, x] |= 1
    sets.append(("v_serpentine", v_serp.ravel()))
    sets += [(f"random{p}", (rng.random(L * L) < p).astype(np.uint8) | ((rng.random(L * L) < p).astype(np.uint8) << 1))
             for p in (0.1, 0.3, 0.5, 0.7, 0.9)]

    def body(rank, comm):
        rows, y_off = shard.slab_rows(L, G, rank)
        return shard.ShardedLattice(xy.SlabState(L, rows, y_off, 3, xy.INIT_HOT), comm)
    lats = shard.run_threads(G, body)
    for name, b in sets:
        want = xo.label(b, L)[0]

        def run(rank, comm, b=b):
            lat = lats[rank]
            rows, y_off = lat.slab.rows, lat.slab.y_off
            lat.slab.slab_label_bonds(b[y_off * L: (y_off + rows) * L])
            g = lat.comm.all_gather(lat.slab.edges)
            lat.slab.slab_flip(g.reshape(-1), G, rank)
            return lat.slab.get_labels()
        got = np.concatenate(shard.run_threads(G, run))
        assert (got == want).all(), name
    for lat in lats:
        lat.slab.destroy()
