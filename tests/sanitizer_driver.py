"""NOT a pytest (nothing collects it): the driver script of the range-checked build, run by hand as
profiles/r2_checked_build.md states.

Workload for compute-sanitizer (memcheck / racecheck / synccheck) and for the range-checked build
(XY_NVCC_EXTRA=-DXY_CHECKED python -m paper_1210_6116_b200.build), kept small on purpose:

    compute-sanitizer --tool memcheck  python tests/sanitizer_driver.py
    compute-sanitizer --tool racecheck python tests/sanitizer_driver.py

Two sweeps plus the getters at L = 64 and L = 1024 for both label widths, with the structure-factor sums
on and off and with the observables switched off: every kernel variant these sizes select runs at least
once.  The Potts sweep and the row-slab path follow.  Results are summarised in
profiles/r2_checked_build.md."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import paper_1210_6116_b200 as xy  # noqa: E402


def main():
    for L in (64, 1024):
        for flags in (0, xy.FLAG_LABELS64, xy.FLAG_FOURIER, xy.FLAG_LABELS64 | xy.FLAG_FOURIER):
            st = xy.XYState(L, 3, xy.INIT_HOT, flags=flags)
            st.sw_sweeps(1.12, 2)
            o = st.measure()
            st.get_bonds(); st.get_labels(); st.get_angles()
            inv = st.debug_check_labels()
            st.set_obs_mode(xy.OBS_NONE)
            st.sw_sweeps(1.12, 1)
            if flags & xy.FLAG_FOURIER:
                st.measure_fourier()
            print(L, flags, o.n_clusters, inv)
            st.destroy()
    if "--big" in sys.argv:                          # the bench workload and the odd-size variants
        for L, init, flags, n in ((16384, xy.INIT_COLD, 0, 30), (4160, xy.INIT_HOT, xy.FLAG_LABELS64, 10),
                                  (8192, xy.INIT_HOT, xy.FLAG_FOURIER, 10)):
            st = xy.XYState(L, 13, init, flags=flags)
            st.sw_sweeps(1.11996, n)
            print(L, flags, st.measure().n_clusters, st.debug_check_labels())
            st.destroy()
    # the Potts sweep and the row-slab path (two slabs of one process) on the same labeling kernels
    for L, q in ((64, 2), (192, 3), (1024, 5)):
        ps = xy.PottsState(L, q, 3, xy.INIT_HOT)
        ps.sweeps(1.0, 3)
        o = ps.measure()
        ps.get_bonds(); ps.get_labels(); ps.get_spins()
        print("potts", L, q, o.n_clusters, o.E)
        ps.destroy()
    from paper_1210_6116_b200 import shard
    for L, G in ((128, 2), (192, 2), (1024, 4)):
        def body(rank, comm):
            rows, y_off = shard.slab_rows(L, G, rank)
            return shard.ShardedLattice(xy.SlabState(L, rows, y_off, 3, xy.INIT_HOT), comm)
        lats = shard.run_threads(G, body)
        shard.run_threads(G, lambda r, comm: lats[r].sweep(1.12, 3))
        res = shard.run_threads(G, lambda r, comm: lats[r].measure())
        for lat in lats:
            lat.slab.get_labels(); lat.slab.get_bonds()
            lat.slab.destroy()
        print("slabs", L, G, res[0]["n_clusters"])
    counts, checked = xy.debug_check_counts()
    print("checked build:", checked, "range-check violations:", counts)
    assert sum(counts) == 0
    print("sanitizer driver done")


if __name__ == "__main__":
    main()
