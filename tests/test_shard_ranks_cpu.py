"""Host logic of the row-slab sharded sweep (paper_1210_6116_b200/shard.py) on CPU: world_size-2 gloo process group.
The slab behind ShardedLattice is a stand-in written here from the oracle's pure functions on CPU tensors (the CUDA
slab state needs a GPU; its parity is tests/test_gpu_slab.py); what is under test is the exchange: who gathers what, in
which order, the record layout, the periodic cut between the last and the first rank, the halo rows, the all-reduce of
the partial sums.  After every sweep the gathered angles and canonical labels must equal the oracle's sweep of the
whole lattice bit for bit."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class OracleSlab:
    """rows [y_off, y_off + rows) of an L x L lattice, same interface as binding.SlabState, on CPU tensors."""

    def __init__(self, L, rows, y_off, seed, hot):
        import torch
        from oracle import xy_oracle as xo
        self.xo, self.L, self.rows, self.y_off, self.seed, self.T = xo, L, rows, y_off, seed, 0
        full = xo.init(L, seed, xo.INIT_HOT if hot else xo.INIT_COLD)
        self.buf = torch.zeros((rows + 1) * L, dtype=torch.float32)
        self.buf[: rows * L] = torch.from_numpy(full[y_off * L: (y_off + rows) * L].copy())
        self.first_row = self.buf[:L]
        self.halo_row = self.buf[rows * L:]
        self.edges = torch.zeros(17 * L, dtype=torch.uint8)
        self.labels = None

    def _embedded(self):
        """my rows and my halo row at their places in an otherwise empty whole lattice"""
        L, rows, y0 = self.L, self.rows, self.y_off
        full = np.zeros(L * L, np.float32)
        full[y0 * L: (y0 + rows) * L] = self.buf[: rows * L].numpy()
        yh = (y0 + rows) % L
        if self.rows < L:
            full[yh * L: (yh + 1) * L] = self.halo_row.numpy()
        return full

    def slab_label(self, beta):
        xo, L, rows, y0 = self.xo, self.L, self.rows, self.y_off
        self.beta, self.phi = beta, xo.phi(self.seed, self.T)
        b = xo.bonds(self._embedded(), L, beta, self.phi, self.seed, self.T)
        mine = np.zeros(L * L, np.uint8)
        mine[y0 * L: (y0 + rows) * L] = b[y0 * L: (y0 + rows) * L]
        self.bonds = mine[y0 * L: (y0 + rows) * L].copy()
        last = slice((y0 + rows - 1) * L, (y0 + rows) * L)
        ycut = (mine[last] >> 1) & 1
        mine[last] &= 1                                    # the y bonds of my last row cross the cut
        self.labels = xo.label(mine, L)[0][y0 * L: (y0 + rows) * L].copy()
        rec = np.zeros(17 * L, np.uint8)
        rec[: 8 * L] = self.labels[:L].astype("<u8").view(np.uint8)
        rec[8 * L: 16 * L] = self.labels[-L:].astype("<u8").view(np.uint8)
        rec[16 * L:] = ycut
        self.edges.copy_(__import__("torch").from_numpy(rec))

    def slab_flip(self, gathered, nranks, rank):
        xo, L = self.xo, self.L
        g = gathered.numpy().reshape(nranks, 17 * L)
        top = [g[r, : 8 * L].view("<u8") for r in range(nranks)]
        bot = [g[r, 8 * L: 16 * L].view("<u8") for r in range(nranks)]
        yb = [g[r, 16 * L:] for r in range(nranks)]
        parent = {}

        def find(a):
            parent.setdefault(a, a)
            while parent[a] != a:
                a = parent[a]
            return a
        for r in range(nranks):
            for x in np.flatnonzero(yb[r]):
                a, b = find(int(bot[r][x])), find(int(top[(r + 1) % nranks][x]))
                if a != b:
                    parent[max(a, b)] = min(a, b)
        canon = self.labels.copy()
        for loc in set(int(v) for v in top[rank]) | set(int(v) for v in bot[rank]):
            canon[self.labels == loc] = find(loc)
        self.canon = canon
        th = self.buf[: self.rows * L].numpy()
        A = xo.reflect_const(self.phi)
        coins = {int(rho): xo.flip_coin(self.seed, int(rho), self.T) for rho in np.unique(canon)}
        for i in np.flatnonzero(np.vectorize(coins.get)(canon)):
            th[i] = xo.reflect(th[i], A)
        self.n_clusters = int((canon == np.arange(self.y_off * L, (self.y_off + self.rows) * L)).sum())
        self.T += 1

    def measure(self):
        """partial sums of my sites; the y links of my last row reach into the halo row"""
        L, rows = self.L, self.rows
        th = self.buf.numpy().astype(np.float64).reshape(rows + 1, L)
        a, right, down = th[:rows], np.roll(th[:rows], -1, axis=1), th[1:]

        class O:
            pass
        o = O()
        o.Mx, o.My = np.cos(a).sum(), np.sin(a).sum()
        o.Cx, o.Sx = np.cos(a - right).sum(), np.sin(a - right).sum()
        o.Cy, o.Sy = np.cos(a - down).sum(), np.sin(a - down).sum()
        o.E = -(o.Cx + o.Cy)
        o.n_bonds_x, o.n_bonds_y = int((self.bonds & 1).sum()), int(((self.bonds >> 1) & 1).sum())
        o.n_clusters, o.sweep, o.beta = self.n_clusters, self.T, self.beta
        return o


def _worker(rank, world, port, L, hot, beta, sweeps, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from oracle import xy_oracle as xo
    from paper_1210_6116_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    comm = shard.DistComm(dist, rank, world)
    rows, y_off = shard.slab_rows(L, world, rank)
    seed = 31
    lat = shard.ShardedLattice(OracleSlab(L, rows, y_off, seed, hot), comm)
    ref = xo.init(L, seed, xo.INIT_HOT if hot else xo.INIT_COLD)
    ok = True
    for t in range(sweeps):
        lat.sweep(beta)
        _, lab, o = xo.sweep(ref, L, seed, t, beta)
        th = comm.all_gather(lat.slab.buf[: rows * L]).reshape(-1).numpy()
        cl = comm.all_gather(torch.from_numpy(lat.slab.canon)).reshape(-1).numpy()
        g = lat.measure()
        ok = ok and (th == ref).all() and (cl == lab).all()
        ok = ok and all(abs(g[k] - getattr(o, k)) <= 1e-9 * L * L for k in ("E", "Mx", "My", "Cx", "Sx", "Cy", "Sy"))
        ok = ok and (g["n_bonds_x"], g["n_bonds_y"], g["n_clusters"]) == (o.n_bonds_x, o.n_bonds_y, o.n_clusters)
        ok = ok and g["sweep"] == t + 1
    out[rank] = bool(ok)
    dist.destroy_process_group()


def _run(L, hot, beta, sweeps, world=2):
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, L, hot, beta, sweeps, out), nprocs=world, join=True)
        res = dict(out)
    assert res == {r: True for r in range(world)}, res


def test_sharded_exchange_world2_hot():
    _run(64, True, 1.12, 4)


def test_sharded_exchange_world2_cold_large_clusters():
    _run(64, False, 2.0, 4)


def test_slab_rows():
    sys.path.insert(0, ROOT)
    from paper_1210_6116_b200 import shard
    assert shard.slab_rows(256, 4, 3) == (64, 192)
    assert shard.slab_rows(65536, 8, 0) == (8192, 0)
    import pytest
    with pytest.raises(ValueError):
        shard.slab_rows(192, 4, 0)                        # 48 rows per slab: not a multiple of 32
