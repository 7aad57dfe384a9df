"""Row-slab sharded sweep: the exchange around the per-rank kernels.

Rank r of G holds rows [r L/G, (r+1) L/G) of the L x L lattice as one slab state (include/xy.h, "row-slab sharding").
One sweep = local phase (direction, bonds, labels inside the slab, edge record) -> ALL-GATHER of the edge records
(17 L bytes per rank, into a buffer allocated once) -> stitch + flip on every rank -> every rank sends its first row
(4 L bytes) to its upper neighbour, whose halo row it is.  Observables are partial sums per slab; `measure` adds
them with one all-reduce.  This module is plumbing only: every step of the path runs in the kernels behind the slab
state; the transport is whatever `comm` wraps (torch.distributed with NCCL on the GPUs, gloo in the CPU test of this
logic, threads of one process for the single-GPU parity test).
"""
import threading

OBS_SUMS = ("E", "Mx", "My", "Cx", "Sx", "Cy", "Sy")
OBS_COUNTS = ("n_bonds_x", "n_bonds_y", "n_clusters")


def slab_rows(L, world, rank):
    """rows and first row of rank's slab: equal slabs, multiples of 32 rows"""
    if L % (32 * world) != 0:
        raise ValueError(f"L={L} does not split into {world} slabs of a multiple of 32 rows")
    rows = L // world
    return rows, rank * rows


class DistComm:
    """torch.distributed (backend nccl on the GPUs, gloo on CPU tensors).  The gathered buffers are allocated once per
    (shape, dtype, device) and reused by every sweep; the halo row travels point to point (only the lower neighbour's
    first row is needed), not through an all-gather."""

    def __init__(self, dist, rank, world):
        self.dist, self.rank, self.world = dist, rank, world
        self._gathered = {}

    def all_gather(self, t):
        """[world, *t.shape]; the returned tensor is this object's buffer and is overwritten by the next call with the
        same shape"""
        import torch
        t = t.contiguous()
        key = (tuple(t.shape), t.dtype, t.device)
        out = self._gathered.get(key)
        if out is None:
            out = self._gathered[key] = torch.empty(self.world * t.numel(), dtype=t.dtype, device=t.device)
        self.dist.all_gather_into_tensor(out, t.reshape(-1))      # flat in, flat out: what gloo and nccl both accept
        return out.view((self.world,) + tuple(t.shape))

    def all_reduce_sum(self, t):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return t

    def shift_up(self, send, recv):
        """recv <- the `send` of rank + 1 (periodic): every rank sends to rank - 1 and receives from rank + 1"""
        if self.world == 1:
            recv.copy_(send)
            return
        d = self.dist
        ops = [d.P2POp(d.isend, send, (self.rank - 1) % self.world), d.P2POp(d.irecv, recv, (self.rank + 1) % self.world)]
        for w in d.batch_isend_irecv(ops):
            w.wait()


class ThreadComm:
    """the ranks are threads of one process sharing one device: for the single-GPU parity test of the slab kernels.
    Host-side rendezvous only (a barrier between depositing and reading); no kernel waits on another."""

    class Shared:
        def __init__(self, world):
            self.world, self.slots, self.barrier = world, [None] * world, threading.Barrier(world)

    def __init__(self, shared, rank):
        self.s, self.rank, self.world = shared, rank, shared.world

    def all_gather(self, t):
        import torch
        self.s.slots[self.rank] = t
        self.s.barrier.wait()
        out = torch.stack([x.clone() for x in self.s.slots])
        self.s.barrier.wait()                       # nobody overwrites a slot before everyone has read it
        return out

    def all_reduce_sum(self, t):
        return self.all_gather(t).sum(dim=0)

    def shift_up(self, send, recv):
        self.s.slots[self.rank] = send
        self.s.barrier.wait()
        recv.copy_(self.s.slots[(self.rank + 1) % self.world])
        if recv.is_cuda:
            import torch
            torch.cuda.current_stream().synchronize()   # the copy has read the neighbour's row before it may sweep on
        self.s.barrier.wait()


class ShardedLattice:
    """One rank's part of the sharded lattice.  `slab` is a SlabState (or, in the CPU test of this logic, an object with
    the same methods and buffers on CPU tensors); `comm` one of the classes above."""

    def __init__(self, slab, comm):
        self.slab, self.comm = slab, comm
        self.rank, self.world = comm.rank, comm.world
        self.exchange_halo()

    def exchange_halo(self):
        self.comm.shift_up(self.slab.first_row, self.slab.halo_row)

    def sweep(self, beta, n=1):
        for _ in range(n):
            self.slab.slab_label(beta)
            gathered = self.comm.all_gather(self.slab.edges)
            self.slab.slab_flip(gathered.reshape(-1), self.world, self.rank)
            self.exchange_halo()

    def pcc_run(self, beta0, sched, on_decision=None):
        """The PCC driver (O8) on the sharded lattice: the controller runs replicated on every rank's device, fed after
        every measured sweep with the all-reduced sums of the new configuration (one 8-double all-reduce per sweep).
        Returns the controller state (binding.PccState) of this rank; all ranks hold the same one."""
        slab = self.slab
        slab.slab_pcc_setup(beta0, sched)
        for n in range(int(sched.n_sweeps)):
            slab.slab_label_pcc()
            gathered = self.comm.all_gather(slab.edges)
            slab.slab_flip(gathered.reshape(-1), self.world, self.rank)
            self.exchange_halo()
            if n >= sched.discard:
                slab.slab_obs_partial()
                slab.pcc_global.copy_(slab.pcc_partial)
                total = self.comm.all_reduce_sum(slab.pcc_global)       # in place with torch.distributed
                if total is not slab.pcc_global:
                    slab.pcc_global.copy_(total)
                slab.slab_pcc_feed()
                if on_decision is not None and (n - sched.discard + 1) % sched.window == 0:
                    on_decision(slab.pcc_get_state())
        return slab.pcc_get_state()

    def measure(self):
        """observables of the whole lattice: the slabs' partial sums added over the ranks"""
        import torch
        o = self.slab.measure()
        dev = self.slab.first_row.device
        sums = torch.tensor([float(getattr(o, k)) for k in OBS_SUMS], dtype=torch.float64, device=dev)
        cnts = torch.tensor([int(getattr(o, k)) for k in OBS_COUNTS], dtype=torch.int64, device=dev)
        sums = self.comm.all_reduce_sum(sums)
        cnts = self.comm.all_reduce_sum(cnts)
        out = {k: float(v) for k, v in zip(OBS_SUMS, sums.tolist())}
        out.update({k: int(v) for k, v in zip(OBS_COUNTS, cnts.tolist())})
        out["sweep"], out["beta"] = int(o.sweep), float(o.beta)
        return out


def run_threads(world, fn):
    """fn(rank, comm) on `world` threads of this process with a ThreadComm; returns the list of results"""
    shared = ThreadComm.Shared(world)
    res, err = [None] * world, [None] * world

    def body(r):
        try:
            res[r] = fn(r, ThreadComm(shared, r))
        except BaseException as e:                  # noqa: BLE001  (re-raised in the caller)
            err[r] = e
            shared.barrier.abort()
    ts = [threading.Thread(target=body, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    for e in err:
        if e is not None:
            raise e
    return res
