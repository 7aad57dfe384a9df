#!/usr/bin/env python
"""bench.py -- throughput of the Swendsen-Wang sweep of the 2D XY model (arXiv 1210.6116) on B200.

    python bench.py --gpus N --steps K --warmup W [--workload cfg4] [--impl reference]

A "step" is ONE whole sweep (projection + bond activation + cluster labeling + flip, with the
observables of every sweep reduced on the device) of one lattice.  Metric: spin updates/s =
L^2 * sweeps / time (BASELINE.json).  Default workload: BASELINE config 4 (L = 16384, beta = 1.11996,
cold start, 500 thermalisation sweeps before anything is timed) -- the size the north_star's
>= 60 % HBM target is stated for.  The path does not shard (clusters span the lattice): --gpus N
runs N independent replicas (seed + rank), one process per GPU, no data-path collective.

One JSON line on stdout (rank 0).  `value`: device-resident throughput; `e2e`: the same through the
C-ABI with HOST buffers every step (xy_set_angles from pinned memory, one sweep, xy_get_angles +
xy_measure back); `roofline`: dominant kernel, algorithmic bytes / CUDA-event time against the
measured HBM copy bandwidth; `cpu_baseline`: the CPU oracle, as it stands, on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import xy_inputs  # noqa: E402

METRIC = "SW spin updates/s"
UNIT = "spin updates/s"

WORKLOADS = {
    # name: (config index in BASELINE.json, L, init, seed, beta, thermalisation sweeps)
    "cfg1": (0, 64, "hot", 1, 1.12, 0),
    "cfg2": (1, 1024, "cold", 7, 1.12, 2000),
    "cfg3": (2, 4096, "hot", 11, 1.11097, 200),      # fixed beta near the PCC run's end point
    "cfg4": (3, 16384, "cold", 13, 1.11996, 500),
    "cfg5": (4, 65536, "hot", 17, 1.11996, 0),
    "L8192": (None, 8192, "cold", 13, 1.11996, 500),
    "L32768": (None, 32768, "hot", 17, 1.11996, 50),
}
CPU_SAMPLE_L = 1024           # the oracle's bounded sample: a 1024^2 lattice of the same model


def bytes_model(L, label_bytes, tw, th):
    """Algorithmic (compulsory) DRAM bytes per site per launch of each kernel, DESIGN.md section 6."""
    w = label_bytes
    return {
        "k_bonds": 4.0 + 0.25,                                  # theta read, packed bond bits written
        "k_label": 0.25 + w + 0.125,                            # bond bits read, provisional label + root bit written
        "k_merge": (tw + th) * (2.0 * w + 0.125) / (tw * th),   # two labels + the bond bit per tile-edge site
        "k_flip": w + 0.125 + 4.0 + 4.0,                        # label + root bit read, theta read, theta written
    }


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_rate(beta, budget_s=20.0, max_sweeps=None):
    """the oracle as it stands, single thread, on a 1024^2 cold-start lattice; returns (rate, sweeps, secs)."""
    from oracle import xy_oracle as xo
    L = CPU_SAMPLE_L
    th = xo.init(L, 13, xo.INIT_COLD)
    t0 = time.perf_counter()
    xo.run(th, L, 13, 0, beta, 1, series=True)
    per = time.perf_counter() - t0
    n = max(2, int(budget_s / max(per, 1e-3)))
    if max_sweeps:
        n = min(n, max_sweeps)
    t0 = time.perf_counter()
    xo.run(th, L, 13, 1, beta, n, series=True)
    dt = time.perf_counter() - t0
    return L * L * n / dt, n, dt


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_oracle_all_cores(beta, budget_s=15.0):
    """nproc independent oracle replicas (one per thread, own lattice and seed; ctypes releases the GIL), the way
    a CPU would parallelise this Monte Carlo: aggregate spin updates/s."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import xy_oracle as xo
    L = CPU_SAMPLE_L
    ncores = os.cpu_count() or 1
    t0 = time.perf_counter()
    xo.run(xo.init(L, 13, xo.INIT_COLD), L, 13, 0, beta, 1, series=True)
    per = time.perf_counter() - t0
    n = max(2, int(budget_s / max(per, 1e-3) / 1.5))       # all cores busy: expect some slowdown per replica

    def replica(r):
        th = xo.init(L, 100 + r, xo.INIT_COLD)
        xo.run(th, L, 100 + r, 0, beta, n, series=True)

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=ncores) as ex:
        list(ex.map(replica, range(ncores)))
    dt = time.perf_counter() - t0
    return ncores * L * L * n / dt, ncores, n, dt


def issue_model(workload):
    """warp instructions per launch of each kernel, from the committed ncu summary (profiles/instr.csv)"""
    out = {}
    path = os.path.join(ROOT, "profiles", "instr.csv")
    if os.path.exists(path):
        try:
            for row in open(path).read().split()[1:]:
                w, kname, n = row.split(",")
                if w == workload:
                    out[kname] = float(n)
        except Exception:
            return {}
    return out


def timed_leg(xy, torch, L, init, seed, beta, flags=0, therm=0, warm=3, K=20, obs="all", per_sweep=False, check=False):
    """one extra workload of the `also` block: K sweeps timed with CUDA events after therm + warm untimed sweeps;
    per_sweep: an event pair around every sweep (time series); check: the device-side label invariants after every
    timed sweep (outside the event pairs)."""
    N = L * L
    lb = 8 if flags & xy.FLAG_LABELS64 else 4
    tw, th = (128, 32) if L % 128 == 0 else (64, 32)
    st = xy.XYState(L, seed, xy_inputs.INIT_CODE[init], flags=flags)
    if obs == "none":
        st.set_obs_mode(xy.OBS_NONE)
    if therm + warm:
        st.sw_sweeps(beta, therm + warm)
    torch.cuda.synchronize()
    bad = 0
    if per_sweep or check:
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K)]
        for k in range(K):
            ev[2 * k].record()
            st.sw_sweeps(beta, 1)
            ev[2 * k + 1].record()
            if check:
                inv = st.debug_check_labels()
                bad += inv["label_above_index"] + inv["root_not_fixed"] + inv["x_bond_split"] + inv["y_bond_split"]
        torch.cuda.synchronize()
        times = sorted(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(K))
        ms = sum(times)
    else:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        st.sw_sweeps(beta, K)
        e1.record()
        torch.cuda.synchronize()
        ms, times = e0.elapsed_time(e1), None
    o = st.measure()
    st.destroy()
    del st
    torch.cuda.empty_cache()
    bps = sum(bytes_model(L, lb, tw, th).values())
    peak, _ = measured_peaks()
    out = {"L": L, "init": init, "seed": seed, "beta": beta, "label_bytes": lb, "observables": obs, "untimed_sweeps": therm + warm,
           "steps": K, "ms_per_step": ms / K, "updates_per_s": N * K / (ms * 1e-3), "bytes_per_site": bps,
           "sweep_roofline_frac": bps * N * K / (ms * 1e-3) / 1e9 / peak,
           "frac_on_survey_R0": (12.5 + 4 * lb) * N * K / (ms * 1e-3) / 1e9 / peak,
           "bond_density": (o.n_bonds_x + o.n_bonds_y) / (2 * N), "clusters_per_site": o.n_clusters / N}
    if (4 + lb) * N < 4 * 126e6:
        out["note"] = "working set comparable to the 126 MB L2: not an HBM measurement"
    if times:
        out["per_sweep_ms"] = {"min": times[0], "median": times[len(times) // 2], "max": times[-1]}
    if check:
        out["label_invariant_violations"] = int(bad)
    return out


def labeling_only(xy, torch, L, kinds=("all_on", "h_stripes", "serpentine"), reps=3):
    """the labeling kernels alone (k_label + k_merge, xy_label_bonds) on adversarial bond sets: ms per launch"""
    st = xy.XYState(L, 1, xy.INIT_COLD)
    st.debug_kernel_timing(True)
    out = {}
    for kind in kinds:
        b = xy_inputs.pattern_bonds(L, kind)
        st.label_bonds(b)
        st.get_kernel_times()
        for _ in range(reps):
            st.label_bonds(b)
        kt = st.get_kernel_times()
        inv = st.debug_check_labels()
        out[kind] = {"k_label_ms": kt["k_label"]["ms"] / reps, "k_merge_ms": kt["k_merge"]["ms"] / reps,
                     "clusters": inv["n_roots"],
                     "violations": inv["label_above_index"] + inv["root_not_fixed"] + inv["x_bond_split"] + inv["y_bond_split"]}
        del b
    st.debug_kernel_timing(False)
    st.destroy()
    torch.cuda.empty_cache()
    return out


def potts_leg(xy, torch, L=16384, q=3, seed=13, therm=100, K=50):
    """q-state Potts sweep at the self-dual point beta_c = ln(1 + sqrt q): the XY sweep's
    k_label / k_merge between k_potts_bonds and k_potts_flip; u32 labels, one byte per spin."""
    import math
    beta = math.log(1.0 + math.sqrt(q))
    N = L * L
    st = xy.PottsState(L, q, seed, xy.INIT_HOT)
    st.sweeps(beta, therm)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    st.sweeps(beta, K)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    o = st.measure()
    st.destroy()
    torch.cuda.empty_cache()
    # spins 1 B read (+ halo re-reads from L2) and bits 0.25 written; label pass as in the XY sweep; flip: labels 4,
    # root bits 0.125, spins 1 written
    bps = (1.0 + 0.25) + (0.25 + 4 + 0.125) + (128 + 32) * (2 * 4 + 0.125) / (128 * 32) + (4 + 0.125 + 1.0)
    peak, _ = measured_peaks()
    return {"L": L, "q": q, "beta": beta, "untimed_sweeps": therm, "steps": K, "ms_per_step": ms / K,
            "updates_per_s": N * K / (ms * 1e-3), "bytes_per_site": bps,
            "sweep_roofline_frac": bps * N * K / (ms * 1e-3) / 1e9 / peak,
            "E_per_site": o.E / N, "bond_density": (o.n_bonds_x + o.n_bonds_y) / (2 * N), "clusters_per_site": o.n_clusters / N}


def run_sharded(args, xy, torch, grp, rank, local_rank, world):
    """--shard: the workload's lattice as `world` row slabs, one per GPU (strong scaling)."""
    from paper_1210_6116_b200 import shard
    cfg_idx, L, init, seed, beta, therm = WORKLOADS[args.workload]
    if args.beta is not None:
        beta = args.beta
    N, K, W = L * L, args.steps, max(args.warmup, 3)
    rows, y_off = shard.slab_rows(L, world, rank)
    slab = xy.SlabState(L, rows, y_off, seed, xy_inputs.INIT_CODE[init])
    if args.obs == "none":
        slab.set_obs_mode(xy.OBS_NONE)
    if world > 1:
        comm = shard.DistComm(grp.dist, rank, world)
    else:
        comm = shard.ThreadComm(shard.ThreadComm.Shared(1), 0)
    lat = shard.ShardedLattice(slab, comm)
    lat.sweep(beta, therm + W)
    grp.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = slab.get_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    grp.barrier()
    e0.record()
    lat.sweep(beta, K)
    e1.record()
    grp.barrier()
    ms = grp.max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop()
    launches = slab.get_launch_count() - launches0
    obs = lat.measure()
    if rank == 0:
        line = {
            "metric": METRIC, "value": N * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"{args.workload}: ONE 2D XY lattice L={L} as {world} row slab(s) of {rows} rows, {init} start "
                                   f"seed {seed}, beta={beta}, {therm} thermalisation sweeps untimed",
                       "L": L, "beta": beta, "parallelism": f"row slabs x{world} (shard.py)",
                       "exchange_bytes_per_sweep_per_rank": {"all_gather_cut_records": 17 * L, "send_recv_first_row": 4 * L}},
            "clocks": clocks, "gpu_launches": int(launches),
            "observables": {"sweep": obs["sweep"], "E_per_site": obs["E"] / N, "m2": (obs["Mx"] ** 2 + obs["My"] ** 2) / N ** 2,
                            "bond_density": (obs["n_bonds_x"] + obs["n_bonds_y"]) / (2 * N), "clusters_per_site": obs["n_clusters"] / N},
        }
        print(json.dumps(line), flush=True)
    slab.destroy()


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import xy_oracle as xo
    _, Lw, init, seed, beta, _ = WORKLOADS[args.workload]
    L = CPU_SAMPLE_L
    th = xo.init(L, seed, xo.INIT_COLD if init == "cold" else xo.INIT_HOT)
    t = 0
    for _ in range(args.warmup):
        xo.run(th, L, seed, t, beta, 1, series=True)
        t += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        xo.run(th, L, seed, t, beta, 1, series=True)
        t += 1
    dt = time.perf_counter() - t0
    val = L * L * args.steps / dt
    sample = f"each step = one oracle sweep of a {L}x{L} lattice of the same model and beta (1/{(Lw // L) ** 2} of the workload's sites), single thread"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: L={Lw} beta={beta} {init} start (timed on the bounded sample)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


class RankGroup:
    """The multi-process plumbing of --gpus N: N independent replicas (seed + rank), one process per
    GPU, no data-path collective.  The process group serves only the barrier around the timed region
    and the max-over-ranks of the device time.  backend "nccl" on the GPUs; "gloo" with device "cpu"
    in the CPU tests (tests/test_bench_ranks_cpu.py)."""

    def __init__(self, rank, world, backend="nccl", device=None, sync=None):
        self.rank, self.world, self.device, self.sync = rank, world, device, sync
        self.dist = None
        if world > 1:
            import torch
            import torch.distributed as dist
            kw = {"device_id": device} if backend == "nccl" else {}
            dist.init_process_group(backend, rank=rank, world_size=world, **kw)
            self.dist, self.torch = dist, torch

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        if self.sync is not None:
            self.sync()

    def max_over_ranks(self, x):
        if self.dist is None:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def replica_seed(seed, rank):
    return seed + rank


def whole_job_value(world, N, K, ms):
    """spin updates/s of the whole job: every replica did K sweeps of N sites in (max over ranks) ms."""
    return world * N * K / (ms * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(WORKLOADS))
    ap.add_argument("--labels64", action="store_true", help="hold labels as 64-bit words")
    ap.add_argument("--fourier", action="store_true",
                    help="also reduce the structure-factor sums of every sweep (xi_2nd; XY_FLAG_FOURIER)")
    ap.add_argument("--beta", type=float, default=None, help="override the workload's beta (sensitivity runs)")
    ap.add_argument("--obs", default="all", choices=["all", "none"],
                    help="none: time the sweeps with the observable sums switched off (xy_set_obs_mode); not the headline")
    ap.add_argument("--repeats", type=int, default=3,
                    help="timed runs of K sweeps, each from a re-created state; the median is reported")
    ap.add_argument("--e2e-steps", type=int, default=None)
    ap.add_argument("--shard", action="store_true",
                    help="ONE lattice split into --gpus row slabs (SURVEY 8(f) #3): strong scaling, NCCL all-gather of the "
                         "cut records and first rows every sweep; with --gpus 1 the single slab stitches onto itself")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true",
                    help="skip the `also` block (configs 3 and 5, masked-observable variants, adversarial labeling)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import paper_1210_6116_b200 as xy

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    grp = RankGroup(rank, world, "nccl", torch.device("cuda", local_rank), torch.cuda.synchronize)
    barrier, max_over_ranks = grp.barrier, grp.max_over_ranks

    if args.shard:
        run_sharded(args, xy, torch, grp, rank, local_rank, world)
        grp.close()
        return

    cfg_idx, L, init, seed, beta, therm = WORKLOADS[args.workload]
    if args.beta is not None:
        beta = args.beta
    N = L * L
    flags = (xy.FLAG_LABELS64 if args.labels64 else 0) | (xy.FLAG_FOURIER if args.fourier else 0)
    label_bytes = 8 if args.labels64 else 4
    tw, th = (128, 32) if L % 128 == 0 else (64, 32)
    K, W = args.steps, max(args.warmup, 0)

    # ---- timed region 1: K sweeps, configuration resident in HBM; --repeats runs, each from a re-created state
    #      (same seed, thermalisation and warm-up: the trajectory is deterministic, only the machine varies), the
    #      MEDIAN run is the reported one (SURVEY.md 8(d) timing protocol) ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    runs, st = [], None
    for rep in range(max(args.repeats, 1)):
        if st is not None:
            st.destroy()
            st = None
        st = xy.XYState(L, replica_seed(seed, rank), xy_inputs.INIT_CODE[init], flags=flags)
        if args.obs == "none":
            st.set_obs_mode(xy.OBS_NONE)
        if therm:
            st.sw_sweeps(beta, therm)
        st.sw_sweeps(beta, W)
        torch.cuda.synchronize()
        launches0 = st.get_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        st.sw_sweeps(beta, K)
        e1.record()
        barrier()
        runs.append((max_over_ranks(e0.elapsed_time(e1)), st.get_launch_count() - launches0))
    clocks = sampler.stop()
    ms, launches = sorted(runs)[len(runs) // 2]
    value = whole_job_value(world, N, K, ms)
    obs = st.measure()

    # ---- timed region 2: the same K sweeps with CUDA events around every kernel ----
    st.debug_kernel_timing(True)
    barrier()
    st.sw_sweeps(beta, K)
    kt = st.get_kernel_times()
    st.debug_kernel_timing(False)
    peak, peak_src = measured_peaks()
    model = bytes_model(L, label_bytes, tw, th)
    kern = {}
    tot_ms = sum(v["ms"] for v in kt.values())
    for name, v in kt.items():
        avg = v["ms"] / max(v["launches"], 1)
        gbs = model[name] * N / (avg * 1e-3) / 1e9 if avg > 0 else 0.0
        kern[name] = {"avg_ms": avg, "share": v["ms"] / tot_ms if tot_ms else 0.0,
                      "bytes_per_site": model[name], "achieved_gbs": gbs, "frac": gbs / peak}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"])
    sweep_bytes = sum(model.values())
    sweep_gbs = sweep_bytes * N * K / (ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")      # workload,kernel,dram_bytes_per_launch (from ncu)
    if os.path.exists(tpath):
        try:
            for row in open(tpath).read().split()[1:]:
                w, kname, nbytes = row.split(",")
                if w == args.workload and kname == dom:
                    traffic = int(nbytes)
        except Exception:
            traffic = None
    # issue-rate roofline beside the HBM one: warp instructions per launch (ncu, profiles/instr.csv) over the
    # time the kernel took, against one warp instruction per cycle and scheduler
    imodel = issue_model(args.workload)
    sm_mhz = clocks.get("sm_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
    issue_peak = sms * 4 * sm_mhz * 1e6
    for name in kern:
        if name in imodel and kern[name]["avg_ms"] > 0:
            kern[name]["warp_instr_per_launch"] = imodel[name]
            kern[name]["issue_frac"] = imodel[name] / (kern[name]["avg_ms"] * 1e-3) / issue_peak
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["achieved_gbs"], "peak": peak,
                "unit": "GB/s", "frac": kern[dom]["frac"], "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": model[dom] * N,
                "limited_by": "instruction issue / shared-memory wavefronts, not DRAM (profiles/r3_cfg4.md): the HBM "
                              "fraction is this kernel's distance from its byte floor",
                "issue": {"warp_instr_per_launch": imodel.get(dom), "peak_warp_instr_per_s": issue_peak,
                          "frac": kern[dom].get("issue_frac")}}

    # ---- e2e: host buffers through the C-ABI every step ----
    e2e = None
    if not args.no_e2e:
        ke = args.e2e_steps or max(3, min(K, 10))
        host = torch.empty(N, dtype=torch.float32, pin_memory=True)
        st.get_angles(host)
        for _ in range(2):
            st.set_angles(host); st.sw_sweeps(beta, 1); st.get_angles(host); st.measure()
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            st.set_angles(host)          # H2D from pinned memory (synchronises)
            st.sw_sweeps(beta, 1)
            st.get_angles(host)          # D2H
            st.measure()                 # D2H of the sweep's record
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0)
        e2e = {"value": world * N * ke / dt, "unit": UNIT, "h2d_bytes_per_step": N * 4,
               "d2h_bytes_per_step": N * 4 + 104, "steps": ke, "ms_per_step": dt / ke * 1e3}
        del host

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, n, dt = cpu_oracle_rate(beta, budget_s=12.0)
        arate, ncores, an, adt = cpu_oracle_all_cores(beta, budget_s=12.0)
        cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{n} oracle sweeps of a {CPU_SAMPLE_L}x{CPU_SAMPLE_L} cold-start lattice at beta={beta} "
                         f"({dt:.1f} s, single thread; 1/{(L // CPU_SAMPLE_L) ** 2 if L >= CPU_SAMPLE_L else 1} of the workload's sites)",
               "all_cores": {"value": arate, "unit": UNIT, "cores": ncores, "cpu": cpu_model(),
                             "sample": f"{ncores} independent replicas (one thread each, own seed) x {an} oracle sweeps of a "
                                       f"{CPU_SAMPLE_L}x{CPU_SAMPLE_L} lattice, {adt:.1f} s"}}

    # ---- also: the ends of the metric's L range, the masked-observable variants, adversarial labeling ----
    also = None
    if rank == 0 and world == 1 and not args.no_also and args.workload == "cfg4":
        st.destroy()
        st = None
        torch.cuda.empty_cache()
        c3, c5 = WORKLOADS["cfg3"], WORKLOADS["cfg5"]
        also = {
            "cfg4_observables_off": timed_leg(xy, torch, L, init, seed, beta, therm=therm, warm=W, K=min(K, 50), obs="none"),
            "cfg3_L4096": timed_leg(xy, torch, c3[1], c3[2], c3[3], c3[4], therm=c3[5], warm=W, K=200),
            "cfg5_L65536_i64_labels": timed_leg(xy, torch, c5[1], c5[2], c5[3], c5[4], flags=xy.FLAG_LABELS64, warm=0, K=200,
                                                per_sweep=True, check=True),
            "cfg5_L65536_u32_labels": timed_leg(xy, torch, c5[1], c5[2], c5[3], c5[4], warm=0, K=200, per_sweep=True),
            "cfg5_L65536_i64_cold_100_warmup": timed_leg(xy, torch, c5[1], "cold", c5[3], c5[4], flags=xy.FLAG_LABELS64,
                                                         warm=100, K=20, per_sweep=True),
            "cfg5_L65536_i64_observables_off": timed_leg(xy, torch, c5[1], c5[2], c5[3], c5[4], flags=xy.FLAG_LABELS64,
                                                         warm=20, K=20, obs="none"),
            "labeling_only_L16384": labeling_only(xy, torch, 16384),
            "potts_q3_L16384": potts_leg(xy, torch),
            "note": "value / ms_per_step above are config 4 with all six sums on; entries here are labelled variants, "
                    "never the headline.  cfg5 is timed from the hot start as BASELINE config 5 states (its first "
                    "sweeps are transient: see per_sweep_ms)",
        }

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "repeats": {"n": len(runs), "ms_per_step": [r[0] / K for r in runs],
                                               "min": min(r[0] for r in runs) / K, "max": max(r[0] for r in runs) / K,
                                               "reported": "median"},
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE config {cfg_idx + 1 if cfg_idx is not None else '-'} ({args.workload}): "
                                   f"2D XY L={L} periodic, {init} start seed {seed}, beta={beta}, "
                                   f"{therm} thermalisation sweeps untimed",
                       "L": L, "beta": beta, "label_bytes": label_bytes, "fourier_sums": bool(args.fourier), "tile": f"{tw}x{th}",
                       "replicas": world, "parallelism": "replicas only (the path does not shard)",
                       "l2": "working set %.2f GiB per sweep >> 126 MB L2, no flush needed" % ((4 + label_bytes + 0.25) * N / 2 ** 30)
                       if (4 + label_bytes) * N > 4 * 126e6 else "working set fits L2: number is NOT an HBM measurement"},
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
            "kernels": kern, "also": also,
            "sweep_roofline": {"bytes_per_site": sweep_bytes, "achieved_gbs": sweep_gbs, "frac": sweep_gbs / peak,
                               "floor_bytes_per_site": 8.0 + 2 * label_bytes,
                               # SURVEY.md 8(d)'s reference model R0 (five separate passes incl. a flatten pass this
                               # design does not have): the same time against 12.5 + 4 w = 28.5 / 44.5 B per site
                               "survey_R0_bytes_per_site": 12.5 + 4 * label_bytes,
                               "frac_on_survey_R0": (12.5 + 4 * label_bytes) * N * K / (ms * 1e-3) / 1e9 / peak,
                               "ns_per_site": ms * 1e6 / (K * N)},
            "observables": {"sweep": int(obs.sweep), "E_per_site": obs.E / N,
                            "m2": (obs.Mx ** 2 + obs.My ** 2) / N ** 2,
                            "bond_density": (obs.n_bonds_x + obs.n_bonds_y) / (2 * N),
                            "clusters_per_site": obs.n_clusters / N},
        }
        print(json.dumps(line), flush=True)
    if st is not None:
        st.destroy()
    grp.close()


if __name__ == "__main__":
    main()
