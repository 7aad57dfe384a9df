"""ctypes binding of include/xy.h: argument marshalling only (same names as the C calls).

PyTorch is used for device memory (the workspace tensor handed to xy_create_ex), pinned host
buffers and streams -- plumbing, not arithmetic.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libxy_b200.so")

INIT_COLD, INIT_HOT = 0, 1
OBS_NONE, OBS_ALL = 0, 1
FLAG_LABELS64 = 1
FLAG_FOURIER = 2


class XYError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"xy error {code}: {msg}")
        self.code = code


def lib_path():
    return _LIB_PATH


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_1210_6116_b200.build` "
            "(nvcc, sm_100a).  This package has no CPU fallback.")
    return C.CDLL(_LIB_PATH)


_lib = _load()


class Obs(C.Structure):
    _fields_ = [("sweep", C.c_uint64), ("beta", C.c_double),
                ("E", C.c_double), ("Mx", C.c_double), ("My", C.c_double),
                ("Cx", C.c_double), ("Sx", C.c_double), ("Cy", C.c_double), ("Sy", C.c_double),
                ("n_bonds_x", C.c_uint64), ("n_bonds_y", C.c_uint64), ("n_clusters", C.c_uint64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


OBS_DTYPE = np.dtype([("sweep", "<u8"), ("beta", "<f8"), ("E", "<f8"), ("Mx", "<f8"), ("My", "<f8"),
                      ("Cx", "<f8"), ("Sx", "<f8"), ("Cy", "<f8"), ("Sy", "<f8"),
                      ("n_bonds_x", "<u8"), ("n_bonds_y", "<u8"), ("n_clusters", "<u8")])
assert OBS_DTYPE.itemsize == C.sizeof(Obs)


class Fourier(C.Structure):
    _fields_ = [("sweep", C.c_uint64), ("Fx", C.c_double * 4), ("Fy", C.c_double * 4)]


FOURIER_DTYPE = np.dtype([("sweep", "<u8"), ("Fx", "<f8", (4,)), ("Fy", "<f8", (4,))])
assert FOURIER_DTYPE.itemsize == C.sizeof(Fourier)


class PccSchedule(C.Structure):
    _fields_ = [("n_sweeps", C.c_uint64), ("discard", C.c_uint64),
                ("window", C.c_uint32), ("dirs", C.c_uint32),
                ("dbeta0", C.c_double), ("halve_every", C.c_uint64),
                ("dbeta_min", C.c_double), ("target", C.c_double)]


class _PccOut(C.Structure):
    _fields_ = [("beta_final", C.c_double), ("dbeta_final", C.c_double), ("beta_mean", C.c_double),
                ("n_decisions", C.c_uint64),
                ("trace_beta", C.POINTER(C.c_double)), ("trace_bY", C.POINTER(C.c_double)),
                ("trace_cap", C.c_uint64), ("trace_len", C.c_uint64)]


class PccState(C.Structure):
    _fields_ = [("beta", C.c_double), ("dbeta", C.c_double), ("acc_e", C.c_double), ("acc_s2", C.c_double),
                ("k", C.c_uint64), ("n_decisions", C.c_uint64),
                ("stage_sum", C.c_double), ("last_sum", C.c_double), ("stage_cnt", C.c_uint64), ("last_cnt", C.c_uint64),
                ("sum_m2", C.c_double), ("sum_chik", C.c_double), ("n_acc", C.c_uint64)]


_vp = C.c_void_p
_SIGS = {
    "xy_create": [C.POINTER(_vp), C.c_uint32, C.c_uint64, C.c_int],
    "xy_create_ex": [C.POINTER(_vp), C.c_uint32, C.c_uint64, C.c_int, C.c_uint32, _vp, C.c_size_t],
    "xy_workspace_bytes": [C.c_uint32, C.c_uint32, C.POINTER(C.c_size_t)],
    "xy_sw_sweeps": [_vp, C.c_double, C.c_uint64, _vp],
    "xy_measure": [_vp, C.POINTER(Obs)],
    "xy_pcc_run": [_vp, C.c_double, C.c_double, C.POINTER(PccSchedule), C.POINTER(_PccOut)],
    "xy_pcc_continue": [_vp, C.POINTER(PccSchedule), C.POINTER(_PccOut)],
    "xy_pcc_get_state": [_vp, C.POINTER(PccState)],
    "xy_pcc_set_state": [_vp, C.POINTER(PccState)],
    "xy_destroy": [_vp],
    "xy_get_angles": [_vp, _vp, C.c_size_t],
    "xy_get_angles_range": [_vp, _vp, C.c_uint64, C.c_size_t],
    "xy_get_labels_range": [_vp, _vp, C.c_uint64, C.c_size_t],
    "xy_get_bonds_range": [_vp, _vp, C.c_uint64, C.c_size_t],
    "xy_debug_check_labels": [_vp, C.POINTER(C.c_uint64)],
    "xy_set_obs_mode": [_vp, C.c_int],
    "xy_set_angles": [_vp, _vp, C.c_size_t],
    "xy_get_labels": [_vp, _vp, C.c_size_t],
    "xy_get_bonds": [_vp, _vp, C.c_size_t],
    "xy_get_series": [_vp, _vp, C.c_uint64, C.c_uint64],
    "xy_measure_fourier": [_vp, C.POINTER(Fourier)],
    "xy_get_fourier_series": [_vp, _vp, C.c_uint64, C.c_uint64],
    "xy_series_capacity": [_vp, C.POINTER(C.c_uint64)],
    "xy_get_sweep": [_vp, C.POINTER(C.c_uint64)],
    "xy_set_sweep": [_vp, C.c_uint64],
    "xy_debug_fix_phi": [_vp, C.c_int, C.c_double],
    "xy_get_fallback_count": [_vp, C.POINTER(C.c_uint64)],
    "xy_debug_kernel_timing": [_vp, C.c_int],
    "xy_get_kernel_times": [_vp, C.POINTER(C.c_double), C.POINTER(C.c_uint64)],
    "xy_get_launch_count": [_vp, C.POINTER(C.c_uint64)],
    "xy_label_bonds": [_vp, _vp, C.c_size_t],
    "xy_debug_check_counts": [C.POINTER(C.c_uint64), C.POINTER(C.c_int)],
    "xy_slab_workspace_bytes": [C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(C.c_size_t)],
    "xy_slab_create": [C.POINTER(_vp), C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, C.c_int, C.c_uint32, _vp, C.c_size_t],
    "xy_slab_buffers": [_vp, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(C.c_size_t), C.POINTER(_vp), C.POINTER(C.c_size_t)],
    "xy_slab_label": [_vp, C.c_double, _vp],
    "xy_slab_label_bonds": [_vp, _vp, C.c_size_t],
    "xy_slab_flip": [_vp, _vp, C.c_uint32, C.c_uint32, _vp],
    "xy_slab_pcc_setup": [_vp, C.c_double, C.c_double, C.POINTER(PccSchedule)],
    "xy_slab_label_pcc": [_vp, _vp],
    "xy_slab_pcc_buffers": [_vp, C.POINTER(_vp), C.POINTER(_vp)],
    "xy_slab_obs_partial": [_vp, _vp],
    "xy_slab_pcc_feed": [_vp, _vp],
    "xy_potts_create": [C.POINTER(_vp), C.c_uint32, C.c_uint32, C.c_uint64, C.c_int],
    "xy_potts_destroy": [_vp],
    "xy_potts_sweeps": [_vp, C.c_double, C.c_uint64, _vp],
    "xy_potts_measure": [_vp, _vp],
    "xy_potts_get_spins": [_vp, _vp, C.c_size_t],
    "xy_potts_set_spins": [_vp, _vp, C.c_size_t],
    "xy_potts_get_sweep": [_vp, C.POINTER(C.c_uint64)],
    "xy_potts_set_sweep": [_vp, C.c_uint64],
    "xy_potts_get_bonds": [_vp, _vp, C.c_size_t],
    "xy_potts_get_labels": [_vp, _vp, C.c_size_t],
    "xy_potts_get_launch_count": [_vp, C.POINTER(C.c_uint64)],
    "xy_observe_static": [_vp, C.c_uint32, _vp, _vp],
    "xy_xi2nd": [C.c_double, C.c_double, C.c_uint32, C.POINTER(C.c_double)],
    "xy_debug_philox": [_vp, _vp, _vp, C.c_size_t],
    "xy_debug_curand_philox": [_vp, _vp, _vp, C.c_size_t],
}
for _name, _args in _SIGS.items():
    _f = getattr(_lib, _name)
    _f.argtypes = _args
    _f.restype = C.c_int
_lib.xy_last_error.restype = C.c_char_p
_lib.xy_last_error.argtypes = []

EXPORTED = tuple(_SIGS) + ("xy_last_error",)


def _check(rc):
    if rc != 0:
        raise XYError(rc, _lib.xy_last_error().decode())


def workspace_bytes(L, flags=0):
    n = C.c_size_t()
    _check(_lib.xy_workspace_bytes(L, flags, C.byref(n)))
    return n.value


def _host_ptr(arr):
    """pointer of a contiguous numpy array or CPU torch tensor (pinned or pageable)."""
    if isinstance(arr, np.ndarray):
        assert arr.flags["C_CONTIGUOUS"]
        return arr.ctypes.data
    assert arr.device.type == "cpu" and arr.is_contiguous()
    return arr.data_ptr()


class XYState:
    """One lattice on the current CUDA device.  Methods mirror the C calls one to one."""

    def __init__(self, L, seed, init=INIT_HOT, flags=0, torch_workspace=True):
        import torch
        if not torch.cuda.is_available():
            raise XYError(-4, "no CUDA device: this library has no CPU fallback")
        self.L, self.N, self.seed, self.flags = L, L * L, seed, flags
        self._h = _vp()
        self._ws = None
        if torch_workspace:
            nbytes = workspace_bytes(L, flags)
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            _check(_lib.xy_create_ex(C.byref(self._h), L, seed, init, flags, self._ws.data_ptr(), nbytes))
        else:
            _check(_lib.xy_create_ex(C.byref(self._h), L, seed, init, flags, None, 0))

    # -- the five calls ---------------------------------------------------------------------
    def sw_sweeps(self, beta, n=1, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        _check(_lib.xy_sw_sweeps(self._h, beta, n, st))

    def measure(self):
        o = Obs()
        _check(_lib.xy_measure(self._h, C.byref(o)))
        return o

    def pcc_get_state(self):
        st = PccState()
        _check(_lib.xy_pcc_get_state(self._h, C.byref(st)))
        return st

    def pcc_set_state(self, st: PccState):
        _check(_lib.xy_pcc_set_state(self._h, C.byref(st)))

    def pcc_continue(self, sched: PccSchedule, trace=True):
        return self.pcc_run(None, sched, trace)

    def pcc_run(self, beta0, sched: PccSchedule, trace=True):
        """beta0 None: xy_pcc_continue (the controller goes on from its state)"""
        out = _PccOut()
        cap = int((sched.n_sweeps - sched.discard) // max(sched.window, 1)) + 1 if trace else 0
        tb = np.zeros(max(cap, 1))
        ty = np.zeros(max(cap, 1))
        out.trace_beta = tb.ctypes.data_as(C.POINTER(C.c_double))
        out.trace_bY = ty.ctypes.data_as(C.POINTER(C.c_double))
        out.trace_cap = cap
        if beta0 is None:
            _check(_lib.xy_pcc_continue(self._h, C.byref(sched), C.byref(out)))
        else:
            _check(_lib.xy_pcc_run(self._h, beta0, sched.dbeta0, C.byref(sched), C.byref(out)))
        n = min(int(out.trace_len), cap)
        return {"beta_final": out.beta_final, "dbeta_final": out.dbeta_final, "beta_mean": out.beta_mean,
                "n_decisions": int(out.n_decisions), "trace_len": int(out.trace_len),
                "trace_beta": tb[:n].copy(), "trace_bY": ty[:n].copy()}

    def destroy(self):
        if self._h:
            _check(_lib.xy_destroy(self._h))
            self._h = _vp()
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- extensions -------------------------------------------------------------------------
    def get_angles(self, out=None, n=None, first=0):
        """n sites from `first` (default: all)"""
        n = self.N - first if n is None else int(n)
        out = np.empty(n, np.float32) if out is None else out
        _check(_lib.xy_get_angles_range(self._h, _host_ptr(out), first, n))
        return out

    def set_angles(self, theta):
        if isinstance(theta, np.ndarray):
            theta = np.ascontiguousarray(theta, np.float32)
        _check(_lib.xy_set_angles(self._h, _host_ptr(theta), self.N))

    def get_labels(self, n=None, first=0):
        n = self.N - first if n is None else int(n)
        out = np.empty(n, np.int64)
        _check(_lib.xy_get_labels_range(self._h, out.ctypes.data, first, n))
        return out

    def get_bonds(self, n=None, first=0):
        n = self.N - first if n is None else int(n)
        out = np.empty(n, np.uint8)
        _check(_lib.xy_get_bonds_range(self._h, out.ctypes.data, first, n))
        return out

    def debug_check_labels(self):
        """device-side invariants of the last sweep's labels: dict of the five counts"""
        c = (C.c_uint64 * 5)()
        _check(_lib.xy_debug_check_labels(self._h, c))
        return {"label_above_index": int(c[0]), "root_not_fixed": int(c[1]), "x_bond_split": int(c[2]),
                "y_bond_split": int(c[3]), "n_roots": int(c[4])}

    def set_obs_mode(self, mode):
        _check(_lib.xy_set_obs_mode(self._h, mode))

    def measure_fourier(self):
        """The 8 structure-factor sums of the current configuration (needs FLAG_FOURIER): array [8] = Fx, Fy."""
        f = Fourier()
        _check(_lib.xy_measure_fourier(self._h, C.byref(f)))
        return np.array(list(f.Fx) + list(f.Fy), dtype=np.float64)

    def get_fourier_series(self, first, count):
        out = np.zeros(count, FOURIER_DTYPE)
        _check(_lib.xy_get_fourier_series(self._h, out.ctypes.data, first, count))
        return out

    def get_series(self, first, count):
        out = np.zeros(count, OBS_DTYPE)
        _check(_lib.xy_get_series(self._h, out.ctypes.data, first, count))
        return out

    def series_capacity(self):
        c = C.c_uint64()
        _check(_lib.xy_series_capacity(self._h, C.byref(c)))
        return c.value

    def get_sweep(self):
        t = C.c_uint64()
        _check(_lib.xy_get_sweep(self._h, C.byref(t)))
        return t.value

    def set_sweep(self, t):
        _check(_lib.xy_set_sweep(self._h, t))

    def debug_fix_phi(self, on, phi=0.0):
        _check(_lib.xy_debug_fix_phi(self._h, 1 if on else 0, phi))

    def get_fallback_count(self):
        c = C.c_uint64()
        _check(_lib.xy_get_fallback_count(self._h, C.byref(c)))
        return c.value

    def debug_kernel_timing(self, on):
        _check(_lib.xy_debug_kernel_timing(self._h, 1 if on else 0))

    def get_kernel_times(self):
        ms = (C.c_double * 4)()
        n = (C.c_uint64 * 4)()
        _check(_lib.xy_get_kernel_times(self._h, ms, n))
        names = ("k_bonds", "k_label", "k_merge", "k_flip")
        return {k: {"ms": ms[i], "launches": int(n[i])} for i, k in enumerate(names)}

    def get_launch_count(self):
        c = C.c_uint64()
        _check(_lib.xy_get_launch_count(self._h, C.byref(c)))
        return c.value

    def label_bonds(self, bonds):
        b = np.ascontiguousarray(bonds, np.uint8)
        _check(_lib.xy_label_bonds(self._h, b.ctypes.data, self.N))


def xi2nd(chi0, chik, L):
    """xy_xi2nd: PAPER.md Eq. 8 from the averaged chi(0) and chi(2 pi / L)"""
    out = C.c_double()
    _check(_lib.xy_xi2nd(chi0, chik, L, C.byref(out)))
    return out.value


def observe_static(theta, L, out=None, stream=None):
    """xy_observe_static: the seven observable sums of the L x L angles in the CUDA tensor `theta` (float32, contiguous),
    for callers whose device memory is all spoken for (a pool or caching allocator owns it, or a cudaMalloc would stall
    busy streams): the kernel's scratch is a fixed array inside the library, so nothing is allocated on the device --
    `out` included if the caller passes it (a CUDA uint8 tensor of sizeof(xy_obs) = 96 bytes; None: this wrapper makes
    one with torch).  Only enqueues; returns `out`, readable as OBS_DTYPE after a synchronise.  Calls on one GPU share
    the scratch and must not overlap; the first call per device does a blocking set-up (see include/xy.h)."""
    import torch
    assert theta.is_cuda and theta.dtype == torch.float32 and theta.is_contiguous() and theta.numel() == L * L
    if out is None:
        out = torch.empty(C.sizeof(Obs), dtype=torch.uint8, device=theta.device)
    assert out.is_cuda and out.is_contiguous() and out.numel() * out.element_size() >= C.sizeof(Obs)
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _check(_lib.xy_observe_static(theta.data_ptr(), L, out.data_ptr(), st))
    return out


def _philox_common(fn, ctr, key):
    ctr = np.ascontiguousarray(ctr, np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    _check(fn(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, ctr.shape[0]))
    return out


def debug_check_counts():
    """(counts[8], checked_build) of the -DXY_CHECKED range checks; all zero from the normal build"""
    c = (C.c_uint64 * 8)()
    flag = C.c_int()
    _check(_lib.xy_debug_check_counts(c, C.byref(flag)))
    return [int(v) for v in c], bool(flag.value)


def debug_philox(ctr, key):
    return _philox_common(_lib.xy_debug_philox, ctr, key)


def debug_curand_philox(ctr, key):
    return _philox_common(_lib.xy_debug_curand_philox, ctr, key)


# ---------------------------------------------------------------------------------------------
# Row slab of a sharded lattice (include/xy.h, section "row-slab sharding"); the exchange between xy_slab_label and
# xy_slab_flip is the caller's: paper_1210_6116_b200/shard.py does it with torch.distributed
# ---------------------------------------------------------------------------------------------
class SlabState(XYState):
    """rows [y_off, y_off + rows) of an L x L lattice on the current CUDA device (marshalling only)."""

    def __init__(self, L, rows, y_off, seed, init=INIT_HOT, flags=0):
        import torch
        if not torch.cuda.is_available():
            raise XYError(-4, "no CUDA device: this library has no CPU fallback")
        self.L, self.rows, self.y_off, self.N, self.seed, self.flags = L, rows, y_off, rows * L, seed, flags
        self._h = _vp()
        n = C.c_size_t()
        _check(_lib.xy_slab_workspace_bytes(L, rows, flags, C.byref(n)))
        self._ws = torch.empty(n.value, dtype=torch.uint8, device="cuda")
        _check(_lib.xy_slab_create(C.byref(self._h), L, rows, y_off, seed, init, flags, self._ws.data_ptr(), n.value))
        first, halo, edges = _vp(), _vp(), _vp()
        rb, eb = C.c_size_t(), C.c_size_t()
        _check(_lib.xy_slab_buffers(self._h, C.byref(first), C.byref(halo), C.byref(rb), C.byref(edges), C.byref(eb)))
        base = self._ws.data_ptr()
        # views into the workspace tensor (the exchange reads / writes them in place)
        self.first_row = self._ws[first.value - base: first.value - base + rb.value].view(torch.float32)
        self.halo_row = self._ws[halo.value - base: halo.value - base + rb.value].view(torch.float32)
        self.edges = self._ws[edges.value - base: edges.value - base + eb.value]
        part, glob = _vp(), _vp()
        _check(_lib.xy_slab_pcc_buffers(self._h, C.byref(part), C.byref(glob)))
        self.pcc_partial = self._ws[part.value - base: part.value - base + 64].view(torch.float64)
        self.pcc_global = self._ws[glob.value - base: glob.value - base + 64].view(torch.float64)

    def slab_label(self, beta, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        _check(_lib.xy_slab_label(self._h, beta, st))

    def _stream(self, stream):
        import torch
        return torch.cuda.current_stream().cuda_stream if stream is None else stream

    def slab_label_bonds(self, bonds):
        b = np.ascontiguousarray(bonds, np.uint8)
        _check(_lib.xy_slab_label_bonds(self._h, b.ctypes.data, b.size))

    def slab_pcc_setup(self, beta0, sched: PccSchedule):
        _check(_lib.xy_slab_pcc_setup(self._h, beta0, sched.dbeta0, C.byref(sched)))

    def slab_label_pcc(self, stream=None):
        _check(_lib.xy_slab_label_pcc(self._h, self._stream(stream)))

    def slab_obs_partial(self, stream=None):
        _check(_lib.xy_slab_obs_partial(self._h, self._stream(stream)))

    def slab_pcc_feed(self, stream=None):
        _check(_lib.xy_slab_pcc_feed(self._h, self._stream(stream)))

    def slab_flip(self, gathered, nranks, rank, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        assert gathered.is_cuda and gathered.is_contiguous() and gathered.numel() * gathered.element_size() == nranks * self.edges.numel()
        _check(_lib.xy_slab_flip(self._h, gathered.data_ptr(), nranks, rank, st))


# ---------------------------------------------------------------------------------------------
# q-state Potts model on the same labeling core (include/xy.h, section "Potts")
# ---------------------------------------------------------------------------------------------
class PottsObs(C.Structure):
    _fields_ = [("sweep", C.c_uint64), ("beta", C.c_double), ("E", C.c_int64),
                ("ex", C.c_uint64), ("ey", C.c_uint64), ("count", C.c_uint64 * 16),
                ("n_bonds_x", C.c_uint64), ("n_bonds_y", C.c_uint64), ("n_clusters", C.c_uint64)]


class PottsState:
    """Owner of one xy_potts (marshalling only)."""

    def __init__(self, L, q, seed, init=INIT_HOT):
        self._h = _vp()
        self.L, self.q, self.N = L, q, L * L
        _check(_lib.xy_potts_create(C.byref(self._h), L, q, seed, init))

    def destroy(self):
        if self._h:
            _check(_lib.xy_potts_destroy(self._h))
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def sweeps(self, beta, n=1, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        _check(_lib.xy_potts_sweeps(self._h, beta, n, st))

    def measure(self):
        o = PottsObs()
        _check(_lib.xy_potts_measure(self._h, C.byref(o)))
        return o

    def get_spins(self, n=None):
        out = np.empty(self.N if n is None else n, np.uint8)
        _check(_lib.xy_potts_get_spins(self._h, out.ctypes.data, out.size))
        return out

    def set_spins(self, spins):
        a = np.ascontiguousarray(spins, np.uint8)
        _check(_lib.xy_potts_set_spins(self._h, a.ctypes.data, a.size))

    def get_sweep(self):
        t = C.c_uint64()
        _check(_lib.xy_potts_get_sweep(self._h, C.byref(t)))
        return t.value

    def set_sweep(self, t):
        _check(_lib.xy_potts_set_sweep(self._h, t))

    def get_bonds(self, n=None):
        out = np.empty(self.N if n is None else n, np.uint8)
        _check(_lib.xy_potts_get_bonds(self._h, out.ctypes.data, out.size))
        return out

    def get_labels(self, n=None):
        out = np.empty(self.N if n is None else n, np.int64)
        _check(_lib.xy_potts_get_labels(self._h, out.ctypes.data, out.size))
        return out

    def get_launch_count(self):
        c = C.c_uint64()
        _check(_lib.xy_potts_get_launch_count(self._h, C.byref(c)))
        return c.value
