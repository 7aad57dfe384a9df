"""ctypes wrapper over oracle/libxy_oracle.so (argument marshalling only).

TEST INFRASTRUCTURE: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs only.  All arithmetic lives in
oracle/xy_oracle.c; this file converts numpy arrays to pointers.
"""
import ctypes as C
import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

u8p = np.ctypeslib.ndpointer(np.uint8, flags="C_CONTIGUOUS")
f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")


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


class PccSchedule(C.Structure):
    _fields_ = [("n_sweeps", C.c_uint64), ("discard", C.c_uint64),
                ("window", C.c_uint32), ("dirs", C.c_uint32),
                ("dbeta0", C.c_double), ("halve_every", C.c_uint64),
                ("dbeta_min", C.c_double), ("target", C.c_double)]


class PccCtrl(C.Structure):
    _fields_ = [("beta", C.c_double), ("dbeta", C.c_double),
                ("acc_e", C.c_double), ("acc_s2", C.c_double),
                ("k", C.c_uint64), ("n_decisions", C.c_uint64),
                ("stage_sum", C.c_double), ("last_sum", C.c_double),
                ("stage_cnt", C.c_uint64), ("last_cnt", C.c_uint64),
                ("last_bY", C.c_double)]


class PccOut(C.Structure):
    _fields_ = [("beta_final", C.c_double), ("dbeta_final", C.c_double), ("beta_mean", C.c_double),
                ("n_decisions", C.c_uint64),
                ("trace_beta", C.POINTER(C.c_double)), ("trace_bY", C.POINTER(C.c_double)),
                ("trace_cap", C.c_uint64), ("trace_len", C.c_uint64)]


def _sig(name, res, args):
    f = getattr(_lib, name)
    f.restype = res
    f.argtypes = args
    return f


_philox = _sig("xyo_philox4x32_10", None, [u32p, u32p, u32p])
_rng = _sig("xyo_rng", None, [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, u32p])
_uniform = _sig("xyo_uniform", C.c_double, [C.c_uint32])
_init = _sig("xyo_init", C.c_int, [f32p, C.c_uint32, C.c_uint64, C.c_int])
_phi = _sig("xyo_phi", C.c_double, [C.c_uint64, C.c_uint64])
_sigma = _sig("xyo_sigma", C.c_double, [C.c_float, C.c_double])
_bond_prob = _sig("xyo_bond_prob", C.c_double, [C.c_double, C.c_double, C.c_double])
_bond_u_site = _sig("xyo_bond_uniforms_site", None,
                    [C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_double), C.POINTER(C.c_double)])
_bonds_from_u = _sig("xyo_bonds_from_u", None,
                     [f32p, C.c_uint32, C.c_double, C.c_double, f64p, f64p, u8p, C.c_void_p, C.c_void_p])
_bonds = _sig("xyo_bonds", None,
              [f32p, C.c_uint32, C.c_double, C.c_double, C.c_uint64, C.c_uint64, u8p, C.c_void_p, C.c_void_p])
_bond_margin = _sig("xyo_bond_margin", C.c_double,
                    [f32p, C.c_uint32, C.c_double, C.c_double, C.c_uint64, C.c_uint64, C.c_uint64, C.c_int])
_label = _sig("xyo_label", C.c_uint64, [u8p, C.c_uint32, i64p])
_flip_coin = _sig("xyo_flip_coin", C.c_int, [C.c_uint64, C.c_uint64, C.c_uint64])
_reflect_const = _sig("xyo_reflect_const", C.c_double, [C.c_double])
_reflect = _sig("xyo_reflect", C.c_float, [C.c_float, C.c_double])
_flip_sites = _sig("xyo_flip_sites", None, [f32p, C.c_uint64, C.c_double, u8p])
_flip = _sig("xyo_flip", C.c_uint64, [f32p, C.c_uint32, i64p, C.c_double, C.c_uint64, C.c_uint64])
_observe = _sig("xyo_observe", None, [f32p, C.c_uint32, C.POINTER(Obs)])
_fourier = _sig("xyo_fourier", None, [f32p, C.c_uint32, C.POINTER(C.c_double)])
_sk = _sig("xyo_sk", C.c_double, [C.POINTER(C.c_double), C.c_uint32])
_xi2nd = _sig("xyo_xi2nd", C.c_double, [C.c_double, C.c_double, C.c_uint32])
_sweep = _sig("xyo_sweep", C.c_int,
              [f32p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double, C.c_int, C.c_double,
               u8p, i64p, C.POINTER(Obs)])
_pcc_init = _sig("xyo_pcc_init", None, [C.POINTER(PccCtrl), C.c_double, C.c_double])
_pcc_feed = _sig("xyo_pcc_feed", C.c_int,
                 [C.POINTER(PccCtrl), C.POINTER(PccSchedule), C.c_double,
                  C.c_double, C.c_double, C.c_double, C.c_double,
                  C.POINTER(C.c_double), C.POINTER(C.c_double)])
_pcc_beta_mean = _sig("xyo_pcc_beta_mean", C.c_double, [C.POINTER(PccCtrl)])
_pcc_run = _sig("xyo_pcc_run", C.c_int,
                [f32p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double, C.c_double,
                 C.POINTER(PccSchedule), C.POINTER(PccOut)])
_run = _sig("xyo_run", C.c_int,
            [f32p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double, C.c_uint64,
             C.c_int, C.c_double, C.c_void_p])

TAG_INIT, TAG_DIR, TAG_BOND, TAG_FLIP, TAG_BOND_LO = 0, 1, 2, 3, 4
INIT_COLD, INIT_HOT = 0, 1


def philox4x32_10(ctr, key):
    out = np.zeros(4, np.uint32)
    _philox(np.ascontiguousarray(ctr, np.uint32), np.ascontiguousarray(key, np.uint32), out)
    return out


def rng(seed, idx, t, tag):
    out = np.zeros(4, np.uint32)
    _rng(seed, idx, t, tag, out)
    return out


def uniform(w):
    return _uniform(int(w))


def init(L, seed, kind):
    theta = np.empty(L * L, np.float32)
    if _init(theta, L, seed, kind) != 0:
        raise ValueError("bad init kind")
    return theta


def phi(seed, t):
    return _phi(seed, t)


def sigma(theta, ph):
    return _sigma(float(theta), ph)


def bond_prob(beta, si, sj):
    return _bond_prob(beta, si, sj)


def bond_uniforms_site(seed, t, i):
    ux, uy = C.c_double(), C.c_double()
    _bond_u_site(seed, t, i, C.byref(ux), C.byref(uy))
    return ux.value, uy.value


def bonds_from_u(theta, L, beta, ph, ux, uy, margins=False):
    N = L * L
    b = np.empty(N, np.uint8)
    if margins:
        mx, my = np.empty(N), np.empty(N)
        _bonds_from_u(theta, L, beta, ph, ux, uy, b, mx.ctypes.data, my.ctypes.data)
        return b, mx, my
    _bonds_from_u(theta, L, beta, ph, ux, uy, b, None, None)
    return b


def bonds(theta, L, beta, ph, seed, t, margins=False):
    N = L * L
    b = np.empty(N, np.uint8)
    if margins:
        mx, my = np.empty(N), np.empty(N)
        _bonds(theta, L, beta, ph, seed, t, b, mx.ctypes.data, my.ctypes.data)
        return b, mx, my
    _bonds(theta, L, beta, ph, seed, t, b, None, None)
    return b


def bond_margin(theta, L, beta, ph, seed, t, i, direction):
    return _bond_margin(theta, L, beta, ph, seed, t, i, direction)


def label(bonds_arr, L):
    lab = np.empty(L * L, np.int64)
    n = _label(np.ascontiguousarray(bonds_arr, np.uint8), L, lab)
    if n == 2 ** 64 - 1:
        raise MemoryError
    return lab, int(n)


def flip_coin(seed, rho, t):
    return _flip_coin(seed, int(rho), t)


def reflect_const(ph):
    return _reflect_const(ph)


def reflect(theta, A):
    return _reflect(float(theta), A)


def flip_sites(theta, ph, flip_site):
    _flip_sites(theta, theta.size, ph, np.ascontiguousarray(flip_site, np.uint8))
    return theta


def flip(theta, L, lab, ph, seed, t):
    return int(_flip(theta, L, lab, ph, seed, t))


def observe(theta, L):
    o = Obs()
    _observe(theta, L, C.byref(o))
    return o


def fourier(theta, L):
    """The 8 structure-factor sums at k = 2 pi / L (x: F[0:4], y: F[4:8]) of one configuration."""
    F = (C.c_double * 8)()
    _fourier(theta, L, F)
    return np.array(F[:], dtype=np.float64)


def sk(F4, L):
    """|sum_r s(r) e^{ikr}|^2 / N from the four sums of one direction."""
    a = (C.c_double * 4)(*[float(v) for v in F4])
    return _sk(a, L)


def xi2nd(chi0, chik, L):
    """PAPER.md:102 Eq. 8."""
    return _xi2nd(chi0, chik, L)


def sweep(theta, L, seed, t, beta, fix_phi=None):
    """One whole sweep in place on theta; returns (bonds, labels, Obs)."""
    N = L * L
    b = np.empty(N, np.uint8)
    lab = np.empty(N, np.int64)
    o = Obs()
    rc = _sweep(theta, L, seed, t, beta, 0 if fix_phi is None else 1,
                0.0 if fix_phi is None else fix_phi, b, lab, C.byref(o))
    if rc != 0:
        raise MemoryError
    return b, lab, o


def run(theta, L, seed, t0, beta, n, fix_phi=None, series=True):
    """n sweeps in place; returns the per-sweep series as a structured array."""
    ser = np.zeros(n, OBS_DTYPE) if series else None
    rc = _run(theta, L, seed, t0, beta, n, 0 if fix_phi is None else 1,
              0.0 if fix_phi is None else fix_phi, ser.ctypes.data if series else None)
    if rc != 0:
        raise MemoryError
    return ser


class PccController:
    """The pure controller state machine (xyo_pcc_init / xyo_pcc_feed)."""

    def __init__(self, beta0, sched: PccSchedule):
        self.c = PccCtrl()
        self.s = sched
        _pcc_init(C.byref(self.c), beta0, sched.dbeta0)

    def feed(self, N, Cx, Sx, Cy=0.0, Sy=0.0):
        b, y = C.c_double(), C.c_double()
        d = _pcc_feed(C.byref(self.c), C.byref(self.s), float(N), Cx, Sx, Cy, Sy, C.byref(b), C.byref(y))
        return (b.value, y.value) if d else None

    @property
    def beta(self):
        return self.c.beta

    @property
    def dbeta(self):
        return self.c.dbeta

    def beta_mean(self):
        return _pcc_beta_mean(C.byref(self.c))


def pcc_run(theta, L, seed, t0, beta0, sched: PccSchedule, trace_cap=0):
    out = PccOut()
    tb = np.zeros(max(trace_cap, 1))
    ty = np.zeros(max(trace_cap, 1))
    out.trace_beta = tb.ctypes.data_as(C.POINTER(C.c_double))
    out.trace_bY = ty.ctypes.data_as(C.POINTER(C.c_double))
    out.trace_cap = trace_cap
    rc = _pcc_run(theta, L, seed, t0, beta0, sched.dbeta0, C.byref(sched), C.byref(out))
    if rc != 0:
        raise MemoryError
    n = min(int(out.trace_len), trace_cap)
    return {"beta_final": out.beta_final, "dbeta_final": out.dbeta_final,
            "beta_mean": out.beta_mean, "n_decisions": int(out.n_decisions),
            "trace_len": int(out.trace_len), "trace_beta": tb[:n].copy(), "trace_bY": ty[:n].copy()}


# ---------------------------------------------------------------------------------------------
# q-state Potts model on the same labeling core (readings P1-P5 in xy_oracle.c)
# ---------------------------------------------------------------------------------------------
class PottsObs(C.Structure):
    _fields_ = [("sweep", C.c_uint64), ("beta", C.c_double), ("E", C.c_int64),
                ("ex", C.c_uint64), ("ey", C.c_uint64), ("count", C.c_uint64 * 16),
                ("n_bonds_x", C.c_uint64), ("n_bonds_y", C.c_uint64), ("n_clusters", C.c_uint64)]


TAG_POTTS = 5
_potts_init = _sig("xyo_potts_init", C.c_int, [u8p, C.c_uint32, C.c_uint32, C.c_uint64, C.c_int])
_potts_bond_prob = _sig("xyo_potts_bond_prob", C.c_double, [C.c_double])
_potts_bonds = _sig("xyo_potts_bonds", None,
                    [u8p, C.c_uint32, C.c_double, C.c_uint64, C.c_uint64, u8p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)])
_potts_new_spin = _sig("xyo_potts_new_spin", C.c_uint32, [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32])
_potts_assign = _sig("xyo_potts_assign", None, [u8p, C.c_uint32, C.c_uint32, i64p, C.c_uint64, C.c_uint64])
_potts_observe = _sig("xyo_potts_observe", None, [u8p, C.c_uint32, C.POINTER(PottsObs)])
_potts_sweep = _sig("xyo_potts_sweep", C.c_int,
                    [u8p, C.c_uint32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double, u8p, i64p, C.POINTER(PottsObs)])


def potts_init(L, q, seed, kind):
    spin = np.empty(L * L, np.uint8)
    if _potts_init(spin, L, q, seed, kind) != 0:
        raise ValueError("bad q or init kind")
    return spin


def potts_bond_prob(beta):
    return _potts_bond_prob(beta)


def potts_bonds(spin, L, beta, seed, t):
    bonds = np.empty(L * L, np.uint8)
    nx, ny = C.c_uint64(), C.c_uint64()
    _potts_bonds(spin, L, beta, seed, t, bonds, C.byref(nx), C.byref(ny))
    return bonds, nx.value, ny.value


def potts_new_spin(seed, rho, t, q):
    return _potts_new_spin(seed, int(rho), t, q)


def potts_assign(spin, L, q, lab, seed, t):
    _potts_assign(spin, L, q, np.ascontiguousarray(lab, np.int64), seed, t)


def potts_observe(spin, L):
    o = PottsObs()
    _potts_observe(spin, L, C.byref(o))
    return o


def potts_sweep(spin, L, q, seed, t, beta):
    """one sweep in place; returns (bonds, labels, obs)"""
    bonds = np.empty(L * L, np.uint8)
    lab = np.empty(L * L, np.int64)
    o = PottsObs()
    if _potts_sweep(spin, L, q, seed, t, beta, bonds, lab, C.byref(o)) != 0:
        raise ValueError("potts sweep failed")
    return bonds, lab, o
