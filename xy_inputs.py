"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no Philox, no bond rule, no
labeling, no reflection): only workload descriptions and numpy-seeded input
fields.  The hot / cold starts of the method itself are produced independently
by each side (oracle: xyo_init; CUDA: xy_create), from the same counter-based
generator definition.

The paper (arXiv 1210.6116) uses no dataset: its workloads are the lattices
themselves (sizes PAPER.md:64, Table I :80-92).  BASELINE.json's five configs
are fully synthetic and are reproduced literally here.
"""
import math

import numpy as np

TWO_PI = 2.0 * math.pi

# BASELINE.json "configs", in order (index 0 = the small case the oracle finishes in seconds).
CONFIGS = [
    dict(name="L64_hot_b1.12", L=64, init="hot", seed=1, beta=1.12, sweeps=1000),
    dict(name="L1024_cold_4beta", L=1024, init="cold", seed=7, betas=(0.90, 1.00, 1.12, 1.30),
         therm=2000, sweeps=10000),
    dict(name="L4096_hot_pcc", L=4096, init="hot", seed=11, beta0=1.05, dbeta0=1e-3,
         halve_every=2000, dbeta_min=1e-6, target=2.0 / math.pi, window=20, dirs=1,
         discard=0, sweeps=20000),
    dict(name="L16384_cold_b1.11996", L=16384, init="cold", seed=13, beta=1.11996,
         therm=500, sweeps=2000),
    dict(name="L65536_hot_b1.11996", L=65536, init="hot", seed=17, beta=1.11996, sweeps=200),
]

INIT_CODE = {"cold": 0, "hot": 1}


def random_angles(L, seed):
    """fp32 angles uniform on the 24-bit grid of [0, 2pi): a generic disordered state."""
    rng = np.random.default_rng(seed)
    k = rng.integers(0, 1 << 24, size=L * L, dtype=np.int64)
    return (k.astype(np.float64) * (TWO_PI / (1 << 24))).astype(np.float32)


def clock_angles(L, q, seed):
    """angles restricted to the q-gon {2 pi k / q}; q = 2 is the Ising limit {0, pi}."""
    rng = np.random.default_rng(seed)
    k = rng.integers(0, q, size=L * L, dtype=np.int64)
    return (k.astype(np.float64) * (TWO_PI / q)).astype(np.float32)


def smooth_angles(L, seed, amplitude=0.6, modes=3):
    """Low-temperature-like field: a few long-wavelength plane waves plus weak noise,
    wrapped into [0, 2pi).  Gives large clusters spanning many tiles."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:L, 0:L].astype(np.float64)
    th = np.full((L, L), rng.uniform(0, TWO_PI))
    for _ in range(modes):
        kx, ky = rng.integers(-2, 3, size=2)
        th += amplitude * np.cos(TWO_PI * (kx * x + ky * y) / L + rng.uniform(0, TWO_PI))
    th += 0.15 * rng.standard_normal((L, L))
    return np.mod(th, TWO_PI).astype(np.float32).ravel()


def vortex_pair_angles(L, seed):
    """A vortex / antivortex pair on the torus plus noise: angles sweep the full circle,
    so sigma changes sign along lines and clusters have ragged, long boundaries."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:L, 0:L].astype(np.float64)
    x1, y1 = L * 0.25 + 0.5, L * 0.5 + 0.5
    x2, y2 = L * 0.75 + 0.5, L * 0.5 + 0.5
    th = np.arctan2(y - y1, x - x1) - np.arctan2(y - y2, x - x2)
    th += 0.1 * rng.standard_normal((L, L))
    return np.mod(th, TWO_PI).astype(np.float32).ravel()


def random_bonds(L, density, seed):
    """byte per site: bit0 = x bond (x,y)-(x+1,y), bit1 = y bond (x,y)-(x,y+1); iid."""
    rng = np.random.default_rng(seed)
    bx = rng.random(L * L) < density
    by = rng.random(L * L) < density
    return (bx.astype(np.uint8) | (by.astype(np.uint8) << 1))


def pattern_bonds(L, kind):
    """Adversarial bond sets for the labeling step."""
    b = np.zeros((L, L), np.uint8)
    if kind == "all_on":
        b[:] = 3
    elif kind == "all_off":
        pass
    elif kind == "wrap_only":          # only the periodic wrap bonds
        b[:, L - 1] |= 1
        b[L - 1, :] |= 2
    elif kind == "h_stripes":          # every row one ring, rows disconnected
        b[:] = 1
    elif kind == "v_stripes":
        b[:] = 2
    elif kind == "serpentine":         # one snake through all sites: longest chains
        b[:, : L - 1] |= 1             # rows connected inside, no wrap
        for y in range(L - 1):
            x = L - 1 if y % 2 == 0 else 0
            b[y, x] |= 2
    elif kind == "comb":               # vertical teeth joined by the top row
        b[: L - 1, :] |= 2
        b[0, : L - 1] |= 1
    elif kind == "checker_islands":    # 2x2 islands
        b[0::2, 0::2] = 3
        b[0::2, 1::2] = 2
        b[1::2, 0::2] = 1
    else:
        raise ValueError(kind)
    return b.ravel()


BOND_PATTERNS = ("all_on", "all_off", "wrap_only", "h_stripes", "v_stripes", "serpentine",
                 "comb", "checker_islands")
