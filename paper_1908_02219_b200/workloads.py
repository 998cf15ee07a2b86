"""Seeded synthetic marker loads (the five BASELINE.json configs).

This module is the ONLY thing the CUDA path and the CPU oracle have in common:
it produces the input arrays (numpy, host) that are then handed, as data, to
both.  It holds none of the method's arithmetic (no ring, no spline, no
deposition) and imports neither side.  The recipe is stated in DESIGN.md
"Input recipe"; it stands in for the ORB5 production decks of PAPER.md:105, 117
(deuterium markers, ~4-8 markers per cell, Maxwellian ring-size spread, fixed
and adaptive N_L), which are not available.

Counter-based: value = f(splitmix64(seed, stream, marker index)), so any chunk
can be generated independently and in parallel, bit-identically.
"""
from __future__ import annotations

import dataclasses
import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

TWO_PI = 2.0 * math.pi

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)

# stream ids
S_S, S_TH, S_PH, S_VP1, S_VP2, S_VT, S_W1, S_W2 = range(8)


@dataclasses.dataclass(frozen=True)
class Config:
    """One synthetic workload (grid in CELLS, marker count, N_L policy)."""
    name: str
    ns: int
    ntheta: int
    nphi: int
    n_markers: int
    rho_star: float
    current: bool                 # deposit j_par as well as rho
    adaptive: bool = False
    n_fixed: int = 4              # fixed N_L, or n_min when adaptive
    n_max: int = 4
    order: str = "random"         # "random" | "sorted" (pre-sorted by cell, R17)
    seed: int = 0
    r0: float = 1.0
    a: float = 0.3
    b0: float = 1.0
    q: float = 1.0
    s_lo: float = 0.1
    s_hi: float = 0.9
    w_sigma: float = 1e-3

    @property
    def rho_ref(self) -> float:
        return self.rho_star      # thermal Larmor radius in units of a (R9)

    @property
    def nodes(self) -> int:
        return (self.ns + 3) * self.ntheta * self.nphi

    @property
    def algorithmic_bytes(self) -> int:
        """each marker field once, each grid node read+written once."""
        return self.n_markers * 8 * (6 if self.current else 5) + \
            (2 if self.current else 1) * self.nodes * 16


CONFIGS = {
    "cfg0": Config("cfg0", 16, 32, 16, 65_536, 1 / 180, current=False),
    "cfg1": Config("cfg1", 128, 256, 64, 1 << 24, 1 / 180, current=False),
    "cfg2": Config("cfg2", 128, 256, 64, 1 << 24, 1 / 180, current=False, adaptive=True, n_max=32),
    "cfg3": Config("cfg3", 256, 512, 128, 1 << 26, 1 / 360, current=True),
    "cfg4": Config("cfg4", 256, 1024, 128, 200_000_000, 1 / 360, current=True, adaptive=True,
                   n_max=16),
    "cfg4s": Config("cfg4s", 256, 1024, 128, 200_000_000, 1 / 360, current=True, adaptive=True,
                    n_max=16, order="sorted"),
}


# the paper's single-node workload: 512 x 1024 x 4
# cells, two kinetic species of 20e6 markers each -- deuterium with adaptive N_L and "heavy"
# electrons (m_i / m_e = 200).  What the paper does not print is read as follows (R21):
# rho*_i = 1/720, so that the thermal ion ring spans the same 0.71 radial cells as in cfg1-cfg4;
# equal temperatures, so rho*_e = rho*_i / sqrt(200); electrons are deposited drift-kinetically
# (N_L = 1: their ring is 0.05 cells wide); q_e = -1; species s uses seed s.  Both species add into
# the same rho / j_par (one handle per species: rho* and q belong to the grid descriptor).
CONFIGS["sn_ion"] = Config("sn_ion", 512, 1024, 4, 20_000_000, 1 / 720, current=True,
                           adaptive=True, n_max=32)
CONFIGS["sn_ele"] = Config("sn_ele", 512, 1024, 4, 20_000_000, 1 / (720 * math.sqrt(200.0)),
                           current=True, n_fixed=1, q=-1.0, seed=1)

# workload name -> the configs (species) deposited into the same grids in one step
WORKLOADS = {name: (name,) for name in CONFIGS}
WORKLOADS["single_node"] = ("sn_ion", "sn_ele")


def scaled(cfg: Config, n_markers: int, name: str | None = None) -> Config:
    """Same grid/policy, fewer markers (parity cases the oracle finishes quickly)."""
    return dataclasses.replace(cfg, n_markers=n_markers, name=name or f"{cfg.name}@{n_markers}")


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + _GOLD) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * _C1) & _M64
        z = ((z ^ (z >> np.uint64(27))) * _C2) & _M64
        return z ^ (z >> np.uint64(31))


def _uniform(seed: int, stream: int, idx: np.ndarray, attempt: int = 0) -> np.ndarray:
    """53-bit uniform in [0,1) from (seed, stream, attempt, index)."""
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0x100000001B3)
                          + np.uint64(stream) * np.uint64(0x9E3779B1)
                          + np.uint64(attempt) * np.uint64(0x85EBCA77C2B2AE63))
        h = _splitmix64(idx.astype(np.uint64) ^ key)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _normal(seed, s1, s2, idx):
    u1 = _uniform(seed, s1, idx)
    u2 = _uniform(seed, s2, idx)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(TWO_PI * u2)


def _field_strength(cfg: Config, s, thetastar):
    """|B| at the guiding centre for the mu = v_perp^2 / 2B column of the recipe
    (BASELINE.json cfg 0: B = 1/(1 + 0.3 s cos theta), theta the geometric angle
    belonging to the sampled straight-field-line angle)."""
    e = (cfg.a / cfg.r0) * s
    th = 2.0 * np.arctan2(np.sqrt(1.0 + e) * np.sin(0.5 * thetastar),
                          np.sqrt(1.0 - e) * np.cos(0.5 * thetastar))
    return cfg.b0 / (1.0 + e * np.cos(th))


def generate_chunk(cfg: Config, start: int, stop: int) -> dict:
    """Markers [start, stop) of the config, in generation (= random) order."""
    idx = np.arange(start, stop, dtype=np.uint64)
    sd = cfg.seed
    s = cfg.s_lo + (cfg.s_hi - cfg.s_lo) * _uniform(sd, S_S, idx)
    th = TWO_PI * _uniform(sd, S_TH, idx)
    ph = TWO_PI * _uniform(sd, S_PH, idx)
    vpar = _normal(sd, S_VP1, S_VP2, idx)
    w = cfg.w_sigma * _normal(sd, S_W1, S_W2, idx)
    B = _field_strength(cfg, s, th)
    vperp = np.sqrt(-2.0 * np.log1p(-_uniform(sd, S_VT, idx)))
    if cfg.adaptive:
        # R12: N_L = n_min*ceil(rho_L/rho_ref) is discontinuous; redraw any marker whose
        # ratio v_perp/B sits within 1e-9 of an integer so CPU and GPU agree on N_L.
        for attempt in range(1, 8):
            r = vperp / B
            bad = np.abs(r - np.rint(r)) < 1e-9
            if not bad.any():
                break
            vperp[bad] = np.sqrt(-2.0 * np.log1p(-_uniform(sd, S_VT, idx[bad], attempt)))
    mu = vperp * vperp / (2.0 * B)
    return dict(s=s, theta=th, phi=ph, vpar=vpar, mu=mu, w=w)


FIELDS = ("s", "theta", "phi", "vpar", "mu", "w")


def cell_key(cfg: Config, s, theta, phi) -> np.ndarray:
    """R17 sort key of the guiding-centre cell, phi-major: (k*Ns + i)*Ntheta + j."""
    i = np.minimum((s * cfg.ns).astype(np.int64), cfg.ns - 1)
    j = np.minimum((theta * (cfg.ntheta / TWO_PI)).astype(np.int64), cfg.ntheta - 1)
    k = np.minimum((phi * (cfg.nphi / TWO_PI)).astype(np.int64), cfg.nphi - 1)
    return (k * cfg.ns + i) * cfg.ntheta + j


def generate(cfg: Config, out: dict | None = None, chunk: int = 1 << 21, workers: int | None = None):
    """All markers of the config as six float64 arrays (dict keyed by FIELDS).

    ``out`` may hold preallocated arrays (e.g. numpy views of pinned torch
    tensors).  ``order == "sorted"`` applies the R17 cell sort afterwards.
    """
    n = cfg.n_markers
    if out is None:
        out = {f: np.empty(n, dtype=np.float64) for f in FIELDS}
    starts = list(range(0, n, chunk))

    def run(a):
        b = min(a + chunk, n)
        part = generate_chunk(cfg, a, b)
        for f in FIELDS:
            out[f][a:b] = part[f]

    workers = workers or min(os.cpu_count() or 1, 16)
    if workers > 1 and len(starts) > 1:
        with ThreadPoolExecutor(workers) as ex:
            list(ex.map(run, starts))
    else:
        for a in starts:
            run(a)
    if cfg.order == "sorted":
        perm = np.argsort(cell_key(cfg, out["s"], out["theta"], out["phi"]), kind="stable")
        for f in FIELDS:
            out[f][:] = out[f][perm]
    return out
