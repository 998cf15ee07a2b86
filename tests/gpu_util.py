"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle,
compare element by element.  Tolerance (north_star, R19): per grid
max|gpu - oracle| <= 1e-12 * max|oracle|."""
import dataclasses

import numpy as np

import oracle as O
from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W

TOL = 1e-12


def oracle_geom(cfg):
    return O.geom(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0,
                  rho_star=cfg.rho_star, q=cfg.q)


def oracle_policy(cfg):
    if cfg.adaptive:
        return O.policy_adaptive(cfg.n_fixed, cfg.n_max, cfg.rho_ref)
    return O.policy_fixed(cfg.n_fixed)


def run_oracle(cfg, m, workers=None):
    rho, jpar, npts, _ = O.deposit_ranges(oracle_geom(cfg), oracle_policy(cfg),
                                          *(m[f] for f in W.FIELDS), current=cfg.current,
                                          workers=workers)
    return rho, jpar, npts


def to_device(m):
    import torch
    return {f: torch.from_numpy(np.ascontiguousarray(m[f])).cuda() for f in W.FIELDS}


def prepare(g, cfg, flags):
    """Scratch an algorithm flag needs before orb_deposit (the ring-data path reserves its Larmor
    ring data outside the deposit call)."""
    if flags & B.ORB_DEPOSIT_ALGO_RING_DATA:
        g.ring_reserve(cfg.n_markers, cfg.n_markers * (cfg.n_max if cfg.adaptive else cfg.n_fixed))


def run_gpu(cfg, m, flags=0, bind_flags=0, dev=None, bin_first=False, theta_map=1, repeat=1):
    """One orb_deposit through the C ABI on cuda:0. -> (rho, jpar, n_points) as numpy."""
    import torch
    d = dev if dev is not None else to_device(m)
    shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
    rho = torch.zeros(shape, dtype=torch.float64, device="cuda")
    jpar = torch.zeros(shape, dtype=torch.float64, device="cuda") if cfg.current else None
    g = B.Grid(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0, rho_star=cfg.rho_star,
               q=cfg.q, theta_map=theta_map)
    try:
        g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"] if cfg.current else None,
                       d["mu"], d["w"], flags=bind_flags, n=cfg.n_markers)
        st = torch.cuda.current_stream().cuda_stream
        if bin_first:
            g.markers_bin(st)
        pol = B.policy_for(cfg, flags=flags)
        prepare(g, cfg, flags)
        for _ in range(repeat):
            g.deposit(rho, jpar, pol, st)
        npts = g.last_points()
        torch.cuda.synchronize()
    finally:
        g.destroy()
    return rho.cpu().numpy(), (jpar.cpu().numpy() if cfg.current else None), npts


def rel_err(got, want):
    return float(np.abs(got - want).max() / np.abs(want).max())


def assert_parity(got, want, what=""):
    err = rel_err(got, want)
    assert err <= TOL, "%s: max|gpu-oracle| / max|oracle| = %.3e > %.0e" % (what, err, TOL)
    return err
