"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(bind -> orb_markers_bin -> orb_grid_zero -> orb_deposit, tile kernel).

cfg1, cfg2, cfg3: the whole grid against the oracle run over all markers (marker ranges on all
host cores, summed in fixed order -- oracle.deposit_ranges).
cfg4 (2e8 markers, random and pre-sorted): the WHOLE grid, element by element, against the
oracle run over all markers once (marker ranges on all host cores, one private grid replica per
range, summed in fixed order: ~9 GB of replicas on 16 cores); the pre-sorted run is compared
with the same oracle grids (deposition does not depend on the marker order, PAPER.md:75, 97;
pin P11).  Only if the host is short of memory for the replicas does the test fall back to 16
sampled toroidal node planes (a plane k receives contributions only from markers whose phi
cell is k-2 .. k+1, so the oracle deposit of just those markers gives every node of it).
Plus properties that hold at any size: charge/current conservation (P1) and the point count.

Tolerance (north_star, R19): max|gpu - oracle| <= 1e-12 * max|oracle| per grid.
"""
import os

import numpy as np
import pytest

import oracle as O
from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W

from gpu_util import TOL, oracle_geom, oracle_policy, rel_err

pytestmark = pytest.mark.gpu


def _host_mem_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable"):
                    return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def _bench_step(cfg, d, bind_flags=0):
    """The step bench.py times, once, on device-resident markers. -> (rho, jpar, n_points, g)"""
    import torch
    g = B.grid_for(cfg)
    shape = g.shape()
    rho = torch.full(shape, 7.0, dtype=torch.float64, device="cuda")   # must be zeroed by the step
    jpar = torch.full(shape, -3.0, dtype=torch.float64, device="cuda") if cfg.current else None
    st = torch.cuda.current_stream().cuda_stream
    g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"] if cfg.current else None, d["mu"],
                   d["w"], flags=bind_flags)
    g.markers_bin(st)
    g.grid_zero(rho, jpar, st)
    g.deposit(rho, jpar, B.policy_for(cfg), st)
    torch.cuda.synchronize()
    npts = g.last_points()
    fallback = g.last_fallback_points()
    g.destroy()
    return rho, jpar, npts, fallback


def _conservation(cfg, m, rho, jpar):
    scale = abs(cfg.q) * np.abs(m["w"]).sum()
    assert abs(float(rho.sum().item()) - cfg.q * m["w"].sum()) <= 1e-11 * scale
    if cfg.current:
        scale_j = abs(cfg.q) * np.abs(m["w"] * m["vpar"]).sum()
        assert abs(float(jpar.sum().item()) - cfg.q * (m["w"] * m["vpar"]).sum()) <= 1e-11 * scale_j


BINNINGS = {"tile_bins": B.ORB_MARKERS_TILE_BINS, "dense": 0}   # bench.py --binning tile | dense


@pytest.mark.parametrize("binning", list(BINNINGS))
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3"])
def test_full_grid_against_oracle(name, binning):
    import torch
    cfg = W.CONFIGS[name]
    m = W.generate(cfg)
    d = {f: torch.from_numpy(m[f]).cuda() for f in W.FIELDS}
    rho, jpar, npts, fallback = _bench_step(cfg, d, bind_flags=BINNINGS[binning])
    del d
    rho_o, jpar_o, npts_o, _ = O.deposit_ranges(oracle_geom(cfg), oracle_policy(cfg),
                                                *(m[f] for f in W.FIELDS), current=cfg.current)
    assert npts == npts_o
    assert fallback < 0.01 * npts          # the shared-memory tile path carries the load
    err = rel_err(rho.cpu().numpy(), rho_o)
    assert err <= TOL, "%s rho: %.3e" % (name, err)
    if cfg.current:
        errj = rel_err(jpar.cpu().numpy(), jpar_o)
        assert errj <= TOL, "%s jpar: %.3e" % (name, errj)
    _conservation(cfg, m, rho, jpar)


@pytest.fixture(scope="module")
def cfg4_case():
    if _host_mem_gb() < 60.0:
        pytest.skip("cfg4 needs ~40 GB of host memory")
    import torch
    if torch.cuda.mem_get_info()[1] < 60e9:
        pytest.skip("cfg4 needs ~25 GB of device memory")
    cfg = W.CONFIGS["cfg4"]
    m = W.generate(cfg)
    og, op = oracle_geom(cfg), oracle_policy(cfg)
    grid_gb = 2 * cfg.nodes * 8 / 1e9                      # rho + jpar of one replica
    workers = min(os.cpu_count() or 1, 32)
    want = {}
    if _host_mem_gb() > workers * grid_gb + 30.0:
        rho_o, jpar_o, npts, _ = O.deposit_ranges(og, op, *(m[f] for f in W.FIELDS), current=True,
                                                  workers=workers)
        want["full"] = (rho_o, jpar_o)
    else:   # fallback: 16 sampled node planes, each from the markers of the 4 phi cells around it
        kcell = np.minimum((m["phi"] * (cfg.nphi / W.TWO_PI)).astype(np.int64), cfg.nphi - 1)
        planes = {}
        for k0 in sorted({0, 1, cfg.nphi - 2, cfg.nphi - 1, *range(5, cfg.nphi, 10)})[:16]:
            near = ((kcell - k0 + 2) % cfg.nphi) < 4          # phi cells k0-2 .. k0+1
            sub = [np.ascontiguousarray(m[f][near]) for f in W.FIELDS]
            rho_o, jpar_o, _, _ = O.deposit_ranges(og, op, *sub, current=True, workers=4)
            planes[k0] = (rho_o[:, :, k0].copy(), jpar_o[:, :, k0].copy())
        want["planes"] = planes
        _, npts = O.nl_histogram(og, op, m["s"], m["theta"], m["mu"])
    return cfg, m, want, npts


def _check_grids(rho, jpar, want):
    if "full" in want:
        rho_o, jpar_o = want["full"]
        err = rel_err(rho.cpu().numpy(), rho_o)
        assert err <= TOL, "cfg4 rho, whole grid: %.3e" % err
        errj = rel_err(jpar.cpu().numpy(), jpar_o)
        assert errj <= TOL, "cfg4 jpar, whole grid: %.3e" % errj
        return
    for k0, (rho_o, jpar_o) in want["planes"].items():
        got = rho[:, :, k0].cpu().numpy()
        assert np.abs(got - rho_o).max() <= TOL * np.abs(rho_o).max(), "rho plane %d" % k0
        gotj = jpar[:, :, k0].cpu().numpy()
        assert np.abs(gotj - jpar_o).max() <= TOL * np.abs(jpar_o).max(), "jpar plane %d" % k0


@pytest.mark.parametrize("binning", list(BINNINGS))
def test_cfg4_random_order_whole_grid(cfg4_case, binning):
    import torch
    cfg, m, want, npts_o = cfg4_case
    d = {f: torch.from_numpy(m[f]).cuda() for f in W.FIELDS}
    rho, jpar, npts, fallback = _bench_step(cfg, d, bind_flags=BINNINGS[binning])
    del d
    assert npts == npts_o
    assert fallback < 0.01 * npts
    _check_grids(rho, jpar, want)
    _conservation(cfg, m, rho, jpar)


def test_cfg4_presorted_whole_grid(cfg4_case):
    """R17: same markers pre-sorted by cell key on the host, bound with ORB_MARKERS_SORTED."""
    import torch
    cfg, m, want, npts_o = cfg4_case
    perm = np.argsort(W.cell_key(cfg, m["s"], m["theta"], m["phi"]), kind="stable")
    d = {f: torch.from_numpy(m[f][perm]).cuda() for f in W.FIELDS}
    del perm
    rho, jpar, npts, fallback = _bench_step(cfg, d, bind_flags=B.ORB_MARKERS_SORTED)
    del d
    assert npts == npts_o
    _check_grids(rho, jpar, want)
    _conservation(cfg, m, rho, jpar)


@pytest.mark.parametrize("adaptive", [True, False])
def test_deposit_host_sliced_pipeline(adaptive):
    """orb_deposit_host above 2^22 markers: the host->device copies travel in slices, each slice is
    appended to the slack tile bins when it lands, and the deposit kernel runs once per group of
    slices (per slice for the algorithms that read the bound arrays).  Result and point count must
    not depend on the slicing: adaptive N_L (block-per-tile kernel), fixed N_L = 4 (persistent
    kernel), and the global-atomics algorithm, against the oracle on all markers."""
    import dataclasses
    cfg = dataclasses.replace(W.scaled(W.CONFIGS["cfg4"], (1 << 22) + 12_345), ns=64, ntheta=128,
                              nphi=32, rho_star=1 / 120.0)
    if not adaptive:
        cfg = dataclasses.replace(cfg, adaptive=False, n_fixed=4)
    m = W.generate(cfg)
    rho_o, jpar_o, npts_o, _ = O.deposit_ranges(oracle_geom(cfg), oracle_policy(cfg),
                                                *(m[f] for f in W.FIELDS), current=True)
    g = B.grid_for(cfg)
    rho = np.empty((cfg.ns + 3, cfg.ntheta, cfg.nphi))
    jpar = np.empty_like(rho)
    for flags in (0, 0, B.ORB_DEPOSIT_ALGO_ATOMIC, 0):   # repeated calls reuse streams and scratch
        rho.fill(np.nan)
        jpar.fill(np.nan)
        npts, up, down = g.deposit_host(m["s"], m["theta"], m["phi"], m["vpar"], m["mu"], m["w"],
                                        rho, jpar, B.policy_for(cfg, flags=flags))
        assert npts == npts_o and up == 6 * 8 * cfg.n_markers and down == 2 * rho.nbytes
        assert rel_err(rho, rho_o) <= TOL
        assert rel_err(jpar, jpar_o) <= TOL
    # the handle stays bound to the library's device copy: a device-side deposit gives the same
    import torch
    rho_d = torch.zeros(rho.shape, dtype=torch.float64, device="cuda")
    g.deposit(rho_d, None, B.policy_for(cfg, flags=B.ORB_DEPOSIT_ZERO_FIRST))
    torch.cuda.synchronize()
    assert rel_err(rho_d.cpu().numpy(), rho_o) <= TOL
    g.destroy()


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_gather_full_size_sampled_markers(name):
    """orb_gather (NEXT-1) at full size in the configuration bench.py times (bind -> bin ->
    gather of 2 fields): the GPU computes every marker; a marker's result depends on that marker
    alone, so the oracle computes a seeded sample of 2^21 markers one by one and those outputs
    are compared element by element.  Property at full size: a constant field returns 1 for
    every marker (partition of unity), which also proves every marker was written."""
    import torch
    if name == "cfg4" and (_host_mem_gb() < 60.0 or torch.cuda.mem_get_info()[1] < 60e9):
        pytest.skip("cfg4 needs ~40 GB of host and ~25 GB of device memory")
    cfg = W.CONFIGS[name]
    m = W.generate(cfg)
    n = cfg.n_markers
    rng = np.random.default_rng(17)
    shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
    fields = [rng.standard_normal(shape), np.ones(shape)]
    d = {f: torch.from_numpy(m[f]).cuda() for f in W.FIELDS if f != "vpar"}
    fd = [torch.from_numpy(f).cuda() for f in fields]
    out = [torch.full((n,), np.nan, dtype=torch.float64, device="cuda") for _ in fields]
    g = B.grid_for(cfg)
    st = torch.cuda.current_stream().cuda_stream
    g.markers_bind(d["s"], d["theta"], d["phi"], None, d["mu"], d["w"])
    g.markers_bin(st)
    g.gather(fd, out, B.policy_for(cfg), st)
    torch.cuda.synchronize()
    npts, fallback = g.last_points(), g.last_fallback_points()
    g.destroy()
    assert fallback < 0.01 * npts
    ones = out[1].cpu().numpy()
    assert np.abs(ones - 1.0).max() <= 1e-13
    idx = np.sort(rng.choice(n, size=1 << 21, replace=False))
    want, _ = O.gather(oracle_geom(cfg), oracle_policy(cfg), m["s"][idx], m["theta"][idx],
                       m["phi"][idx], m["mu"][idx], fields[0], workers=os.cpu_count())
    got = out[0][torch.from_numpy(idx).cuda()].cpu().numpy()
    assert np.abs(got - want).max() <= TOL * np.abs(want).max()
    _, npts_o = O.nl_histogram(oracle_geom(cfg), oracle_policy(cfg), m["s"], m["theta"], m["mu"])
    assert npts == npts_o


def test_single_node_two_species_workload():
    """SURVEY 8(f) NEXT-4, the paper's single-node case: 512 x 1024 x 4 cells,
    deuterium (adaptive N_L) and heavy electrons (N_L = 1, q = -1) of 20e6 markers each, both
    added into the same rho / j_par.  N_phi = 4: every point touches all four toroidal node
    planes through the periodic wrap.  Whole grid against the oracle."""
    import torch
    cfgs = [W.CONFIGS[n] for n in W.WORKLOADS["single_node"]]
    shape = (cfgs[0].ns + 3, cfgs[0].ntheta, cfgs[0].nphi)
    rho = torch.full(shape, 5.0, dtype=torch.float64, device="cuda")
    jpar = torch.full(shape, -1.0, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    rho_o, jpar_o = np.zeros(shape), np.zeros(shape)
    w_sum = 0.0
    for i, cfg in enumerate(cfgs):
        m = W.generate(cfg)
        d = {f: torch.from_numpy(m[f]).cuda() for f in W.FIELDS}
        g = B.grid_for(cfg)
        g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"])
        g.markers_bin(st)
        if i == 0:
            g.grid_zero(rho, jpar, st)
        g.deposit(rho, jpar, B.policy_for(cfg), st)
        torch.cuda.synchronize()
        npts, fallback = g.last_points(), g.last_fallback_points()
        g.destroy()
        r, j, npts_o, _ = O.deposit_ranges(oracle_geom(cfg), oracle_policy(cfg),
                                           *(m[f] for f in W.FIELDS), current=True)
        rho_o += r
        jpar_o += j
        w_sum += cfg.q * m["w"].sum()
        assert npts == npts_o
        assert fallback < 0.02 * npts
    assert rel_err(rho.cpu().numpy(), rho_o) <= TOL
    assert rel_err(jpar.cpu().numpy(), jpar_o) <= TOL
    assert abs(float(rho.sum().item()) - w_sum) <= 1e-11 * 2e7 * 1e-3
