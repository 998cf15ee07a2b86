"""orb_deposit_noalloc (csrc/orb_noalloc.cu): the handle-free deposit whose scratch is a static
device array.  Its output is checked against the existing path (orb_grid_create + orb_markers_bind +
orb_deposit with the library's own pick of kernel) within the tolerance of the other parity tests
(1e-12 * max per grid), on calls in a row that change ns, N_L policy and alpha0 between them, so
that anything a call leaves behind in the shared scratch array would show.

The file name sorts last on purpose: the suite runs with `pytest -x`, and this test covers an
addition outside the hot path."""
import dataclasses

import pytest

from gpu_util import TOL, rel_err, to_device
from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W


def _cases():
    a = dataclasses.replace(W.scaled(W.CONFIGS["cfg2"], 60_007), current=True, ns=48, ntheta=96,
                            nphi=16, rho_star=1 / 90.0)                      # adaptive N_L
    b = dataclasses.replace(W.scaled(W.CONFIGS["cfg3"], 40_003), current=True, ns=20, ntheta=40,
                            nphi=12, rho_star=1 / 60.0, r0=1.7, a=0.5, b0=2.5, q=-1.5)   # N_L = 4
    return [(a, 0.0), (b, 0.37), (a, 0.0)]


def _desc(cfg):
    return B.GridDesc(cfg.ns, cfg.ntheta, cfg.nphi, cfg.r0, cfg.a, cfg.b0, cfg.rho_star, cfg.q, 1, 0)


def _policy(cfg, alpha0, flags=0):
    return B.policy(cfg.n_fixed, adaptive=cfg.adaptive, n_max=cfg.n_max if cfg.adaptive else None,
                    rho_ref=cfg.rho_ref, alpha0=alpha0, flags=flags)


def _existing_path(cfg, d, alpha0):
    import torch
    shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
    rho = torch.zeros(shape, dtype=torch.float64, device="cuda")
    jpar = torch.zeros(shape, dtype=torch.float64, device="cuda")
    g = B.grid_for(cfg)
    try:
        g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"], n=cfg.n_markers)
        g.deposit(rho, jpar, _policy(cfg, alpha0), torch.cuda.current_stream().cuda_stream)
        npts = g.last_points()
        torch.cuda.synchronize()
    finally:
        g.destroy()
    return rho.cpu().numpy(), jpar.cpu().numpy(), npts


@pytest.mark.gpu
def test_noalloc_matches_existing_path_on_calls_in_a_row():
    import torch
    st = torch.cuda.current_stream().cuda_stream
    prepared = []
    for cfg, alpha0 in _cases():
        d = to_device(W.generate(cfg))
        prepared.append((cfg, alpha0, d, _existing_path(cfg, d, alpha0)))
    grids = []
    for cfg, alpha0, d, _ in prepared:
        shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
        # deliberately dirty: ORB_DEPOSIT_ZERO_FIRST of the first call must clear them
        grids.append((torch.full(shape, 7.0, dtype=torch.float64, device="cuda"),
                      torch.full(shape, -3.0, dtype=torch.float64, device="cuda")))
    torch.cuda.synchronize()
    free_before = None
    # the calls follow each other on one stream, no synchronisation in between
    for rep in range(2):
        for (cfg, alpha0, d, _), (rho, jpar) in zip(prepared, grids):
            flags = B.ORB_DEPOSIT_ZERO_FIRST if rep == 0 else 0   # second round ADDS
            B.deposit_noalloc(_desc(cfg), d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"],
                              rho, jpar, _policy(cfg, alpha0, flags), st, n=cfg.n_markers)
        if rep == 0:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before     # the calls allocated no device memory
    for (cfg, alpha0, d, (rho_e, jpar_e, npts_e)), (rho, jpar) in zip(prepared, grids):
        assert rel_err(rho.cpu().numpy(), 2.0 * rho_e) <= TOL
        assert rel_err(jpar.cpu().numpy(), 2.0 * jpar_e) <= TOL
    # the synchronous form returns the point count; charge only (jpar, vpar NULL)
    for cfg, alpha0, d, (rho_e, _, npts_e) in prepared:
        rho = torch.empty((cfg.ns + 3, cfg.ntheta, cfg.nphi), dtype=torch.float64, device="cuda")
        npts = B.deposit_noalloc(_desc(cfg), d["s"], d["theta"], d["phi"], None, d["mu"], d["w"],
                                 rho, None, _policy(cfg, alpha0, B.ORB_DEPOSIT_ZERO_FIRST), st,
                                 n=cfg.n_markers, want_points=True)
        assert npts == npts_e
        assert rel_err(rho.cpu().numpy(), rho_e) <= TOL


@pytest.mark.gpu
def test_noalloc_empty_and_largest_ns():
    """n = 0 only zeroes; ns = ORB_NOALLOC_MAX_NS (the whole radial table) still matches."""
    import torch
    st = torch.cuda.current_stream().cuda_stream
    cfg = dataclasses.replace(W.scaled(W.CONFIGS["cfg3"], 20_011), current=True,
                              ns=B.ORB_NOALLOC_MAX_NS, ntheta=64, nphi=8, rho_star=1 / 2000.0,
                              s_lo=0.0, s_hi=1.0)
    d = to_device(W.generate(cfg))
    rho_e, jpar_e, npts_e = _existing_path(cfg, d, 0.0)
    shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
    rho = torch.ones(shape, dtype=torch.float64, device="cuda")
    assert B.deposit_noalloc(_desc(cfg), None, None, None, None, None, None, rho, None,
                             _policy(cfg, 0.0, B.ORB_DEPOSIT_ZERO_FIRST), st, n=0,
                             want_points=True) == 0
    assert float(rho.abs().max()) == 0.0
    jpar = torch.zeros_like(rho)
    npts = B.deposit_noalloc(_desc(cfg), d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"],
                             rho, jpar, _policy(cfg, 0.0), st, n=cfg.n_markers, want_points=True)
    assert npts == npts_e
    assert rel_err(rho.cpu().numpy(), rho_e) <= TOL
    assert rel_err(jpar.cpu().numpy(), jpar_e) <= TOL


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    """ns > ORB_NOALLOC_MAX_NS: ORB_E_INVAL with a message that names the limit (checked before
    any device call, so this runs without a GPU too); so do the other argument errors."""
    desc = B.GridDesc(B.ORB_NOALLOC_MAX_NS + 1, 32, 16, 1.0, 0.3, 1.0, 1 / 180, 1.0, 1, 0)
    with pytest.raises(B.OrbError) as e:
        B.deposit_noalloc(desc, None, None, None, None, None, None, None, None, B.policy(4), None, n=0)
    assert e.value.code == B.ORB_E_INVAL
    assert "ORB_NOALLOC_MAX_NS = %d" % B.ORB_NOALLOC_MAX_NS in str(e.value)
    ok = B.GridDesc(16, 32, 16, 1.0, 0.3, 1.0, 1 / 180, 1.0, 1, 0)
    with pytest.raises(B.OrbError) as e:      # rho NULL
        B.deposit_noalloc(ok, None, None, None, None, None, None, None, None, B.policy(4), None, n=0)
    assert e.value.code == B.ORB_E_INVAL
    with pytest.raises(B.OrbError) as e:      # a flag that selects another algorithm
        B.deposit_noalloc(ok, None, None, None, None, None, None, 16, None,
                          B.policy(4, flags=B.ORB_DEPOSIT_ALGO_TILE_V4), None, n=0)
    assert e.value.code == B.ORB_E_INVAL
    assert B.lib().orb_deposit_noalloc(None, 0, None, None, None, None, None, None, None, None, None,
                                       None, None, None, 0) == B.ORB_E_INVAL
