"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs."""
import dataclasses
import math

import numpy as np
import pytest

from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W

from gpu_util import (assert_parity, oracle_geom, oracle_policy, rel_err, run_gpu, run_oracle,
                      to_device)

pytestmark = pytest.mark.gpu

ALGOS = {
    "atomic": B.ORB_DEPOSIT_ALGO_ATOMIC,
    "atomic_nobin": B.ORB_DEPOSIT_ALGO_ATOMIC | B.ORB_DEPOSIT_NO_BIN,
    "tile_v4": B.ORB_DEPOSIT_ALGO_TILE_V4,
    "tile": 0,          # the product path: persistent warp-specialised tile kernel (v5)
}


def small(cfg_name, n, **kw):
    return dataclasses.replace(W.scaled(W.CONFIGS[cfg_name], n), **kw)


CASES = {
    # name: config (sizes span several tiles and a ragged tail; oracle finishes in seconds)
    "cfg0": W.CONFIGS["cfg0"],
    "cfg0_current": small("cfg0", 50_001, current=True),
    "cfg1_small": small("cfg1", 300_007),
    "cfg2_small": small("cfg2", 200_003),
    "cfg3_small": small("cfg3", 250_001),
    "cfg4_small": small("cfg4", 150_011),
    "cfg4s_small": small("cfg4s", 150_011),
    "edge_rings": small("cfg0", 20_011, current=True, s_lo=0.0, s_hi=1.0, rho_star=1 / 25.0),
    "odd_grid": small("cfg0", 30_013, current=True, ns=23, ntheta=37, nphi=19, s_lo=0.0, s_hi=1.0),
    "tiny_grid": small("cfg0", 5_003, current=True, ns=4, ntheta=4, nphi=4, s_lo=0.0, s_hi=1.0),
    "nl1": small("cfg0", 40_009, current=True, n_fixed=1),
    "nl7": small("cfg0", 20_011, current=True, n_fixed=7),
    "nl32": small("cfg0", 5_003, current=True, n_fixed=32, rho_star=1 / 40.0),
}


@pytest.fixture(scope="module")
def oracle_results():
    return {}


def get_case(name, oracle_results):
    if name not in oracle_results:
        cfg = CASES[name]
        m = W.generate(cfg)
        oracle_results[name] = (cfg, m, run_oracle(cfg, m))
    return oracle_results[name]


@pytest.mark.parametrize("algo", list(ALGOS))
@pytest.mark.parametrize("name", list(CASES))
def test_parity(name, algo, oracle_results):
    cfg, m, (rho_o, jpar_o, npts_o) = get_case(name, oracle_results)
    bind_flags = B.ORB_MARKERS_SORTED if cfg.order == "sorted" else 0
    rho, jpar, npts = run_gpu(cfg, m, flags=ALGOS[algo], bind_flags=bind_flags)
    assert npts == npts_o
    assert_parity(rho, rho_o, "%s/%s rho" % (name, algo))
    if cfg.current:
        assert_parity(jpar, jpar_o, "%s/%s jpar" % (name, algo))
    # conservation (P1) on the GPU result itself
    scale = cfg.q * np.abs(m["w"]).sum()
    assert abs(rho.sum() - cfg.q * m["w"].sum()) < 1e-12 * scale


def test_theta_map_identity(oracle_results):
    """theta_map = 0 (theta* == theta) switch."""
    import oracle as O
    cfg = small("cfg0", 20_011, current=True)
    m = W.generate(cfg)
    g = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, rho_star=cfg.rho_star, theta_map=0)
    rho_o, jpar_o, _ = O.deposit(g, oracle_policy(cfg), *(m[f] for f in W.FIELDS))
    for algo in ALGOS.values():
        rho, jpar, _ = run_gpu(cfg, m, flags=algo, theta_map=0)
        assert_parity(rho, rho_o)
        assert_parity(jpar, jpar_o)


def test_deposit_adds_and_zero_first():
    cfg = small("cfg0", 10_007, current=True)
    m = W.generate(cfg)
    r1, j1, _ = run_gpu(cfg, m)
    r2, j2, _ = run_gpu(cfg, m, repeat=2)
    assert rel_err(r2, 2 * r1) < 1e-13 and rel_err(j2, 2 * j1) < 1e-13
    r3, j3, _ = run_gpu(cfg, m, flags=B.ORB_DEPOSIT_ZERO_FIRST, repeat=2)
    assert rel_err(r3, r1) < 1e-13 and rel_err(j3, j1) < 1e-13


def test_all_markers_in_one_cell_conserves_charge():
    """Atomics stress: every marker in the same cell; charge must be conserved."""
    import oracle as O
    cfg = small("cfg0", 100_003, current=True)
    m = W.generate(cfg)
    m["s"][:] = 0.5 + 1e-3 * (m["s"] - 0.5)
    m["theta"][:] = 1.0 + 1e-3 * m["theta"]
    m["phi"][:] = 2.0 + 1e-3 * m["phi"]
    rho_o, jpar_o, _ = run_oracle(cfg, m)
    for algo in ALGOS.values():
        rho, jpar, _ = run_gpu(cfg, m, flags=algo)
        assert_parity(rho, rho_o)
        assert_parity(jpar, jpar_o)
        assert abs(rho.sum() - m["w"].sum()) < 1e-12 * np.abs(m["w"]).sum()


def test_empty_and_single_marker():
    import torch
    cfg = small("cfg0", 1, current=True)
    m = W.generate(cfg)
    rho_o, jpar_o, _ = run_oracle(cfg, m)
    for algo in ALGOS.values():
        rho, jpar, npts = run_gpu(cfg, m, flags=algo)
        assert npts == 4
        assert_parity(rho, rho_o)
    # n = 0
    g = B.Grid(16, 32, 16)
    z = torch.zeros(2, dtype=torch.float64, device="cuda")
    rho = torch.zeros(g.shape(), dtype=torch.float64, device="cuda")
    g.markers_bind(z, z, z, z, z, z, n=0)
    g.deposit(rho, None, B.policy(4), torch.cuda.current_stream().cuda_stream)
    assert g.last_points() == 0 and float(rho.abs().max()) == 0.0
    g.destroy()


def test_binning_is_a_sort(oracle_results):
    """a7: binned order has non-decreasing cell keys, is a permutation, and the separately run
    bin pass + deposit equals deposit alone (P11)."""
    cfg, m, (rho_o, _, _) = get_case("cfg1_small", oracle_results)
    rho_a, _, _ = run_gpu(cfg, m, bin_first=True)
    assert_parity(rho_a, rho_o)


def test_error_codes():
    import torch
    g = B.Grid(16, 32, 16)
    rho = torch.zeros(g.shape(), dtype=torch.float64, device="cuda")
    with pytest.raises(B.OrbError) as e:
        g.deposit(rho, None, B.policy(4))
    assert e.value.code == B.ORB_E_STATE
    z = torch.zeros(16, dtype=torch.float64, device="cuda")
    g.markers_bind(z, z, z, None, z, z)
    with pytest.raises(B.OrbError) as e:
        g.deposit(rho, rho, B.policy(4))        # jpar without vpar
    assert e.value.code == B.ORB_E_INVAL
    for bad in (B.policy(0), B.policy(33), B.policy(4, adaptive=True, n_max=2, rho_ref=1.0),
                B.policy(4, adaptive=True, n_max=8, rho_ref=0.0)):
        with pytest.raises(B.OrbError) as e:
            g.deposit(rho, None, bad)
        assert e.value.code == B.ORB_E_INVAL
    with pytest.raises(B.OrbError) as e:
        g.markers_bind(z[1:], z, z, None, z, z, n=8)   # misaligned
    assert e.value.code == B.ORB_E_INVAL
    g.destroy()


def test_deposit_host_roundtrip(oracle_results):
    cfg, m, (rho_o, jpar_o, npts_o) = get_case("cfg3_small", oracle_results)
    g = B.grid_for(cfg)
    rho = np.empty((cfg.ns + 3, cfg.ntheta, cfg.nphi))
    jpar = np.empty_like(rho)
    npts, up, down = g.deposit_host(m["s"], m["theta"], m["phi"], m["vpar"], m["mu"], m["w"],
                                    rho, jpar, B.policy_for(cfg))
    g.destroy()
    assert npts == npts_o and up == 6 * 8 * cfg.n_markers and down == 2 * rho.nbytes
    assert_parity(rho, rho_o)
    assert_parity(jpar, jpar_o)


@pytest.mark.parametrize("adaptive", [False, True])
def test_nondefault_geometry_charge_field_and_gyrophase(adaptive):
    """Every descriptor / policy field away from its default: r0, a, b0, q, rho_star, alpha0
    (R1, R2, R6, R7, R10), fixed and adaptive N_L, all three algorithms."""
    import torch
    import oracle as O
    cfg = small("cfg0", 30_011, current=True, ns=20, ntheta=40, nphi=12, r0=1.7, a=0.5, b0=2.5,
                q=-1.5, rho_star=1 / 60.0, adaptive=adaptive, n_fixed=4 if adaptive else 6,
                n_max=16 if adaptive else 6, s_lo=0.02, s_hi=0.98)
    alpha0 = 0.37
    m = W.generate(cfg)
    og = oracle_geom(cfg)
    op = (O.policy_adaptive(cfg.n_fixed, cfg.n_max, cfg.rho_ref, alpha0) if adaptive
          else O.policy_fixed(cfg.n_fixed, alpha0))
    rho_o, jpar_o, npts_o = O.deposit(og, op, *(m[f] for f in W.FIELDS), current=True)
    d = to_device(m)
    for flags in ALGOS.values():
        g = B.grid_for(cfg)
        rho = torch.zeros(g.shape(), dtype=torch.float64, device="cuda")
        jpar = torch.zeros_like(rho)
        g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"])
        pol = B.policy(cfg.n_fixed, adaptive=adaptive, n_max=cfg.n_max if adaptive else None,
                       rho_ref=cfg.rho_ref, alpha0=alpha0, flags=flags)
        g.deposit(rho, jpar, pol, torch.cuda.current_stream().cuda_stream)
        npts = g.last_points()
        g.destroy()
        assert npts == npts_o
        assert_parity(rho.cpu().numpy(), rho_o, "rho flags=%d" % flags)
        assert_parity(jpar.cpu().numpy(), jpar_o, "jpar flags=%d" % flags)


def test_fp64_probe_is_plausible():
    """orb_probe_dfma (the roof bench.py reports roofline_alu against): between half and 1.2x of
    the nominal SMs x 64 lanes x 2 flop x clock."""
    import torch
    p = torch.cuda.get_device_properties(0)
    nominal = p.multi_processor_count * 64 * 2 * (p.clock_rate * 1e3 if hasattr(p, "clock_rate") else 1.965e9) / 1e12
    got = B.probe_dfma(0)
    assert 0.5 * nominal < got < 1.2 * nominal, (got, nominal)
