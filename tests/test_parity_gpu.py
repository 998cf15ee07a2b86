"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs."""
import dataclasses
import math

import numpy as np
import pytest

from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W

from gpu_util import (assert_parity, oracle_geom, oracle_policy, prepare, rel_err, run_gpu,
                      run_oracle, to_device)

pytestmark = pytest.mark.gpu

ALGOS = {
    "atomic": B.ORB_DEPOSIT_ALGO_ATOMIC,
    "atomic_nobin": B.ORB_DEPOSIT_ALGO_ATOMIC | B.ORB_DEPOSIT_NO_BIN,
    "tile_v4": B.ORB_DEPOSIT_ALGO_TILE_V4,       # one block per tile
    "tile_ws": B.ORB_DEPOSIT_ALGO_TILE_WS,       # persistent, warp-specialised, 64-byte operand records
    "ring_data": B.ORB_DEPOSIT_ALGO_RING_DATA,   # NEXT-3: Larmor ring data + cell-owner loop
    "tile": 0,          # the product path: the library picks by N_L policy (fixed N_L <= 4: the
                        # persistent kernel with whole-tile chunks, orb_deposit_ws2.cu)
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


def _binned(cfg, m, bind_flags=0):
    """Runs orb_markers_bin alone and reads the binned order back (orb_debug_binned)."""
    import torch
    d = to_device(m)
    g = B.grid_for(cfg)
    g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"], flags=bind_flags)
    g.markers_bin(torch.cuda.current_stream().cuda_stream)
    rec, cs = g.debug_binned(cfg.n_markers)
    g.destroy()
    return rec, cs


def test_binning_is_a_sort(oracle_results):
    """a7 (bucket sort of PAPER.md:167; R17, R18): the binned order has non-decreasing cell keys,
    the per-cell offsets are the histogram's exclusive scan, the records are a permutation of the
    bound markers (multiset preserved), and bin pass + deposit equals the oracle (P11)."""
    cfg, m, (rho_o, _, _) = get_case("cfg1_small", oracle_results)
    n = cfg.n_markers
    rec, cs = _binned(cfg, m)
    assert rec is not None and rec.shape == (n, 8)
    key_in = W.cell_key(cfg, m["s"], m["theta"], m["phi"])
    key_out = W.cell_key(cfg, rec[:, 0], rec[:, 1], rec[:, 2])
    assert (np.diff(key_out) >= 0).all(), "binned keys must be non-decreasing"
    ncells = cfg.ns * cfg.ntheta * cfg.nphi
    hist = np.bincount(key_in, minlength=ncells)
    assert cs[0] == 0 and cs[-1] == n
    assert (np.diff(cs.astype(np.int64)) == hist).all(), "cell_start must be the exclusive scan"
    # every record sits inside its own cell's range
    assert (cs[key_out] <= np.arange(n)).all() and (np.arange(n) < cs[key_out + 1]).all()
    # multiset of markers preserved (all six fields, bit for bit)
    src = np.stack([m[f] for f in W.FIELDS], axis=1)
    order_in = np.lexsort(src.T[::-1])
    order_out = np.lexsort(rec[:, :6].T[::-1])
    assert (src[order_in].view(np.uint64) == rec[order_out, :6].view(np.uint64)).all()
    # slot 6 carries the marker's index in bound order (what orb_gather writes results back by)
    orig = rec[:, 6].copy().view(np.int64)
    assert (np.sort(orig) == np.arange(n)).all()
    assert (src[orig].view(np.uint64) == rec[:, :6].view(np.uint64)).all()
    assert (rec[:, 7] == 0).all()
    rho_a, _, _ = run_gpu(cfg, m, bin_first=True)
    assert_parity(rho_a, rho_o)


def test_binning_of_presorted_markers_locates_cells(oracle_results):
    """ORB_MARKERS_SORTED: no records are written; cell_start alone must delimit the cells."""
    cfg, m, _ = get_case("cfg4s_small", oracle_results)
    rec, cs = _binned(cfg, m, bind_flags=B.ORB_MARKERS_SORTED)
    assert rec is None
    key = W.cell_key(cfg, m["s"], m["theta"], m["phi"])
    assert (np.diff(key) >= 0).all()
    hist = np.bincount(key, minlength=cfg.ns * cfg.ntheta * cfg.nphi)
    assert (np.diff(cs.astype(np.int64)) == hist).all()


def test_sorted_flag_on_unsorted_markers_stays_correct(oracle_results):
    """ORB_MARKERS_SORTED is a hint (include/orb.h): bound to markers that are NOT sorted the
    result must still be the oracle's (sorted == unsorted)."""
    for name in ("cfg3_small", "cfg4_small"):
        cfg, m, (rho_o, jpar_o, npts_o) = get_case(name, oracle_results)
        for algo in ("tile", "tile_ws", "tile_v4"):
            rho, jpar, npts = run_gpu(cfg, m, flags=ALGOS[algo], bind_flags=B.ORB_MARKERS_SORTED)
            assert npts == npts_o
            assert_parity(rho, rho_o, "%s/%s rho" % (name, algo))
            assert_parity(jpar, jpar_o, "%s/%s jpar" % (name, algo))


@pytest.mark.parametrize("adaptive", [False, True])
def test_angles_outside_0_2pi_and_radial_bounds(adaptive):
    """include/orb.h: theta*, phi are 'any finite angle' (R13 wrap) and s in [0, 1] INCLUSIVE.
    theta*, phi in [-7 pi, 9 pi]; a share of the markers has s exactly 0 and exactly 1, angles
    exactly 0, 2 pi, -2 pi and on cell boundaries."""
    cfg = small("cfg0", 60_013, current=True, s_lo=0.0, s_hi=1.0, adaptive=adaptive,
                n_max=16 if adaptive else 4, rho_star=1 / 60.0)
    m = W.generate(cfg)
    n = cfg.n_markers
    turns = (np.arange(n) % 8) - 4                         # -4 .. 3 full turns
    m["theta"] = m["theta"] + W.TWO_PI * turns + (np.arange(n) % 2) * np.pi   # [-8pi, 9pi)
    m["theta"] = np.clip(m["theta"], -7 * np.pi, 9 * np.pi)
    m["phi"] = m["phi"] + W.TWO_PI * ((np.arange(n) // 8) % 8 - 3.5)          # [-7pi, 9pi)
    m["s"][0:n:17] = 0.0
    m["s"][1:n:17] = 1.0
    m["theta"][2:n:17] = 0.0
    m["theta"][3:n:17] = W.TWO_PI
    m["theta"][4:n:17] = -W.TWO_PI
    m["phi"][5:n:17] = 0.0
    m["phi"][6:n:17] = W.TWO_PI
    m["phi"][7:n:17] = 3 * W.TWO_PI / cfg.nphi             # on a cell boundary
    m["theta"][8:n:17] = -5 * W.TWO_PI / cfg.ntheta
    assert m["theta"].min() < -6 * np.pi and m["theta"].max() > 8 * np.pi
    assert m["phi"].min() < -6 * np.pi and m["phi"].max() > 8 * np.pi
    rho_o, jpar_o, npts_o = run_oracle(cfg, m)
    for algo, flags in ALGOS.items():
        rho, jpar, npts = run_gpu(cfg, m, flags=flags)
        assert npts == npts_o
        assert_parity(rho, rho_o, "wrapped/%s rho" % algo)
        assert_parity(jpar, jpar_o, "wrapped/%s jpar" % algo)


def test_radial_coordinate_outside_0_1_deposits_at_the_bound():
    """include/orb.h: 's outside [0,1] is treated as the nearest bound' (R11) -- s = -0.2 and 1.2
    must give exactly what s = 0 and s = 1 give (and never write out of bounds)."""
    cfg = small("cfg0", 20_011, current=True, s_lo=0.0, s_hi=1.0)
    m = W.generate(cfg)
    n = cfg.n_markers
    bad = dict(m)
    bad["s"] = m["s"].copy()
    bad["s"][0:n:5] = -0.2
    bad["s"][1:n:5] = 1.2
    bad["s"][2:n:5] = -1e-300
    ref = dict(m)
    ref["s"] = np.clip(bad["s"], 0.0, 1.0)
    rho_o, jpar_o, npts_o = run_oracle(cfg, ref)
    for algo, flags in ALGOS.items():
        rho, jpar, npts = run_gpu(cfg, bad, flags=flags)
        assert npts == npts_o
        assert_parity(rho, rho_o, "clamped s/%s rho" % algo)
        assert_parity(jpar, jpar_o, "clamped s/%s jpar" % algo)


def test_cuda_graph_capture_of_bin_zero_deposit(oracle_results):
    """no host synchronisation and no allocation inside orb_markers_bin /
    orb_grid_zero / orb_deposit -- the three calls are captured into ONE CUDA graph (capture
    fails on any synchronising call), replayed 3 times, and the grids match the oracle."""
    import torch
    for name in ("cfg3_small", "cfg4_small"):
        cfg, m, (rho_o, jpar_o, npts_o) = get_case(name, oracle_results)
        d = to_device(m)
        g = B.grid_for(cfg)
        rho = torch.full(g.shape(), 3.0, dtype=torch.float64, device="cuda")
        jpar = torch.full(g.shape(), -2.0, dtype=torch.float64, device="cuda")
        pol = B.policy_for(cfg)
        g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"])
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            st = torch.cuda.current_stream().cuda_stream
            g.markers_bin(st)
            g.grid_zero(rho, jpar, st)
            g.deposit(rho, jpar, pol, st)
        for _ in range(3):
            rho.fill_(9.0)
            graph.replay()
        torch.cuda.synchronize()
        assert g.last_points() == npts_o
        assert_parity(rho.cpu().numpy(), rho_o, name + " graph rho")
        assert_parity(jpar.cpu().numpy(), jpar_o, name + " graph jpar")
        del graph
        g.destroy()


def test_ring_data_capacity_overflow_is_benign(oracle_results):
    """NEXT-3: Larmor ring data reserved for fewer points than the markers produce -- the points
    beyond the reservation are deposited directly and counted; the grids still match the oracle."""
    import torch
    cfg, m, (rho_o, jpar_o, npts_o) = get_case("cfg4_small", oracle_results)
    d = to_device(m)
    g = B.grid_for(cfg)
    rho = torch.zeros(g.shape(), dtype=torch.float64, device="cuda")
    jpar = torch.zeros_like(rho)
    g.markers_bind(d["s"], d["theta"], d["phi"], d["vpar"], d["mu"], d["w"])
    with pytest.raises(B.OrbError) as e:
        g.deposit(rho, jpar, B.policy_for(cfg, flags=B.ORB_DEPOSIT_ALGO_RING_DATA))
    assert e.value.code == B.ORB_E_STATE            # no orb_ring_reserve yet
    g.ring_reserve(cfg.n_markers, npts_o // 2)
    g.deposit(rho, jpar, B.policy_for(cfg, flags=B.ORB_DEPOSIT_ALGO_RING_DATA),
              torch.cuda.current_stream().cuda_stream)
    assert g.last_points() == npts_o
    assert g.last_fallback_points() == npts_o - npts_o // 2
    g.destroy()
    assert_parity(rho.cpu().numpy(), rho_o)
    assert_parity(jpar.cpu().numpy(), jpar_o)


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
        prepare(g, cfg, flags)
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
