"""-m gpu: orb_gather (get fields + gyroaverage) through
the C ABI against oracle_gather, element by element on the same seeded inputs, plus the
adjointness with orb_deposit on the GPU results themselves.

Tolerance: per field max|gpu - oracle| <= 1e-12 * max|oracle| (the deposit's bar, R19: both sides
sum the same <= 64 * N_L products per marker in fp64, in different orders).
"""
import dataclasses

import numpy as np
import pytest

import oracle as O
from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import workloads as W

from gpu_util import TOL, oracle_geom, oracle_policy, rel_err, run_gpu, to_device

pytestmark = pytest.mark.gpu

ALGOS = {"tile": 0, "direct": B.ORB_DEPOSIT_NO_BIN}


def small(cfg_name, n, **kw):
    return dataclasses.replace(W.scaled(W.CONFIGS[cfg_name], n), **kw)


CASES = {
    "cfg0": W.CONFIGS["cfg0"],
    "cfg1_small": small("cfg1", 300_007),
    "cfg2_small": small("cfg2", 200_003),
    "cfg3_small": small("cfg3", 250_001),
    "cfg4_small": small("cfg4", 150_011),
    "cfg4s_small": small("cfg4s", 150_011),
    "edge_rings": small("cfg0", 20_011, s_lo=0.0, s_hi=1.0, rho_star=1 / 25.0),
    "odd_grid": small("cfg0", 30_013, ns=23, ntheta=37, nphi=19, s_lo=0.0, s_hi=1.0),
    "tiny_grid": small("cfg0", 5_003, ns=4, ntheta=4, nphi=4, s_lo=0.0, s_hi=1.0),
    "nl1": small("cfg0", 40_009, n_fixed=1),
    "nl7": small("cfg0", 20_011, n_fixed=7),
    "nl32": small("cfg0", 5_003, n_fixed=32, rho_star=1 / 40.0),
}


def fields_for(cfg, nf, seed=3):
    """Seeded synthetic fields on the grid nodes: smooth modes + noise (no method arithmetic)."""
    rng = np.random.default_rng(seed)
    shape = (cfg.ns + 3, cfg.ntheta, cfg.nphi)
    i, j, k = np.meshgrid(*(np.arange(n) for n in shape), indexing="ij", sparse=True)
    out = []
    for f in range(nf):
        smooth = np.cos(2 * np.pi * (f + 1) * j / cfg.ntheta + 0.3 * f) * np.sin(
            2 * np.pi * k / cfg.nphi + 0.1 * i)
        out.append(np.ascontiguousarray(smooth + 0.25 * rng.standard_normal(shape)))
    return out


def gather_gpu(cfg, m, fields, flags=0, bind_flags=0, theta_map=1, alpha0=0.0, graph=False):
    import torch
    d = to_device(m)
    fd = [torch.from_numpy(f).cuda() for f in fields]
    out = [torch.full((cfg.n_markers,), np.nan, dtype=torch.float64, device="cuda") for _ in fields]
    g = B.Grid(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0, rho_star=cfg.rho_star,
               q=cfg.q, theta_map=theta_map)
    try:
        g.markers_bind(d["s"], d["theta"], d["phi"], None, d["mu"], d["w"], flags=bind_flags,
                       n=cfg.n_markers)
        pol = B.policy(cfg.n_fixed, adaptive=cfg.adaptive, n_max=cfg.n_max if cfg.adaptive else None,
                       rho_ref=cfg.rho_ref, alpha0=alpha0, flags=flags)
        st = torch.cuda.current_stream().cuda_stream
        g.gather(fd, out, pol, st)
        npts = g.last_points()
        fallback = g.last_fallback_points()
        torch.cuda.synchronize()
    finally:
        g.destroy()
    return [o.cpu().numpy() for o in out], npts, fallback


def gather_oracle(cfg, m, fields, alpha0=0.0, theta_map=1, workers=None):
    og = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0,
                rho_star=cfg.rho_star, q=cfg.q, theta_map=theta_map)
    op = (O.policy_adaptive(cfg.n_fixed, cfg.n_max, cfg.rho_ref, alpha0) if cfg.adaptive
          else O.policy_fixed(cfg.n_fixed, alpha0))
    outs, npts = [], 0
    for f in fields:
        o, npts = O.gather(og, op, m["s"], m["theta"], m["phi"], m["mu"], f, workers=workers)
        outs.append(o)
    return outs, npts


@pytest.fixture(scope="module")
def oracle_results():
    return {}


def get_case(name, oracle_results):
    if name not in oracle_results:
        cfg = CASES[name]
        m = W.generate(cfg)
        fields = fields_for(cfg, 3)
        oracle_results[name] = (cfg, m, fields, gather_oracle(cfg, m, fields, workers=None))
    return oracle_results[name]


@pytest.mark.parametrize("algo", list(ALGOS))
@pytest.mark.parametrize("name", list(CASES))
def test_gather_parity(name, algo, oracle_results):
    cfg, m, fields, (want, npts_o) = get_case(name, oracle_results)
    bind_flags = B.ORB_MARKERS_SORTED if cfg.order == "sorted" else 0
    got, npts, fallback = gather_gpu(cfg, m, fields, flags=ALGOS[algo], bind_flags=bind_flags)
    assert npts == npts_o
    for f in range(len(fields)):
        assert np.isfinite(got[f]).all(), "every marker must receive a value (bound order)"
        err = rel_err(got[f], want[f])
        assert err <= TOL, "%s/%s field %d: %.3e" % (name, algo, f, err)


@pytest.mark.parametrize("nf", [1, 2, 5, 8])
def test_gather_field_counts(nf, oracle_results):
    """1..ORB_MAX_FIELDS fields in one call (two per launch inside the library)."""
    cfg = CASES["cfg3_small"]
    m = W.generate(cfg)
    fields = fields_for(cfg, nf, seed=nf)
    want, _ = gather_oracle(cfg, m, fields)
    got, _, _ = gather_gpu(cfg, m, fields)
    for f in range(nf):
        assert rel_err(got[f], want[f]) <= TOL


def test_gather_is_the_adjoint_of_deposit_on_the_gpu(oracle_results):
    """sum_n rho[n] F[n] = q sum_p w_p out[p] with rho from orb_deposit and out from orb_gather,
    both computed on the GPU (fixed and adaptive N_L)."""
    for name in ("cfg3_small", "cfg4_small", "edge_rings"):
        cfg, m, fields, _ = get_case(name, oracle_results)
        cfg_c = dataclasses.replace(cfg, current=False)
        rho, _, _ = run_gpu(cfg_c, m)
        got, _, _ = gather_gpu(cfg, m, fields[:1])
        lhs = float((rho * fields[0]).sum())
        rhs = float(cfg.q * (m["w"] * got[0]).sum())
        scale = abs(cfg.q) * np.abs(m["w"]).sum() * np.abs(fields[0]).max()
        assert abs(lhs - rhs) <= 1e-12 * scale


def test_gather_sorted_flag_on_unsorted_markers_and_bound_order(oracle_results):
    """Results come back in BOUND order whatever the binning did; ORB_MARKERS_SORTED on unsorted
    data stays correct (every point then reads the grid directly)."""
    cfg, m, fields, (want, _) = get_case("cfg3_small", oracle_results)
    got, _, fallback = gather_gpu(cfg, m, fields[:2], bind_flags=B.ORB_MARKERS_SORTED)
    for f in range(2):
        assert rel_err(got[f], want[f]) <= TOL
    perm = np.random.default_rng(0).permutation(cfg.n_markers)
    mp = {f: np.ascontiguousarray(m[f][perm]) for f in W.FIELDS}
    got, _, _ = gather_gpu(cfg, mp, fields[:1])
    assert rel_err(got[0], want[0][perm]) <= TOL


def test_gather_nondefault_geometry_gyrophase_theta_map_and_wrapped_angles():
    cfg = small("cfg0", 30_011, ns=20, ntheta=40, nphi=12, r0=1.7, a=0.5, b0=2.5, q=-1.5,
                rho_star=1 / 60.0, adaptive=True, n_fixed=4, n_max=16, s_lo=0.0, s_hi=1.0)
    m = W.generate(cfg)
    n = cfg.n_markers
    m["theta"] = m["theta"] + W.TWO_PI * ((np.arange(n) % 8) - 4)
    m["phi"] = m["phi"] + W.TWO_PI * ((np.arange(n) // 8) % 8 - 3.5)
    m["s"][0:n:17] = 0.0
    m["s"][1:n:17] = 1.0
    fields = fields_for(cfg, 2)
    for theta_map in (1, 0):
        want, npts_o = gather_oracle(cfg, m, fields, alpha0=0.37, theta_map=theta_map)
        for algo, flags in ALGOS.items():
            got, npts, _ = gather_gpu(cfg, m, fields, flags=flags, theta_map=theta_map, alpha0=0.37)
            assert npts == npts_o
            for f in range(2):
                assert rel_err(got[f], want[f]) <= TOL, (theta_map, algo, f)


def test_gather_empty_and_errors():
    import torch
    g = B.Grid(16, 32, 16)
    F = torch.zeros(g.shape(), dtype=torch.float64, device="cuda")
    z = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(B.OrbError) as e:
        g.gather([F], [z], B.policy(4))
    assert e.value.code == B.ORB_E_STATE
    g.markers_bind(z, z, z, None, z, z, n=0)
    g.gather([F], [z], B.policy(4), torch.cuda.current_stream().cuda_stream)
    assert g.last_points() == 0
    g.markers_bind(z, z, z, None, z, z)
    with pytest.raises(B.OrbError) as e:
        g.gather([F] * 9, [z] * 9, B.policy(4))
    assert e.value.code == B.ORB_E_INVAL
    with pytest.raises(B.OrbError) as e:
        g.gather([None], [z], B.policy(4))
    assert e.value.code == B.ORB_E_INVAL
    g.destroy()


def test_gather_cuda_graph_capture(oracle_results):
    """No host synchronisation / allocation inside orb_markers_bin + orb_gather (graph capture)."""
    import torch
    cfg, m, fields, (want, npts_o) = get_case("cfg4_small", oracle_results)
    d = to_device(m)
    fd = [torch.from_numpy(f).cuda() for f in fields[:2]]
    out = [torch.zeros(cfg.n_markers, dtype=torch.float64, device="cuda") for _ in range(2)]
    g = B.grid_for(cfg)
    g.markers_bind(d["s"], d["theta"], d["phi"], None, d["mu"], d["w"])
    pol = B.policy_for(cfg)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        st = torch.cuda.current_stream().cuda_stream
        g.markers_bin(st)
        g.gather(fd, out, pol, st)
    for _ in range(2):
        for o in out:
            o.fill_(np.nan)
        graph.replay()
    torch.cuda.synchronize()
    assert g.last_points() == npts_o
    for f in range(2):
        assert rel_err(out[f].cpu().numpy(), want[f]) <= TOL
    del graph
    g.destroy()
