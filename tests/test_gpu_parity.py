"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on the
same seeded inputs.  Graphs come from the oracle here (order + brute-force preceding kNN + depth sort), so
these tests isolate the conditioning kernels; the GPU builder has its own parity tests.

Tolerances (BASELINE.json north_star; definitions DESIGN.md R-16):
  fp64: max|dv| / max|v_ref| <= 1e-10, same for xi; |dlogdet| / |logdet| <= 1e-10
  fp32: max|dv| <= 1e-4 std(v_ref); logdet relative <= 1e-5; the inverse in units of v: max_i s_i |dxi_i| <= 1e-4 std(v_ref)
        (xi_i = (v_i - m_i) / s_i, so s_i dxi_i is the error of m_i + s_i xi_i, the quantity the forward bound is for)
"""
import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu

F64_TOL = 1e-10
F32_V_TOL = 1e-4
F32_LOGDET_TOL = 1e-5


@pytest.fixture(scope="module")
def gp():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_11402_b200 as gp
    gp.lib()
    return gp


_graph_cache = {}


def oracle_graph(orc, cid, n, dtype, k=None, n0=None):
    key = (cid, n, dtype, k, n0)
    if key not in _graph_cache:
        cfg = W.CONFIGS[cid]
        x = W.make_points(cfg, dtype, n).astype(np.float64)       # promoted exactly (O-1)
        g = orc.build_graph(x, k or cfg.k, n0 if n0 is not None else min(cfg.n0, n))
        _graph_cache[key] = g
    return _graph_cache[key]


def to_dev(gp, g, dtype, flags=0):
    return gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype=dtype, flags=flags)


def kern_of(cfg):
    return dict(kind=cfg.kind, sigma=cfg.sigma, ell=cfg.ell, jitter=cfg.jitter)


def run_all(gp, orc, g, kd, dtype, cid, flags=0):
    """forward / inverse / logdet on the GPU and in the oracle; returns the error measures."""
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    n = g.n
    xi_h = W.make_noise(cid, n, dtype, "xi")
    okern = orc.Kernel(**kd)
    v_ref = orc.forward(g.x, okern, xi_h.astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr, batch_off=g.batch_off)
    ld_ref = orc.logdet(g.x, okern, n0=g.n0, k=g.k, nbr=g.nbr)

    G = to_dev(gp, g, dtype, flags)
    K = gp.Kernel(**kd)
    xi = torch.as_tensor(xi_h, device="cuda").to(tdt)
    v = gp.gp_forward(G, K, xi)
    assert gp.check_errors(G.workspace(gp.GP_OP_FORWARD)) == 0
    v_h = v.cpu().numpy().astype(np.float64)

    # inverse of the ORACLE's v rounded to the working dtype, compared with the oracle's inverse of the same
    v_in = v_ref.astype(xi_h.dtype)
    xi_ref = orc.inverse(g.x, okern, v_in.astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr)
    xi_back = gp.gp_inverse(G, K, torch.as_tensor(v_in, device="cuda"))
    assert gp.check_errors(G.workspace(gp.GP_OP_INVERSE)) == 0
    xi_b = xi_back.cpu().numpy().astype(np.float64)

    ld = float(gp.gp_logdet(G, K).cpu()[0])
    assert gp.check_errors(G.workspace(gp.GP_OP_LOGDET)) == 0
    s_ref = orc.cond_std(g.x, okern, n0=g.n0, k=g.k, nbr=g.nbr)
    return dict(
        xi_in_v_units=(np.abs(xi_b - xi_ref) * s_ref).max() / v_ref.std(),
        v_rel_max=np.abs(v_h - v_ref).max() / np.abs(v_ref).max(),
        v_over_std=np.abs(v_h - v_ref).max() / v_ref.std(),
        xi_rel_max=np.abs(xi_b - xi_ref).max() / np.abs(xi_ref).max(),
        xi_abs=np.abs(xi_b - xi_ref).max(),
        ld_rel=abs(ld - ld_ref) / abs(ld_ref),
    )


@pytest.mark.parametrize("flags", [0, 2], ids=["specialised", "generic"])
def test_config1_fp64_full_size(gp, orc, flags):
    """BASELINE config 1 at its full size: N=4096, k=8, SE, fp64, jitter 1e-6."""
    cfg = W.CONFIGS[1]
    g = oracle_graph(orc, 1, cfg.n, "f64")
    e = run_all(gp, orc, g, kern_of(cfg), "f64", 1, flags)
    assert e["v_rel_max"] <= F64_TOL, e
    assert e["xi_rel_max"] <= F64_TOL, e
    assert e["ld_rel"] <= F64_TOL, e


def test_dense_cross_check_n256_all_preceding(gp, orc):
    """BASELINE config 1's cross-check: N=256 with c(i) = all preceding (n0 = N) equals the dense Cholesky
    v = L xi and log det K, computed here by LAPACK through numpy."""
    import torch
    cfg = W.CONFIGS[1]
    n = 256
    x = W.make_points(cfg, "f64", n)
    perm = orc.order(x)
    xt = x[perm]
    r = np.sqrt(((xt[:, None, :] - xt[None, :, :]) ** 2).sum(-1))
    Kd = cfg.sigma ** 2 * (np.exp(-r * r / (2 * cfg.ell ** 2)) + cfg.jitter * np.eye(n))
    L = np.linalg.cholesky(Kd)
    xi = W.make_noise(1, n, "f64")
    G = gp.graph_from_arrays(xt, np.zeros((0, 8), np.int32), np.array([n], np.int64), n, dtype="f64")
    Kn = gp.Kernel(**kern_of(cfg))
    v = gp.gp_forward(G, Kn, torch.as_tensor(xi, device="cuda")).cpu().numpy()
    assert np.abs(v - L @ xi).max() / np.abs(L @ xi).max() <= F64_TOL
    ld = float(gp.gp_logdet(G, Kn).cpu()[0])
    assert abs(ld - 2 * np.log(np.diag(L)).sum()) / abs(ld) <= F64_TOL
    xi_back = gp.gp_inverse(G, Kn, torch.as_tensor(L @ xi, device="cuda")).cpu().numpy()
    assert np.abs(xi_back - xi).max() <= 1e-9


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config2_uniform_matern_k16(gp, orc, dtype):
    """Config 2's shape (k=16, Matern-3/2, n0=1024) at N=32768: several hundred CTAs, ragged last batch."""
    cfg = W.CONFIGS[2]
    n = 32768 + 37
    g = oracle_graph(orc, 2, n, dtype)
    e = run_all(gp, orc, g, kern_of(cfg), dtype, 2)
    if dtype == "f64":
        assert e["v_rel_max"] <= F64_TOL and e["xi_rel_max"] <= F64_TOL and e["ld_rel"] <= F64_TOL, e
    else:
        assert e["v_over_std"] <= F32_V_TOL, e
        assert e["xi_in_v_units"] <= F32_V_TOL, e
        assert e["ld_rel"] <= F32_LOGDET_TOL, e


def test_config3_clustered_fp32(gp, orc):
    cfg = W.CONFIGS[3]
    n = 32768
    g = oracle_graph(orc, 3, n, "f32")
    e = run_all(gp, orc, g, kern_of(cfg), "f32", 3)
    assert e["v_over_std"] <= F32_V_TOL, e
    assert e["xi_in_v_units"] <= F32_V_TOL, e
    assert e["ld_rel"] <= F32_LOGDET_TOL, e


def test_config4_radial2d_k32_exp_fp32(gp, orc):
    cfg = W.CONFIGS[4]
    n = 16384 + 5
    g = oracle_graph(orc, 4, n, "f32")
    e = run_all(gp, orc, g, kern_of(cfg), "f32", 4)
    assert e["v_over_std"] <= F32_V_TOL, e
    assert e["xi_in_v_units"] <= F32_V_TOL, e
    assert e["ld_rel"] <= F32_LOGDET_TOL, e


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(8, 3, 50, 3001), (16, 2, 33, 2500), (5, 3, 5, 700), (1, 1, 1, 300)])
def test_ragged_sizes_all_kernels_fp64(gp, orc, kind, k, d, n0, n):
    """Odd head sizes (n0 not a multiple of the head block), k with and without a register kernel, d = 1..3."""
    rng_cfg = W.CONFIGS[1]
    x = W.make_points(rng_cfg, "f64", n)[:, :d].copy()
    g = orc.build_graph(x, k, n0)
    kd = dict(kind=kind, sigma=1.7, ell=0.2, jitter=1e-6)
    e = run_all(gp, orc, g, kd, "f64", 1)
    assert e["v_rel_max"] <= 1e-9 and e["xi_rel_max"] <= 1e-9 and e["ld_rel"] <= 1e-10, e


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(8, 3, 50, 3001), (8, 2, 40, 2600), (16, 3, 64, 4001), (16, 2, 33, 2500),
                                      (32, 2, 70, 2300), (32, 3, 64, 2100), (5, 3, 5, 700), (7, 2, 9, 900)])
def test_every_fp32_shape_all_kernels(gp, orc, kind, k, d, n0, n):
    """Every fp32 kernel shape the library instantiates - packed one-thread-per-point (k = 8, 16; d = 2, 3), lane
    group (k = 32; d = 2, 3) - and the shared-memory fallback (odd k), each with the three covariance functions,
    dataflow and per-batch forward.  Jitter 1e-3 and ell = 0.2 on uniform points: a well-conditioned fp32 problem."""
    import torch
    x = W.make_points(W.CONFIGS[1], "f32", n)[:, :d].copy()
    g = orc.build_graph(x.astype(np.float64), k, n0)
    kd = dict(kind=kind, sigma=1.3, ell=0.2, jitter=1e-3)
    e = run_all(gp, orc, g, kd, "f32", 1)
    assert e["v_over_std"] <= F32_V_TOL, e
    assert e["ld_rel"] <= F32_LOGDET_TOL, e
    assert e["xi_in_v_units"] <= F32_V_TOL, e
    e2 = run_all(gp, orc, g, kd, "f32", 1, flags=gp.GP_FLAG_PER_BATCH_LAUNCH)
    assert e2["v_over_std"] <= F32_V_TOL, e2


@pytest.mark.parametrize("k,d", [(16, 2), (8, 2), (16, 3)])
def test_fp64_lane_group_and_register_shapes(gp, orc, k, d):
    """fp64: k = 16 runs on the lane-group kernel (d = 2, 3), k = 8 on the one-thread register kernel (d = 2)."""
    n, n0 = 2777, 48
    x = W.make_points(W.CONFIGS[1], "f64", n)[:, :d].copy()
    g = orc.build_graph(x, k, n0)
    kd = dict(kind="matern32", sigma=0.8, ell=0.15, jitter=1e-6)
    e = run_all(gp, orc, g, kd, "f64", 1)
    assert e["v_rel_max"] <= 1e-9 and e["xi_rel_max"] <= 1e-9 and e["ld_rel"] <= 1e-10, e


def test_markov_exponential_1d_on_gpu(gp, orc):
    """P-8 on the GPU: d=1, exponential kernel, sorted points, c(i) = {i-1}, no jitter: Vecchia is exact and
    log det = sum log(1 - exp(-2 dx / ell))."""
    n = 2000
    x = np.cumsum(0.01 + W.uniform(77, 0, 0, n, np.float64))[:, None]
    nbr = np.arange(0, n - 1, dtype=np.int32)[:, None]
    boff = np.arange(1, n + 1, dtype=np.int64)
    G = gp.graph_from_arrays(x, nbr, boff, 1, dtype="f64")
    ell = 0.7
    ld = float(gp.gp_logdet(G, gp.Kernel("exp", 1.0, ell, 0.0)).cpu()[0])
    ref = np.log1p(-np.exp(-2 * np.diff(x[:, 0]) / ell)).sum()
    assert abs(ld - ref) / abs(ref) <= 1e-10


def test_not_positive_definite_is_reported(gp, orc):
    """Duplicate points with zero jitter: the conditional variance is 0 -> counted, NaN written, no crash."""
    import torch
    n, k, n0 = 200, 4, 8
    x = W.make_points(W.CONFIGS[1], "f64", n)
    x[150] = x[10]
    g = orc.build_graph(x, k, n0)
    G = to_dev(gp, g, "f64")
    xi = torch.as_tensor(W.make_noise(1, n, "f64"), device="cuda")
    v = gp.gp_forward(G, gp.Kernel("se", 1.0, 0.1, 0.0), xi)
    nbad = gp.check_errors(G.workspace(gp.GP_OP_FORWARD))
    assert nbad >= 1
    assert int(torch.isnan(v).sum()) >= 1


def test_argument_errors(gp, orc):
    import ctypes as C
    import torch
    g = oracle_graph(orc, 1, 4096, "f64")
    G = to_dev(gp, g, "f64")
    xi = torch.zeros(g.n, dtype=torch.float64, device="cuda")
    with pytest.raises(gp.GraphGPError) as ei:
        gp.gp_forward(G, gp.Kernel("se", -1.0, 0.1, 0.0), xi)
    assert ei.value.status == gp.GP_ERR_INVALID_ARG
    cg, ck = G.c(), gp.Kernel("se", 1.0, 0.1, 1e-6).c()
    st = gp.lib().gp_forward(C.byref(cg), C.byref(ck), xi.data_ptr(), xi.data_ptr(), None, 0, None)
    assert st == gp.GP_ERR_WORKSPACE
    bad = G.batch_off.copy()
    bad[1] = bad[0]
    G2 = gp.Graph(x=G.x, nbr=G.nbr, batch_off=bad, n0=G.n0)
    with pytest.raises(gp.GraphGPError):
        gp.gp_forward(G2, gp.Kernel("se", 1.0, 0.1, 1e-6), xi)


@pytest.mark.parametrize("cid,n,dtype", [(1, 4096, "f64"), (2, 5000, "f32"), (2, 50000, "f32"), (3, 30011, "f32"),
                                         (2, 20011, "f64"), (4, 20000, "f32")])   # the last two: lane-group dataflow
def test_dataflow_forward_equals_per_batch_forward(gp, orc, cid, n, dtype):
    """The single-launch dataflow forward and the literal loop over batches of Alg. 1 apply the
    same weights to the same neighbour values: they agree to rounding (the weights are reached by a different
    substitution order), and both match the oracle."""
    import torch
    cfg = W.CONFIGS[cid]
    g = oracle_graph(orc, cid, n, dtype)
    tdt = torch.float64 if dtype == "f64" else torch.float32
    xi_h = W.make_noise(cid, n, dtype, "xi")
    xi = torch.as_tensor(xi_h, device="cuda").to(tdt)
    K = gp.Kernel(**kern_of(cfg))
    outs = []
    for flags in (0, gp.GP_FLAG_FLOW_CARRY, gp.GP_FLAG_FLOW_WEIGHTS, gp.GP_FLAG_PER_BATCH_LAUNCH):
        G = to_dev(gp, g, dtype, flags)
        for _ in range(3):                       # repeated calls reuse the workspace: pending markers are reset
            v = gp.gp_forward(G, K, xi)
        assert gp.check_errors(G.workspace(gp.GP_OP_FORWARD)) == 0
        outs.append(v.cpu().numpy().astype(np.float64))
    v_ref = orc.forward(g.x, orc.Kernel(**kern_of(cfg)), xi_h.astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr,
                        batch_off=g.batch_off)
    tol = F64_TOL if dtype == "f64" else F32_V_TOL
    scale = np.abs(v_ref).max() if dtype == "f64" else v_ref.std()
    for o in outs:
        assert np.isfinite(o).all()
        assert np.abs(o - outs[-1]).max() / scale <= tol
        assert np.abs(o - v_ref).max() / scale <= tol
