"""GPU parity of the forward-mode derivative of gp_forward and the VJP of gp_inverse (SURVEY.md section
8(f)-2) against the fp64 oracle, plus the duality <v_bar, JVP> = <VJP, tangent> computed on the GPU alone.
Tolerances: fp64 1e-9 relative (max norm), theta_bar 1e-8 per component; fp32 1e-3 (north_star's gradient bar)."""
import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gp():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_11402_b200 as gp
    gp.lib()
    return gp


def run(gp, orc, g, kd, dtype, cid):
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    n = g.n
    dev = lambda a: torch.as_tensor(a, device="cuda").to(tdt)
    xi_h = W.make_noise(cid, n, dtype, "xi")
    dxi_h = W.make_noise(cid + 20, n, dtype, "xi")
    vb_h = W.make_noise(cid, n, dtype, "vbar")
    h_h = W.make_noise(cid + 30, n, dtype, "vbar")
    dsig, dell = 0.3, -0.2 * kd["ell"]
    OK, K = orc.Kernel(**kd), gp.Kernel(**kd)
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype=dtype)
    kw = dict(n0=g.n0, k=g.k, nbr=g.nbr, batch_off=g.batch_off)
    xi = dev(xi_h)
    v = gp.gp_forward(G, K, xi)
    v_h = v.cpu().numpy().astype(np.float64)
    # JVP at the point the GPU produced
    dv = gp.gp_jvp(G, K, xi, v, dev(dxi_h), dsig, dell)
    assert gp.check_errors(G.workspace(gp.GP_OP_VJP)) == 0
    dv_ref = orc.jvp(g.x, OK, xi_h.astype(np.float64), v_h, dxi_h.astype(np.float64), dsig, dell, **kw)
    e_jvp = np.abs(dv.cpu().numpy() - dv_ref).max() / np.abs(dv_ref).max()
    # duality on the GPU alone
    xib, tb = gp.gp_vjp(G, K, xi, v, dev(vb_h))
    lhs = float((dev(vb_h).double() * dv.double()).sum().cpu())
    rhs = float((xib.double() * dev(dxi_h).double()).sum().cpu()) + float(tb[0].cpu()) * dsig + float(tb[1].cpu()) * dell
    e_dual = abs(lhs - rhs) / max(abs(lhs), abs(rhs))
    # inverse VJP at (v, xi_back)
    xi_back = gp.gp_inverse(G, K, v)
    vbi, tbi = gp.gp_inverse_vjp(G, K, v, xi_back, dev(h_h))
    assert gp.check_errors(G.workspace(gp.GP_OP_VJP)) == 0
    vbi_ref, tbi_ref = orc.inverse_vjp(g.x, OK, v_h, xi_back.cpu().numpy().astype(np.float64), h_h.astype(np.float64),
                                       n0=g.n0, k=g.k, nbr=g.nbr)
    e_vb = np.abs(vbi.cpu().numpy() - vbi_ref).max() / np.abs(vbi_ref).max()
    e_tb = np.abs(tbi.cpu().numpy() - tbi_ref) / np.abs(tbi_ref)
    return dict(jvp=e_jvp, dual=e_dual, vbar=e_vb, tb=e_tb)


def graph_for(orc, cid, n, dtype, k=None, n0=None):
    cfg = W.CONFIGS[cid]
    x = W.make_points(cfg, dtype, n).astype(np.float64)
    return orc.build_graph(x, k or cfg.k, n0 if n0 is not None else min(cfg.n0, n))


def kern_of(cfg):
    return dict(kind=cfg.kind, sigma=cfg.sigma, ell=cfg.ell, jitter=cfg.jitter)


def test_config1_fp64(gp, orc):
    cfg = W.CONFIGS[1]
    g = graph_for(orc, 1, cfg.n, "f64")
    e = run(gp, orc, g, kern_of(cfg), "f64", 1)
    assert e["jvp"] <= 1e-9 and e["dual"] <= 1e-9 and e["vbar"] <= 1e-9 and (e["tb"] <= 1e-8).all(), e


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(16, 2, 33, 2500), (5, 3, 5, 700), (8, 3, 40, 3000)])
def test_fp64_shapes(gp, orc, kind, k, d, n0, n):
    x = W.make_points(W.CONFIGS[1], "f64", n)[:, :d].copy()
    g = orc.build_graph(x, k, n0)
    e = run(gp, orc, g, dict(kind=kind, sigma=1.7, ell=0.2, jitter=1e-6), "f64", 1)
    assert e["jvp"] <= 1e-8 and e["dual"] <= 1e-8 and e["vbar"] <= 1e-8 and (e["tb"] <= 1e-7).all(), e


@pytest.mark.parametrize("cid,n", [(2, 32768 + 37), (3, 32768)])
def test_fp32_k16_matern(gp, orc, cid, n):
    cfg = W.CONFIGS[cid]
    g = graph_for(orc, cid, n, "f32")
    e = run(gp, orc, g, kern_of(cfg), "f32", cid)
    assert e["jvp"] <= 1e-3 and e["dual"] <= 1e-3 and e["vbar"] <= 1e-3 and (e["tb"] <= 1e-3).all(), e


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(8, 2, 40, 2600), (16, 3, 64, 4001), (32, 2, 70, 2300), (7, 2, 9, 900)])
def test_fp32_shapes(gp, orc, kind, k, d, n0, n):
    x = W.make_points(W.CONFIGS[1], "f32", n)[:, :d].copy()
    g = orc.build_graph(x.astype(np.float64), k, n0)
    e = run(gp, orc, g, dict(kind=kind, sigma=1.3, ell=0.2, jitter=1e-3), "f32", 1)
    assert e["jvp"] <= 1e-3 and e["dual"] <= 1e-3 and e["vbar"] <= 1e-3 and (e["tb"] <= 1e-3).all(), e
