"""GPU parity of the kernel-parameter derivatives: gp_vjp and the gradient
of gp_logdet through the C ABI against the fp64 oracle, plus a finite-difference check that uses the GPU forward
only (so it does not depend on the oracle at all).

Tolerances (BASELINE.json north_star; definitions DESIGN.md R-16):
  fp64: xi_bar max|d| / max|ref| <= 1e-9, theta_bar per component <= 1e-8 relative (atomics reorder the sums)
  fp32: theta_bar per component <= 1e-3 relative, xi_bar max|d| / max|ref| <= 1e-3
"""
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


def run_vjp(gp, orc, g, kd, dtype, cid, flags=0):
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    n = g.n
    xi_h = W.make_noise(cid, n, dtype, "xi")
    vb_h = W.make_noise(cid, n, dtype, "vbar")
    okern = orc.Kernel(**kd)
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype=dtype, flags=flags)
    K = gp.Kernel(**kd)
    xi = torch.as_tensor(xi_h, device="cuda").to(tdt)
    v = gp.gp_forward(G, K, xi)
    v_h = v.cpu().numpy().astype(np.float64)
    # the oracle differentiates at the same point (xi, v): v as the GPU produced it
    xib_ref, tb_ref = orc.vjp(g.x, okern, xi_h.astype(np.float64), v_h, vb_h.astype(np.float64), n0=g.n0, k=g.k,
                              nbr=g.nbr, batch_off=g.batch_off)
    xib, tb = gp.gp_vjp(G, K, xi, v, torch.as_tensor(vb_h, device="cuda").to(tdt))
    assert gp.check_errors(G.workspace(gp.GP_OP_VJP)) == 0
    xib = xib.cpu().numpy().astype(np.float64)
    tb = tb.cpu().numpy()
    ld_ref, gld_ref = orc.logdet(g.x, okern, n0=g.n0, k=g.k, nbr=g.nbr, grad=True)
    ld, gld = gp.gp_logdet(G, K, grad=True)
    return dict(xib=np.abs(xib - xib_ref).max() / np.abs(xib_ref).max(),
                tb=np.abs(tb - tb_ref) / np.abs(tb_ref),
                ld=abs(float(ld.cpu()[0]) - ld_ref) / abs(ld_ref),
                gld=np.abs(gld.cpu().numpy() - gld_ref) / np.abs(gld_ref))


def graph_for(orc, cid, n, dtype, k=None, n0=None):
    cfg = W.CONFIGS[cid]
    x = W.make_points(cfg, dtype, n).astype(np.float64)
    return orc.build_graph(x, k or cfg.k, n0 if n0 is not None else min(cfg.n0, n))


def kern_of(cfg):
    return dict(kind=cfg.kind, sigma=cfg.sigma, ell=cfg.ell, jitter=cfg.jitter)


def test_config1_fp64_vjp_and_logdet_grad(gp, orc):
    cfg = W.CONFIGS[1]
    g = graph_for(orc, 1, cfg.n, "f64")
    e = run_vjp(gp, orc, g, kern_of(cfg), "f64", 1)
    assert e["xib"] <= 1e-9 and (e["tb"] <= 1e-8).all() and e["ld"] <= 1e-10 and (e["gld"] <= 1e-8).all(), e


def test_dense_head_only_vjp_fp64(gp, orc):
    """n0 = N = 256 (c(i) = all preceding): the whole VJP runs through the dense head."""
    cfg = W.CONFIGS[1]
    g = graph_for(orc, 1, 256, "f64", n0=256)
    for kind in ("se", "matern32", "exp"):
        kd = dict(kind=kind, sigma=1.3, ell=0.15, jitter=1e-6)
        e = run_vjp(gp, orc, g, kd, "f64", 1)
        assert e["xib"] <= 1e-9 and (e["tb"] <= 1e-8).all() and (e["gld"] <= 1e-8).all(), (kind, e)


@pytest.mark.parametrize("cid,n", [(2, 32768 + 37), (3, 32768)])
def test_fp32_k16_matern_vjp(gp, orc, cid, n):
    cfg = W.CONFIGS[cid]
    g = graph_for(orc, cid, n, "f32")
    e = run_vjp(gp, orc, g, kern_of(cfg), "f32", cid)
    assert e["xib"] <= 1e-3 and (e["tb"] <= 1e-3).all() and (e["gld"] <= 1e-3).all(), e


@pytest.mark.parametrize("flags", [0, 2], ids=["specialised", "generic"])
@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
def test_fp32_k8_all_kernels_vjp(gp, orc, kind, flags):
    g = graph_for(orc, 1, 6000, "f32", k=8, n0=64)
    kd = dict(kind=kind, sigma=0.8, ell=0.12, jitter=1e-4)
    e = run_vjp(gp, orc, g, kd, "f32", 1, flags)
    assert e["xib"] <= 1e-3 and (e["tb"] <= 1e-3).all() and (e["gld"] <= 1e-3).all(), e


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(16, 2, 33, 2500), (5, 3, 5, 700), (1, 1, 1, 300)])
def test_ragged_sizes_fp64_vjp(gp, orc, kind, k, d, n0, n):
    x = W.make_points(W.CONFIGS[1], "f64", n)[:, :d].copy()
    g = orc.build_graph(x, k, n0)
    kd = dict(kind=kind, sigma=1.7, ell=0.2, jitter=1e-6)
    e = run_vjp(gp, orc, g, kd, "f64", 1)
    assert e["xib"] <= 1e-8 and (e["tb"] <= 1e-7).all() and (e["gld"] <= 1e-8).all(), e


def test_vjp_matches_finite_differences_of_the_gpu_forward(gp, orc):
    """Independent of the oracle's derivative code: theta_bar = d/dtheta <v_bar, forward(xi; theta)> by central
    differences of the GPU forward (fp64), and xi_bar . dxi = <v_bar, forward(xi + dxi) - forward(xi - dxi)> / 2."""
    import torch
    cfg = W.CONFIGS[1]
    g = graph_for(orc, 1, 3000, "f64")
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype="f64")
    n = g.n
    xi = torch.as_tensor(W.make_noise(1, n, "f64", "xi"), device="cuda")
    vb = torch.as_tensor(W.make_noise(1, n, "f64", "vbar"), device="cuda")
    sig, ell, jit = 1.1, 0.1, 1e-6

    def F(s, l, x):
        return float((vb * gp.gp_forward(G, gp.Kernel("matern32", s, l, jit), x)).sum().cpu())

    K = gp.Kernel("matern32", sig, ell, jit)
    v = gp.gp_forward(G, K, xi)
    xib, tb = gp.gp_vjp(G, K, xi, v, vb)
    tb = tb.cpu().numpy()
    h = 1e-6
    fd_s = (F(sig * (1 + h), ell, xi) - F(sig * (1 - h), ell, xi)) / (2 * h * sig)
    fd_l = (F(sig, ell * (1 + h), xi) - F(sig, ell * (1 - h), xi)) / (2 * h * ell)
    assert abs(tb[0] - fd_s) <= 1e-6 * abs(fd_s)
    assert abs(tb[1] - fd_l) <= 1e-6 * abs(fd_l)
    dxi = torch.as_tensor(W.make_noise(7, n, "f64", "xi"), device="cuda")
    lin = (F(sig, ell, xi + dxi) - F(sig, ell, xi - dxi)) / 2          # forward is linear in xi
    assert abs(float((xib * dxi).sum().cpu()) - lin) <= 1e-9 * abs(lin)


def test_host_variants_match_device_variants(gp, orc):
    """gp_forward_host / gp_inverse_host / gp_vjp_host (pinned host buffers) give the device calls' results."""
    import torch
    cfg = W.CONFIGS[2]
    n = 20000
    g = graph_for(orc, 2, n, "f32")
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype="f32")
    K = gp.Kernel(**kern_of(cfg))
    xi_p = torch.as_tensor(W.make_noise(2, n, "f32", "xi")).pin_memory()
    vb_p = torch.as_tensor(W.make_noise(2, n, "f32", "vbar")).pin_memory()
    v_p, xi2_p, xib_p = (torch.empty_like(xi_p).pin_memory() for _ in range(3))
    tb_p = torch.empty(2, dtype=torch.float64).pin_memory()
    dev = [torch.empty(n, dtype=torch.float32, device="cuda") for _ in range(4)]
    tb_d = torch.empty(2, dtype=torch.float64, device="cuda")
    gp.gp_forward_host(G, K, xi_p, v_p, dev[0], dev[1])
    gp.gp_inverse_host(G, K, v_p, xi2_p, dev[0], dev[1])
    gp.gp_vjp_host(G, K, xi_p, v_p, vb_p, xib_p, tb_p, (dev[0], dev[1], dev[2], dev[3], tb_d))
    torch.cuda.synchronize()
    v = gp.gp_forward(G, K, xi_p.cuda())
    assert torch.equal(v.cpu(), v_p)
    assert torch.equal(gp.gp_inverse(G, K, v).cpu(), xi2_p)
    xib, tb = gp.gp_vjp(G, K, xi_p.cuda(), v, vb_p.cuda())
    assert np.abs(xib.cpu().numpy() - xib_p.numpy()).max() <= 1e-5 * np.abs(xib_p.numpy()).max()
    assert np.allclose(tb.cpu().numpy(), tb_p.numpy(), rtol=1e-6)


@pytest.mark.parametrize("kind", ["se", "matern32", "exp"])
@pytest.mark.parametrize("k,d,n0,n", [(8, 2, 40, 2600), (16, 2, 33, 2500), (16, 3, 64, 4001), (32, 2, 70, 2300), (7, 2, 9, 900)])
def test_every_fp32_shape_vjp(gp, orc, kind, k, d, n0, n):
    """fp32 VJP and log-determinant gradient on every shape: packed two-phase kernels (k = 8, 16; d = 2, 3), and the
    shared-memory gradient kernel for the shapes without one (k = 32, odd k); dataflow and per-batch variants."""
    x = W.make_points(W.CONFIGS[1], "f32", n)[:, :d].copy()
    g = orc.build_graph(x.astype(np.float64), k, n0)
    kd = dict(kind=kind, sigma=1.3, ell=0.2, jitter=1e-3)
    for flags in (0, 1):
        e = run_vjp(gp, orc, g, kd, "f32", 1, flags)
        assert e["xib"] <= 1e-3 and (e["tb"] <= 1e-3).all() and (e["gld"] <= 1e-3).all(), (flags, e)
