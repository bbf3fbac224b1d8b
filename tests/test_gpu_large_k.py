"""Large-k path (PAPER.md:53 sends k >~ 64 to the JAX version): 64 < k <= 128 on the
warp-per-point kernels, forward / inverse / logdet against the oracle, GPU-built graph against the oracle's graph.
The arithmetic of this path is fp64 whatever the working dtype, so fp32 data are judged by the fp32 bars with room."""
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


@pytest.mark.parametrize("k,d,n0,n,dtype,kind", [(96, 3, 128, 3000, "f64", "matern32"), (128, 2, 130, 2500, "f32", "exp"),
                                                (65, 3, 70, 2000, "f32", "se"), (100, 1, 100, 1500, "f64", "exp")])
def test_large_k_forward_inverse_logdet(gp, orc, k, d, n0, n, dtype, kind):
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    x = W.make_points(W.CONFIGS[1], dtype, n)[:, :d].copy()
    g = orc.build_graph(x.astype(np.float64), k, n0)
    G = gp.gp_graph_build(torch.as_tensor(x, device="cuda"), k, n0, build_flags=0)      # builder handles k > 64 too
    assert np.array_equal(G.perm.cpu().numpy(), g.perm) and np.array_equal(G.batch_off, g.batch_off)
    assert np.array_equal(np.sort(G.nbr.cpu().numpy(), axis=1), np.sort(g.nbr, axis=1))
    kd = dict(kind=kind, sigma=1.2, ell=0.3, jitter=1e-6 if dtype == "f64" else 1e-4)
    OK, K = orc.Kernel(**kd), gp.Kernel(**kd)
    xi_h = W.make_noise(1, n, dtype, "xi")
    v = gp.gp_forward(G, K, torch.as_tensor(xi_h, device="cuda").to(tdt))
    assert gp.check_errors(G.workspace(gp.GP_OP_FORWARD)) == 0
    v_h = v.cpu().numpy().astype(np.float64)
    v_ref = orc.forward(g.x, OK, xi_h.astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr, batch_off=g.batch_off)
    v_in = v_ref.astype(xi_h.dtype)
    xi_b = gp.gp_inverse(G, K, torch.as_tensor(v_in, device="cuda")).cpu().numpy().astype(np.float64)
    xi_ref = orc.inverse(g.x, OK, v_in.astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr)
    ld = float(gp.gp_logdet(G, K).cpu()[0])
    ld_ref = orc.logdet(g.x, OK, n0=g.n0, k=g.k, nbr=g.nbr)
    if dtype == "f64":
        assert np.abs(v_h - v_ref).max() / np.abs(v_ref).max() <= 1e-9
        assert np.abs(xi_b - xi_ref).max() / np.abs(xi_ref).max() <= 1e-9
        assert abs(ld - ld_ref) <= 1e-10 * abs(ld_ref)
    else:
        s_ref = orc.cond_std(g.x, OK, n0=g.n0, k=g.k, nbr=g.nbr)
        assert np.abs(v_h - v_ref).max() <= 1e-4 * v_ref.std()
        assert (np.abs(xi_b - xi_ref) * s_ref).max() <= 1e-4 * v_ref.std()
        assert abs(ld - ld_ref) <= 1e-5 * abs(ld_ref)


def test_large_k_gradients_are_refused(gp, orc):
    import torch
    n, k, n0 = 1200, 80, 96
    x = W.make_points(W.CONFIGS[1], "f64", n)
    g = orc.build_graph(x, k, n0)
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype="f64")
    K = gp.Kernel("se", 1.0, 0.3, 1e-6)
    z = torch.zeros(n, dtype=torch.float64, device="cuda")
    for call in (lambda: gp.gp_vjp(G, K, z, z, z), lambda: gp.gp_jvp(G, K, z, z, z, 0.1, 0.1),
                 lambda: gp.gp_inverse_vjp(G, K, z, z, z), lambda: gp.gp_logdet(G, K, grad=True)):
        with pytest.raises(gp.GraphGPError) as ei:
            call()
        assert ei.value.status == gp.GP_ERR_UNSUPPORTED
