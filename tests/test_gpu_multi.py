"""Multi-sample apply (gp_forward_multi / gp_inverse_multi) against the oracle:
sample s of the [n, S] call must equal the oracle's forward / inverse on column s, element by element.
Tolerances: north_star (fp64 1e-10; fp32 max|dv| <= 1e-4 std(v), the inverse in units of v, R-16)."""
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


def noise(cid, n, S, dtype):
    return np.stack([W.make_noise(cid + 10 * s, n, dtype, "xi") for s in range(S)], axis=1).copy()


@pytest.mark.parametrize("cid,n,dtype,S", [(1, 4096, "f64", 1), (1, 4096, "f64", 5), (2, 20011, "f32", 4), (2, 20011, "f32", 16),
                                           (3, 30011, "f32", 3), (3, 30011, "f32", 8)])
def test_multi_equals_oracle_per_sample(gp, orc, cid, n, dtype, S):
    import torch
    cfg = W.CONFIGS[cid]
    x = W.make_points(cfg, dtype, n).astype(np.float64)
    g = orc.build_graph(x, cfg.k, min(cfg.n0, n))
    kd = dict(kind=cfg.kind, sigma=cfg.sigma, ell=cfg.ell, jitter=cfg.jitter)
    OK, K = orc.Kernel(**kd), gp.Kernel(**kd)
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype=dtype)
    xi_h = noise(cid, n, S, dtype)
    v = gp.gp_forward_multi(G, K, torch.as_tensor(xi_h, device="cuda"))
    v_h = v.cpu().numpy().astype(np.float64)
    v_ref = np.stack([orc.forward(g.x, OK, xi_h[:, s].astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr, batch_off=g.batch_off)
                      for s in range(S)], axis=1)
    s_ref = orc.cond_std(g.x, OK, n0=g.n0, k=g.k, nbr=g.nbr)
    v_in = v_ref.astype(xi_h.dtype)
    xi_b = gp.gp_inverse_multi(G, K, torch.as_tensor(v_in, device="cuda")).cpu().numpy().astype(np.float64)
    xi_ref = np.stack([orc.inverse(g.x, OK, v_in[:, s].astype(np.float64), n0=g.n0, k=g.k, nbr=g.nbr) for s in range(S)], axis=1)
    if dtype == "f64":
        assert np.abs(v_h - v_ref).max() / np.abs(v_ref).max() <= 1e-10
        assert np.abs(xi_b - xi_ref).max() / np.abs(xi_ref).max() <= 1e-10
    else:
        for s in range(S):
            assert np.abs(v_h[:, s] - v_ref[:, s]).max() <= 1e-4 * v_ref[:, s].std(), s
            assert (np.abs(xi_b[:, s] - xi_ref[:, s]) * s_ref).max() <= 1e-4 * v_ref[:, s].std(), s
    # and the single-sample calls give the same numbers as column 0 (same weights, same apply order up to rounding)
    v0 = gp.gp_forward(G, K, torch.as_tensor(np.ascontiguousarray(xi_h[:, 0]), device="cuda")).cpu().numpy().astype(np.float64)
    tol = 1e-10 * np.abs(v_ref).max() if dtype == "f64" else 1e-4 * v_ref[:, 0].std()
    assert np.abs(v0 - v_h[:, 0]).max() <= tol


def test_multi_unsupported_shape_and_bad_arguments(gp, orc):
    import torch
    cfg = W.CONFIGS[4]
    x = W.make_points(cfg, "f32", 3000).astype(np.float64)
    g = orc.build_graph(x, 32, 64)
    G = gp.graph_from_arrays(g.x, g.nbr, g.batch_off, g.n0, dtype="f32")
    K = gp.Kernel("exp", 1.0, 0.01, 1e-4)
    xi = torch.zeros((3000, 4), device="cuda")
    with pytest.raises(gp.GraphGPError) as ei:
        gp.gp_forward_multi(G, K, xi)
    assert ei.value.status == gp.GP_ERR_UNSUPPORTED          # k = 32 has no multi-sample kernel
    with pytest.raises(ValueError):
        gp.gp_forward_multi(G, K, xi[:, 0])
