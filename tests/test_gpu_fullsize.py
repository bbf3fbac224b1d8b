"""Parity at BASELINE.json's FULL sizes (configs 3 and 4, N = 2^24), in the launch configuration bench.py times:
GPU-built graph, default flags.  The oracle cannot run 2^24 points end to end in a test, so
  * sampled outputs are checked one by one: for sampled positions i the oracle's Eq. 2 (w, s^2 from
    oracle.condition, fp64) is applied to the SAME neighbour values, which checks v_i (forward) and xi_i (inverse);
  * a PREFIX of the graph order (itself a valid generation graph: every neighbour precedes its point) is run end to
    end through the oracle: forward values and the log-determinant;
  * graph invariants (P-10) hold at full size.
Tolerances: north_star (fp32: max|dv| <= 1e-4 std(v), logdet 1e-5 relative)."""
import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gp():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    if torch.cuda.get_device_properties(0).total_memory < 40 * 2 ** 30:
        pytest.skip("needs a large-memory GPU")
    import paper_2606_11402_b200 as gp
    gp.lib()
    return gp


@pytest.mark.parametrize("cid,prefix", [(3, 1 << 20), (4, 1 << 18)])
def test_full_size_sampled_and_prefix(gp, orc, cid, prefix):
    import torch
    cfg = W.CONFIGS[cid]
    n, k, n0 = cfg.n, cfg.k, cfg.n0
    assert n == 1 << 24
    x = W.make_points(cfg, "f32", n)
    G = gp.gp_graph_build(torch.as_tensor(x, device="cuda"), k, n0)
    del x
    K = gp.Kernel(cfg.kind, cfg.sigma, cfg.ell, cfg.jitter)
    OK = orc.Kernel(cfg.kind, cfg.sigma, cfg.ell, cfg.jitter)
    xi_h = W.make_noise(cid, n, "f32", "xi")
    xi = torch.as_tensor(xi_h, device="cuda")
    v = gp.gp_forward(G, K, xi)
    assert gp.check_errors(G.workspace(gp.GP_OP_FORWARD)) == 0
    xi_back = gp.gp_inverse(G, K, v)
    assert gp.check_errors(G.workspace(gp.GP_OP_INVERSE)) == 0
    v_h = v.cpu().numpy().astype(np.float64)
    xib_h = xi_back.cpu().numpy().astype(np.float64)
    assert np.isfinite(v_h).all()
    std = v_h.std()

    # graph invariants at full size
    nbr = G.nbr.cpu().numpy()
    depth = G.depth.cpu().numpy()
    rows = np.arange(n0, n, dtype=np.int64)
    assert (nbr < rows[:, None]).all()
    assert np.array_equal(depth[n0:], 1 + depth[nbr.astype(np.int64)].max(axis=1))
    assert G.batch_off[0] == n0 and G.batch_off[-1] == n

    # sampled outputs, one by one
    xg = G.x.cpu().numpy().astype(np.float64)
    rng = np.random.default_rng(100 + cid)
    sample = np.sort(rng.choice(np.arange(n0, n), 4096, replace=False))
    worst_v = worst_xi = 0.0
    for i in sample:
        c = nbr[i - n0]
        w, s2 = orc.condition(xg, OK, int(i), c)
        m = float(w @ v_h[c.astype(np.int64)])
        s = np.sqrt(s2)
        worst_v = max(worst_v, abs(v_h[i] - (m + s * float(xi_h[i]))))
        worst_xi = max(worst_xi, abs(xib_h[i] - (v_h[i] - m) / s))
    assert worst_v <= 1e-4 * std, (worst_v, std)
    # xi = (v - m) / s amplifies the rounding of m by 1/s: judged on the same scale as v (R-16)
    assert worst_xi <= 2e-3, worst_xi

    # prefix end to end
    M = prefix
    boff = np.unique(np.minimum(G.batch_off, M))
    v_ref = orc.forward(xg[:M], OK, xi_h[:M].astype(np.float64), n0=n0, k=k, nbr=nbr[:M - n0], batch_off=boff)
    assert np.abs(v_h[:M] - v_ref).max() <= 1e-4 * v_ref.std()
    Gp = gp.Graph(x=G.x[:M].contiguous(), nbr=G.nbr[:M - n0].contiguous(), batch_off=boff, n0=n0)
    ld = float(gp.gp_logdet(Gp, K).cpu()[0])
    ld_ref = orc.logdet(xg[:M], OK, n0=n0, k=k, nbr=nbr[:M - n0])
    assert abs(ld - ld_ref) <= 1e-5 * abs(ld_ref), (ld, ld_ref)
