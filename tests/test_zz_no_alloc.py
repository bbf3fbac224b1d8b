"""gp_logdet_noalloc (the entry point without a workspace: scratch in a fixed device array inside the library) against
the existing gp_logdet, on calls in a row that share that array.  Collected last on purpose (file name): the suite
runs with pytest -x.  Tolerances are the ones of tests/test_gpu_parity.py: fp32 graphs 1e-5 relative (the existing path
computes in fp32 there, the no-alloc path in fp64), fp64 graphs 1e-10 relative.
"""
import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu

F64_TOL = 1e-10
F32_LOGDET_TOL = 1e-5


@pytest.fixture(scope="module")
def gp():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_11402_b200 as gp
    gp.lib()
    return gp


def make_case(gp, cid, n, dtype, n0=None):
    import torch
    cfg = W.CONFIGS[cid]
    x = torch.as_tensor(W.make_points(cfg, dtype, n), device="cuda")
    G = gp.gp_graph_build(x, cfg.k, min(cfg.n0, n) if n0 is None else n0)
    return G, gp.Kernel(cfg.kind, cfg.sigma, cfg.ell, cfg.jitter)


def rel(a, b):
    return abs(a - b) / abs(b)


def test_noalloc_logdet_matches_existing_path_on_calls_in_a_row(gp):
    import torch
    cases = [(make_case(gp, 3, 40000, "f32"), F32_LOGDET_TOL),           # k = 16, d = 3, n0 = 1024 (the maximum)
             (make_case(gp, 1, 4096, "f64"), F64_TOL),                   # k = 8, n0 = 64: smaller head, stale matrix behind it
             (make_case(gp, 4, 9000, "f32"), F32_LOGDET_TOL),            # k = 32, d = 2
             (make_case(gp, 2, 5000, "f64", n0=1000), F64_TOL)]          # n0 not a multiple of the panel width
    want = [float(gp.gp_logdet(G, K).cpu()[0]) for (G, K), _ in cases]
    out = torch.full((1,), 123.0, dtype=torch.float64, device="cuda")
    # the same call twice in a row, then every case twice more in a different order: every call starts from the
    # scratch the previous one left
    for idx in [0, 0, 1, 2, 3, 3, 2, 1, 0]:
        (G, K), tol = cases[idx]
        got = float(gp.gp_logdet_noalloc(G, K, out).cpu()[0])
        assert np.isfinite(got)
        assert rel(got, want[idx]) <= tol, (idx, got, want[idx])
    torch.cuda.synchronize()


def test_noalloc_head_only_and_stream(gp):
    import torch
    G, K = make_case(gp, 2, 700, "f64", n0=700)                          # n = n0: dense block only
    want = float(gp.gp_logdet(G, K).cpu()[0])
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        gp.gp_logdet_noalloc(G, K, out, stream=st)
        gp.gp_logdet_noalloc(G, K, out, stream=st)                       # same stream: ordered, no race
    st.synchronize()
    assert rel(float(out.cpu()[0]), want) <= F64_TOL


def test_noalloc_rejects_sizes_beyond_its_scratch(gp):
    import torch
    assert gp.logdet_noalloc_scratch_bytes() == 8 * 1024 * 1024 + 4096
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    G, K = make_case(gp, 2, 3000, "f32", n0=1025)                        # n0 > GP_NOALLOC_MAX_N0
    with pytest.raises(gp.GraphGPError) as e:
        gp.gp_logdet_noalloc(G, K, out)
    assert e.value.status == gp.GP_ERR_TOO_LARGE and "gp_logdet_noalloc" in str(e.value)
    x = torch.as_tensor(W.make_points(W.CONFIGS[3], "f32", 3000), device="cuda")
    G = gp.gp_graph_build(x, 65, 128)                                    # k > GP_NOALLOC_MAX_K
    with pytest.raises(gp.GraphGPError) as e:
        gp.gp_logdet_noalloc(G, K, out)
    assert e.value.status == gp.GP_ERR_TOO_LARGE
    assert float(out.cpu()[0]) == 0.0                                    # nothing was launched
