"""GPU graph builder (gp_graph_build) against the oracle: tree order, preceding-kNN sets, depths and batches
are integer work, so everything is compared bit-exactly (neighbours as sets, ties by index; north_star)."""
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


def build_gpu(gp, x, k, n0, flags):
    import torch
    return gp.gp_graph_build(torch.as_tensor(x, device="cuda"), k, n0, build_flags=flags)


def as_user_sets(perm, nbr, n0):
    """row (as user id of the point) -> sorted user ids of its neighbours"""
    users = perm[n0:]
    sets = np.sort(perm[nbr.astype(np.int64)], axis=1)
    order = np.argsort(users)
    return users[order], sets[order]


@pytest.mark.parametrize("cid,n,dtype", [(1, 4096, "f64"), (2, 20000, "f32"), (3, 30011, "f32"), (4, 9000, "f32"),
                                         (5, 16384, "f32"), (1, 65, "f64"), (1, 64, "f64")])
def test_builder_matches_oracle_exactly_in_tree_order(gp, orc, cid, n, dtype):
    """Without the spatial flag the graph order is the oracle's: tree order stably sorted by depth."""
    cfg = W.CONFIGS[cid]
    n0 = min(cfg.n0, n)
    x = W.make_points(cfg, dtype, n)
    ref = orc.build_graph(x.astype(np.float64), cfg.k, n0)
    G = build_gpu(gp, x, cfg.k, n0, 0)
    assert np.array_equal(G.perm.cpu().numpy(), ref.perm)
    assert np.array_equal(G.depth.cpu().numpy(), ref.depth)
    assert np.array_equal(G.batch_off, ref.batch_off)
    assert np.array_equal(G.x.cpu().numpy().astype(np.float64), ref.x)
    assert np.array_equal(np.sort(G.nbr.cpu().numpy(), axis=1), np.sort(ref.nbr, axis=1))


@pytest.mark.parametrize("cid,n,dtype", [(2, 20000, "f32"), (3, 30011, "f32"), (4, 9000, "f32")])
def test_builder_spatial_batches_same_graph_different_inner_order(gp, orc, cid, n, dtype):
    """With GP_BUILD_SPATIAL_BATCHES only the order INSIDE a batch changes (any is legal)."""
    cfg = W.CONFIGS[cid]
    n0 = min(cfg.n0, n)
    x = W.make_points(cfg, dtype, n)
    ref = orc.build_graph(x.astype(np.float64), cfg.k, n0)
    G = build_gpu(gp, x, cfg.k, n0, gp.GP_BUILD_SPATIAL_BATCHES)
    perm = G.perm.cpu().numpy()
    assert np.array_equal(perm[:n0], ref.perm[:n0])
    assert np.array_equal(np.sort(perm), np.arange(n))
    assert np.array_equal(G.batch_off, ref.batch_off)
    assert np.array_equal(G.depth.cpu().numpy(), ref.depth)           # depth is sorted: equal as arrays
    assert np.array_equal(G.x.cpu().numpy(), x[perm])
    u1, s1 = as_user_sets(perm, G.nbr.cpu().numpy(), n0)
    u2, s2 = as_user_sets(ref.perm, ref.nbr, n0)
    assert np.array_equal(u1, u2) and np.array_equal(s1, s2)
    nbr = G.nbr.cpu().numpy()
    rows = np.arange(n0, n)
    assert (nbr < rows[:, None]).all()
    # every neighbour lies in an EARLIER batch
    bstart = G.batch_off[np.searchsorted(G.batch_off, rows, side="right") - 1]
    assert (nbr < bstart[:, None]).all()


def test_builder_ties_duplicate_coordinates(gp, orc):
    """Many equal coordinates (grid points, duplicates): order ties by user id, kNN ties by tree index."""
    n, k, n0 = 6000, 8, 64
    g = np.stack(np.meshgrid(np.arange(20), np.arange(20), np.arange(15), indexing="ij"), -1).reshape(-1, 3)
    x = (g[:n].astype(np.float32) * 0.05).astype(np.float32)
    x[100:200] = x[0:100]                                   # exact duplicates
    ref = orc.build_graph(x.astype(np.float64), k, n0)
    G = build_gpu(gp, x, k, n0, 0)
    assert np.array_equal(G.perm.cpu().numpy(), ref.perm)
    assert np.array_equal(np.sort(G.nbr.cpu().numpy(), axis=1), np.sort(ref.nbr, axis=1))
    assert np.array_equal(G.batch_off, ref.batch_off)


def test_builder_large_sampled_rows(gp, orc):
    """N = 2^20: full order equality, sampled rows against brute force, graph invariants (P-10)."""
    cfg = W.CONFIGS[3]
    n, n0, k = 1 << 20, 1024, 16
    x = W.make_points(cfg, "f32", n)
    G = build_gpu(gp, x, k, n0, gp.GP_BUILD_SPATIAL_BATCHES)
    perm = G.perm.cpu().numpy()
    perm_tree = orc.order(x.astype(np.float64))
    tree_of_user = np.empty(n, np.int64)
    tree_of_user[perm_tree] = np.arange(n)
    assert np.array_equal(perm[:n0], perm_tree[:n0])
    assert np.array_equal(np.sort(perm), np.arange(n))
    x_tree = x[perm_tree].astype(np.float64)
    rng = np.random.default_rng(5)
    pos = np.sort(rng.choice(np.arange(n0, n), 2048, replace=False))
    nbr = G.nbr.cpu().numpy()
    got = np.sort(tree_of_user[perm[nbr[pos - n0].astype(np.int64)]], axis=1)
    want = np.sort(orc.knn_rows(x_tree, k, tree_of_user[perm[pos]]), axis=1)
    assert np.array_equal(got, want)
    depth = G.depth.cpu().numpy()
    assert (depth[:n0] == 0).all()
    assert np.array_equal(depth[n0:], 1 + depth[nbr.astype(np.int64)].max(axis=1))
    assert (np.diff(depth) >= 0).all()
    assert G.batch_off[0] == n0 and G.batch_off[-1] == n
    assert np.array_equal(np.flatnonzero(np.diff(depth[n0:])) + n0 + 1, G.batch_off[1:-1])
    assert (np.sort(nbr, axis=1)[:, 1:] != np.sort(nbr, axis=1)[:, :-1]).all()


@pytest.mark.parametrize("n,d,k,dtype", [(20000, 3, 16, "f32"), (20000, 2, 32, "f32"), (9000, 1, 5, "f64"),
                                         (12000, 3, 64, "f32"), (7000, 2, 3, "f64"), (30000, 3, 100, "f32"),
                                         (5000, 4, 6, "f32"), (65537, 3, 8, "f64"), (131, 2, 4, "f32")])
def test_builder_fast_and_plain_stages_agree_row_for_row(gp, orc, n, d, k, dtype):
    """Default stages (presorted lists split by one stable partition per level; shared-memory kNN walk) against the
    plain ones (GP_BUILD_PLAIN_ORDER: a radix sort per level; GP_BUILD_PLAIN_KNN: local-memory walk): same tree order,
    same rows in the same (nearest first, ties by tree index) order, same depths - and that is the oracle's graph."""
    rng = np.random.default_rng(1000 + k)
    x = rng.standard_normal((n, d)).astype(np.float32 if dtype == "f32" else np.float64)
    x[50:90] = x[10:50]                                       # exact duplicates: ties in d^2 and in every coordinate
    x[:, 0] = np.round(x[:, 0] * 8) / 8                       # many equal coordinates in the first split dimension
    n0 = 128 if n > 128 else 64
    fast = build_gpu(gp, x, k, n0, 0)
    for flags in (gp.GP_BUILD_PLAIN_KNN, gp.GP_BUILD_PLAIN_ORDER, gp.GP_BUILD_PLAIN_KNN | gp.GP_BUILD_PLAIN_ORDER):
        plain = build_gpu(gp, x, k, n0, flags)
        assert np.array_equal(fast.perm.cpu().numpy(), plain.perm.cpu().numpy())
        assert np.array_equal(fast.nbr.cpu().numpy(), plain.nbr.cpu().numpy())
        assert np.array_equal(fast.depth.cpu().numpy(), plain.depth.cpu().numpy())
        assert np.array_equal(fast.batch_off, plain.batch_off)
    if k <= 64 and n <= 30000:
        ref = orc.build_graph(x.astype(np.float64), k, n0)
        assert np.array_equal(fast.perm.cpu().numpy(), ref.perm)
        assert np.array_equal(fast.nbr.cpu().numpy(), ref.nbr)
