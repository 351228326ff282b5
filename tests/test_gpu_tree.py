"""GPU parity for the stage II consumer (single-linkage guide tree) against
oracle/slink_oracle.py.  Similarity ties make the tree non-unique: what is unique (the sorted merge
similarities, the partitions at thresholds between tie values) is compared exactly, and the rest is
checked for validity (a spanning tree whose edge weights are the true similarities)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def feed(F, tri, k, block):
    """Stream packed-triangular similarities `tri` (float32, k leaves) into a tree in row blocks."""
    import torch
    t = F.famsa_tree_create(k)
    for i0 in range(0, k, block):
        i1 = min(i0 + block, k)
        a, b = F.famsa_rows_pairs(0, i0), F.famsa_rows_pairs(0, i1)
        blk = torch.from_numpy(tri[a:b].copy()).cuda() if b > a else torch.zeros(1, dtype=torch.float32, device="cuda")
        F.famsa_tree_update(t, i0, i1, blk)
    return t


def kruskal_weights(tri, k):
    ii, jj = np.tril_indices(k, -1)
    order = np.argsort(-tri.astype(np.float64), kind="stable")
    parent = np.arange(k)
    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]; x = parent[x]
        return x
    w = []
    for e in order:
        ra, rb = find(ii[e]), find(jj[e])
        if ra != rb:
            parent[ra] = rb; w.append(tri[e])
            if len(w) == k - 1:
                break
    return np.array(w, dtype=np.float32)


def check_tree(a, b, w, tri, k):
    assert a.size == b.size == w.size == k - 1
    assert np.all(a > b) and np.all(a < k) and np.all(b >= 0)
    assert np.array_equal(w, tri[a * (a - 1) // 2 + b])          # each edge carries its true similarity
    parent = np.arange(k)
    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]; x = parent[x]
        return x
    for x, y in zip(a, b):
        rx, ry = find(x), find(y)
        assert rx != ry                                          # no cycle: k-1 acyclic edges span
        parent[rx] = ry


@pytest.mark.parametrize("levels", [None, 6, 1])
def test_random_matrices_vs_oracle(F, levels):
    from oracle import slink_oracle as so
    rng = np.random.default_rng(3)
    for k in (2, 3, 17, 70, 140):
        n = k * (k - 1) // 2
        tri = (rng.random(n) if levels is None else rng.integers(1, levels + 1, n) / 4.0).astype(np.float32)
        if levels == 6:
            tri[rng.integers(0, n, 2)] = np.inf                  # identical sequences (R12)
        ref = so.single_linkage(so.full_matrix(k, tri.astype(np.float64)))
        heights = so.merge_heights(ref)
        for block in (1, 3, 64, k):
            with feed(F, tri, k, block) as t:
                a, b, w = F.famsa_tree_edges(t)
                check_tree(a, b, w, tri, k)
                assert np.array_equal(np.sort(w.astype(np.float64))[::-1], heights)
                ia, ib, mw, size = F.famsa_tree_finish(t)
            assert np.array_equal(mw.astype(np.float64), heights)                 # descending merge similarities
            assert size[-1] == k and np.all(ia < ib)
            assert sorted(np.concatenate([ia, ib]).tolist()) == list(range(2 * k - 2))   # every cluster merged once
            merges = list(zip(ia.tolist(), ib.tolist(), mw.astype(np.float64).tolist(), size.tolist()))
            vals = np.unique(heights)
            for thr in list((vals[:-1] + vals[1:]) / 2)[:: max(1, len(vals) // 5)] + [-1.0]:
                if not np.isfinite(thr):
                    continue
                la, lb = so.cut(merges, k, thr), so.cut(ref, k, thr)
                assert np.array_equal(la, lb)                    # same partition at a threshold between tie values


def test_larger_vs_kruskal_and_block_independence(F):
    rng = np.random.default_rng(8)
    k = 2500
    tri = (rng.integers(1, 4000, k * (k - 1) // 2) / 64.0).astype(np.float32)    # many ties
    ref = np.sort(kruskal_weights(tri, k))[::-1]
    for block in (1024, 700, 2500):
        with feed(F, tri, k, block) as t:
            a, b, w = F.famsa_tree_edges(t)
            check_tree(a, b, w, tri, k)
            assert np.array_equal(np.sort(w)[::-1], ref)
            _, _, mw, size = F.famsa_tree_finish(t)
            assert np.array_equal(mw, ref) and size[-1] == k


def test_guide_tree_end_to_end(F, oracle):
    """Stages I + II fused on the device (famsa_guide_tree) against LCS oracle -> single-linkage oracle."""
    from oracle import slink_oracle as so
    from paper_1603_06958_b200 import synth
    for cfg, k, block in ((0, 150, 64), (2, 90, 1024), (1, 200, 7)):
        seqs, offsets = synth.family(cfg, k=k, seed=21)
        _, sref = oracle.rows(seqs, offsets, 0, k)
        ref = so.single_linkage(so.full_matrix(k, sref))
        heights = so.merge_heights(ref)
        with F.famsa_pack(seqs, offsets) as ctx:
            ia, ib, mw, size = F.famsa_guide_tree(ctx, block)
        mw = mw.astype(np.float64)
        inf = np.isinf(heights)
        assert np.array_equal(np.isinf(mw), inf)
        assert np.all(np.abs(mw[~inf] - heights[~inf]) <= 1e-6 * heights[~inf])
        assert size[-1] == k and np.all(np.diff(mw[~inf]) <= 0)


def test_guide_tree_tiny_sets(F, oracle):
    """famsa_guide_tree at the smallest sizes and block shapes (k = 2, 3, 5, 33; blocks of 1, 2, 1024 rows)."""
    from oracle import slink_oracle as so
    from paper_1603_06958_b200 import synth
    for k in (2, 3, 5, 33):
        seqs, offsets = synth.family(0, k=k, seed=300 + k)
        _, sref = oracle.rows(seqs, offsets, 0, k)
        heights = so.merge_heights(so.single_linkage(so.full_matrix(k, sref)))
        for block in (1, 2, 1024):
            with F.famsa_pack(seqs, offsets) as ctx:
                ia, ib, mw, size = F.famsa_guide_tree(ctx, block)
            mw = mw.astype(np.float64)
            inf = np.isinf(heights)
            assert mw.size == k - 1 and size[-1] == k and np.array_equal(np.isinf(mw), inf)
            assert np.all(np.abs(mw[~inf] - heights[~inf]) <= 1e-6 * heights[~inf])
            assert sorted(np.concatenate([ia, ib]).tolist()) == list(range(2 * k - 2))


def feed_blocks(F, tri, k, blocks):
    import torch
    t = F.famsa_tree_create(k)
    for i0, i1 in blocks:
        a, b = F.famsa_rows_pairs(0, i0), F.famsa_rows_pairs(0, i1)
        blk = torch.from_numpy(tri[a:b].copy()).cuda() if b > a else torch.zeros(1, dtype=torch.float32, device="cuda")
        F.famsa_tree_update(t, i0, i1, blk)
    return t


def test_any_order_and_rank_forests_merge(F):
    """Row blocks in any order give the same tree weights; the forests of two 'ranks' that each consumed
    every other block (the multi-GPU deal of bench.py), merged as edges, give the tree of the whole matrix."""
    rng = np.random.default_rng(12)
    k, block = 1500, 128
    tri = (rng.integers(1, 3000, k * (k - 1) // 2) / 32.0).astype(np.float32)
    ref = np.sort(kruskal_weights(tri, k))[::-1]
    blocks = [(a, min(a + block, k)) for a in range(0, k, block)]
    for order in (blocks[::-1], [blocks[i] for i in rng.permutation(len(blocks))]):
        with feed_blocks(F, tri, k, order) as t:
            a, b, w = F.famsa_tree_edges(t)
            check_tree(a, b, w, tri, k)
            assert np.array_equal(np.sort(w)[::-1], ref)
    forests = []
    for rank in range(2):
        with feed_blocks(F, tri, k, blocks[rank::2]) as t:
            assert F.famsa_tree_edge_count(t) <= k - 1
            forests.append(F.famsa_tree_edges(t))
            if rank == 1 and blocks[-1] not in blocks[rank::2]:
                with pytest.raises(F.FamsaError):
                    F.famsa_tree_finish(t)                       # this rank alone has not seen every row
    with feed_blocks(F, tri, k, []) as t:
        for a, b, w in forests:
            F.famsa_tree_merge_edges(t, a, b, w)
        a, b, w = F.famsa_tree_edges(t)
        check_tree(a, b, w, tri, k)
        assert np.array_equal(np.sort(w)[::-1], ref)
        _, _, mw, size = F.famsa_tree_finish(t)
        assert np.array_equal(mw, ref) and size[-1] == k
    # merging edges into a tree that also consumes dense blocks afterwards
    with feed_blocks(F, tri, k, []) as t:
        F.famsa_tree_merge_edges(t, *forests[0])
        for i0, i1 in blocks[1::2]:
            a0, b0 = F.famsa_rows_pairs(0, i0), F.famsa_rows_pairs(0, i1)
            import torch
            F.famsa_tree_update(t, i0, i1, torch.from_numpy(tri[a0:b0].copy()).cuda())
        _, _, w = F.famsa_tree_edges(t)
        assert np.array_equal(np.sort(w)[::-1], ref)


def test_tree_errors(F):
    import torch
    t = F.famsa_tree_create(5)
    buf = torch.ones(32, dtype=torch.float32, device="cuda")
    for i0, i1 in ((3, 2), (0, 6), (-1, 2)):
        with pytest.raises(F.FamsaError) as e:
            F.famsa_tree_update(t, i0, i1, buf)
        assert e.value.code == F.FAMSA_ERANGE
    F.famsa_tree_update(t, 3, 5, buf)                            # any order is legal ...
    assert F.famsa_tree_edge_count(t) == 4
    with pytest.raises(F.FamsaError) as e:
        F.famsa_tree_finish(t)                                   # ... but not every row has been consumed
    assert e.value.code == F.FAMSA_ERANGE
    F.famsa_tree_update(t, 0, 3, buf)
    _, _, w, size = F.famsa_tree_finish(t)
    assert np.all(w == 1.0) and size[-1] == 5
    with pytest.raises(F.FamsaError) as e:
        F.famsa_tree_merge_edges(t, [7], [0], [1.0])             # leaf out of range
    assert e.value.code == F.FAMSA_ERANGE
    t.free()
    for k in (0, 1):
        t = F.famsa_tree_create(k)
        if k:
            F.famsa_tree_update(t, 0, 1, None)
        assert F.famsa_tree_finish(t)[0].size == 0
        t.free()


def test_guide_forest_parts_merge_to_the_guide_tree(F):
    """The multi-GPU deal on one device: forests of parts 0/3, 1/3, 2/3 of the row blocks, merged, equal
    the single-pass guide tree (sorted merge similarities; sizes)."""
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(1, k=700, seed=33)
    with F.famsa_pack(seqs, offsets) as ctx:
        ia, ib, mw, size = F.famsa_guide_tree(ctx, 64)
        forests = [F.famsa_guide_forest(ctx, 64, part, 3) for part in range(3)]
        root = forests[0]
        for other in forests[1:]:
            F.famsa_tree_merge_edges(root, *F.famsa_tree_edges(other))
        ia2, ib2, mw2, size2 = F.famsa_tree_finish(root)
        for t in forests:
            t.free()
    assert np.array_equal(mw, mw2) and size2[-1] == 700 and np.array_equal(np.sort(size), np.sort(size2))


def test_guide_tree_vs_scipy_at_k4000(F):
    """Stages I + II on the device at k = 4000 against a library routine: scipy's single linkage run on the
    rank-transformed similarities the device itself produced (so only stage II is under test here; stage I
    has its own parity tests).  The merge similarities must agree exactly."""
    from scipy.cluster.hierarchy import linkage
    from paper_1603_06958_b200 import synth
    import torch
    k = 4000
    seqs, offsets = synth.family(1, k=k, seed=71)
    with F.famsa_pack(seqs, offsets) as ctx:
        n = F.famsa_rows_pairs(0, k)
        sim = torch.empty(n, dtype=torch.float32, device="cuda")
        F.famsa_lcs_rows(ctx, 0, k, None, sim)
        torch.cuda.synchronize()
        tri = sim.cpu().numpy()
        ia, ib, mw, size = F.famsa_guide_tree(ctx, 512)
    vals, inv = np.unique(tri, return_inverse=True)                   # ascending similarities (inf last)
    dist_rows = (len(vals) - inv).astype(np.float64)                  # highest similarity -> distance 1
    # scipy wants the condensed matrix in (i < j) row-major order; ours is (i > j) by rows: reorder
    ii, jj = np.tril_indices(k, -1)                                   # our order: pair (ii, jj), jj < ii
    cond_index = k * jj - jj * (jj + 1) // 2 + (ii - jj - 1)          # position of (jj, ii) in scipy's order
    cond = np.empty_like(dist_rows)
    cond[cond_index] = dist_rows
    Z = linkage(cond, method="single")
    heights = vals[len(vals) - Z[:, 2].astype(np.int64)]              # back to similarities, descending
    assert np.array_equal(heights, mw) and size[-1] == k
