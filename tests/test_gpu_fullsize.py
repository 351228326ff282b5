"""Full-size parity in the launch configuration bench.py times (1024-row blocks of the packed
BASELINE.json configs[1] and configs[4] sets), on sampled outputs the oracle computes one by one."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

BLOCK_ROWS = 1024


def check_blocks(F, oracle, seqs, offsets, block_ids, n_per_block, want_sim=True):
    import torch
    k = len(offsets) - 1
    perm_ref = oracle.sort_perm(offsets)
    checked = 0
    with F.famsa_pack(seqs, offsets) as ctx:
        assert np.array_equal(F.famsa_perm(ctx), perm_ref)
        lens = F.famsa_lengths(ctx)
        for b in block_ids:
            i0, i1 = b * BLOCK_ROWS, min((b + 1) * BLOCK_ROWS, k)
            n = F.famsa_rows_pairs(i0, i1)
            lcs = torch.full((n,), 0xFFFF, dtype=torch.uint16, device="cuda")
            sim = torch.full((n,), -1.0, dtype=torch.float32, device="cuda") if want_sim else None
            F.famsa_lcs_rows(ctx, i0, i1, lcs, sim)
            # seeded sample inside the block: uniform + first/last rows + word-boundary lengths
            rng = np.random.default_rng(1000 + b)
            lo = max(i0, 1)
            rows = rng.integers(lo, i1, n_per_block)
            rows[:64] = lo
            rows[64:128] = i1 - 1
            special = np.flatnonzero(np.isin(lens[lo:i1] % 32, (0, 1, 31))) + lo
            if special.size:
                rows[128:192] = rng.choice(special, 64)
            cols = (rng.random(n_per_block) * rows).astype(np.int64)
            cols[:8] = 0
            cols[64:72] = rows[64:72] - 1                                  # first and last column of a row
            pos = rows * (rows - 1) // 2 - i0 * (i0 - 1) // 2 + cols
            idx = torch.from_numpy(pos).cuda()
            torch.cuda.synchronize()
            lg = lcs.view(torch.int16)[idx].cpu().numpy().view(np.uint16).astype(np.int64)
            lref, sref = oracle.pairs(seqs, offsets, perm_ref[rows], perm_ref[cols], want_sim=want_sim)
            assert np.array_equal(lg, lref), (b, np.flatnonzero(lg != lref)[:5])
            if want_sim:
                sg = sim[idx].cpu().numpy().astype(np.float64)
                fin = np.isfinite(sref)
                assert np.array_equal(np.isinf(sg), ~fin)
                assert np.all(np.abs(sg[fin] - sref[fin]) <= 1e-6 * np.abs(sref[fin]))
            # a property that holds for EVERY entry of the block, checked on the device:
            # 0 < LCS <= |A| (row i is the shorter sequence) -- every entry was written
            li = torch.from_numpy(np.repeat(lens[i0:i1].astype(np.int32), np.arange(i0, i1))).cuda()
            lv = lcs.view(torch.int16).to(torch.int32).bitwise_and(0xFFFF)
            assert bool((lv <= li).all())
            del lcs, sim, li, lv
            checked += n_per_block
    return checked


@pytest.fixture(scope="module")
def family4():
    """BASELINE.json configs[4] (k = 415 519), generated once for this module (~45 s of host time)."""
    from paper_1603_06958_b200 import synth
    return synth.family(4)


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def duplicate_pairs(seqs, offsets, inv_perm):
    """(i, j < i) in SORTED index space for every pair of byte-identical input sequences (the generator
    plants three such pairs; they are the entries where indel = 0, R12).  Plain hashing of the
    input bytes: none of the method's arithmetic."""
    seen, pi, pj = {}, [], []
    buf = seqs.tobytes()
    for t in range(len(offsets) - 1):
        key = buf[int(offsets[t]):int(offsets[t + 1])]
        if key in seen:
            a, b = int(inv_perm[seen[key]]), int(inv_perm[t])
            pi.append(max(a, b)); pj.append(min(a, b))
        else:
            seen[key] = t
    return np.array(pi, np.int64), np.array(pj, np.int64)


def test_config1_full_size_sampled(F, oracle):
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(1)
    assert len(offsets) - 1 == 10000
    assert check_blocks(F, oracle, seqs, offsets, range(10), 2500) == 25000


def test_config4_full_size_sampled(F, oracle, family4):
    """k = 415 519: the set bench.py times; blocks from the long end, the middle and the short end."""
    seqs, offsets = family4
    k = len(offsets) - 1
    assert k == 415519
    last = (k - 1) // BLOCK_ROWS
    assert check_blocks(F, oracle, seqs, offsets, [0, 1, 96, 240, last - 1, last], 6000) == 36000


def test_config4_one_million_sampled_pairs_of_the_full_sweep(F, oracle, family4):
    """BASELINE.json configs[4]: "~8.6e10 pairs computed as streamed row blocks, oracle checked on 1e6 seeded
    sampled pairs".  The WHOLE sweep runs in the bench configuration (1024-row blocks, LCS + similarity);
    from every block the sampled entries are gathered on the device; all of them are then checked against
    the oracle: 1e6 uniform pairs plus the strata of synth.sample_pairs (longest x longest, shortest,
    block-boundary rows, lengths = 0, 1, 31 mod 32) and the planted duplicates."""
    import torch
    from paper_1603_06958_b200 import synth
    seqs, offsets = family4
    k = len(offsets) - 1
    perm_ref = oracle.sort_perm(offsets)
    with F.famsa_pack(seqs, offsets) as ctx:
        lens = F.famsa_lengths(ctx)
        si, sj = synth.sample_pairs(k, 1_000_000, seed=20260406, lengths_sorted=lens, block_rows=BLOCK_ROWS)
        inv = np.empty(k, np.int64); inv[perm_ref] = np.arange(k)
        di, dj = duplicate_pairs(seqs, offsets, inv)                       # the planted duplicates join the sample
        assert di.size >= 3
        key = np.unique(np.concatenate([si * k + sj, di * k + dj]))
        si, sj = key // k, key % k
        assert si.size >= 1_000_000 and np.all(sj < si)
        order = np.argsort(si, kind="stable")
        si, sj = si[order], sj[order]
        nblocks = (k + BLOCK_ROWS - 1) // BLOCK_ROWS
        bounds = np.searchsorted(si, np.arange(nblocks + 1) * BLOCK_ROWS)
        max_pairs = F.famsa_rows_pairs(k - BLOCK_ROWS, k)
        lcs = torch.empty(max_pairs, dtype=torch.uint16, device="cuda")
        sim = torch.empty(max_pairs, dtype=torch.float32, device="cuda")
        got_l = torch.empty(si.size, dtype=torch.int16, device="cuda")
        got_s = torch.empty(si.size, dtype=torch.float32, device="cuda")
        pos_all = torch.from_numpy(si * (si - 1) // 2 + sj).cuda()
        for b in range(nblocks):
            i0, i1 = b * BLOCK_ROWS, min((b + 1) * BLOCK_ROWS, k)
            F.famsa_lcs_rows(ctx, i0, i1, lcs, sim)
            lo, hi = int(bounds[b]), int(bounds[b + 1])
            if hi > lo:
                idx = pos_all[lo:hi] - i0 * (i0 - 1) // 2
                got_l[lo:hi] = lcs.view(torch.int16)[idx]
                got_s[lo:hi] = sim[idx]
        torch.cuda.synchronize()
        gl = got_l.cpu().numpy().view(np.uint16).astype(np.int64)
        gs = got_s.cpu().numpy().astype(np.float64)
    lref, sref = oracle.pairs(seqs, offsets, perm_ref[si], perm_ref[sj])
    bad = np.flatnonzero(gl != lref)
    assert bad.size == 0, (bad[:5], gl[bad[:5]], lref[bad[:5]])
    fin = np.isfinite(sref)
    assert np.array_equal(np.isinf(gs), ~fin) and (~fin).sum() >= 3      # the planted duplicates are in the sample
    assert np.all(np.abs(gs[fin] - sref[fin]) <= 1e-6 * np.abs(sref[fin]))


def test_config4_guide_tree_full_size(F, oracle, family4):
    """Stages I + II at the size README/BASELINE quote (k = 415 519): the guide tree the device
    builds from 406 streamed row blocks is checked for VALIDITY with the oracle, since several trees are
    correct under similarity ties (R19):
      1. each of the k-1 spanning-tree edges carries the true similarity of its pair (oracle, 415 518 pairs);
      2. the edges span all k leaves without a cycle;
      3. the dendrogram is well formed (every cluster merged exactly once, sizes add up to k, merge
         similarities non-increasing and equal to the sorted edge similarities), and the merge height of
         every tree edge's endpoints is that edge's similarity;
      4. the cycle property of a maximum spanning tree on 10^6 seeded sampled pairs: the oracle's
         similarity(i, j) never exceeds the merge similarity at which i and j first share a cluster."""
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    from oracle import slink_oracle as so
    seqs, offsets = family4
    k = len(offsets) - 1
    perm_ref = oracle.sort_perm(offsets)
    with F.famsa_pack(seqs, offsets) as ctx:
        assert np.array_equal(F.famsa_perm(ctx), perm_ref)
        forest = F.famsa_guide_forest(ctx, BLOCK_ROWS, 0, 1)
        a, b, w = F.famsa_tree_edges(forest)
        ia, ib, mw, size = F.famsa_tree_finish(forest)
        forest.free()
    # 1
    assert a.size == k - 1 and np.all(a > b) and a.max() < k and b.min() >= 0
    _, sref = oracle.pairs(seqs, offsets, perm_ref[a], perm_ref[b])
    fin = np.isfinite(sref)
    assert np.array_equal(np.isinf(w), ~fin)
    assert np.all(np.abs(w[fin].astype(np.float64) - sref[fin]) <= 1e-6 * sref[fin])
    # 2
    g = coo_matrix((np.ones(k - 1), (a, b)), shape=(k, k))
    assert connected_components(g, directed=False)[0] == 1            # k-1 edges + connected = a spanning tree
    # 3
    assert np.all(ia < ib) and size[-1] == k
    assert np.array_equal(np.sort(np.concatenate([ia, ib])), np.arange(2 * k - 2))
    csize = np.concatenate([np.ones(k, np.int64), size])
    assert np.array_equal(csize[ia] + csize[ib], size)
    mwf = mw[np.isfinite(mw)]
    assert np.all(np.diff(mwf) <= 0) and np.array_equal(np.isinf(mw), np.arange(k - 1) < np.isinf(mw).sum())
    assert np.array_equal(np.sort(w)[::-1], mw)
    assert np.array_equal(so.dendrogram_pair_heights(k, ia, ib, mw, a, b), w.astype(np.float64))
    # 4
    rng = np.random.default_rng(20261104)
    qi = rng.integers(1, k, 1_000_000)
    qj = (rng.random(qi.size) * qi).astype(np.int64)
    h = so.dendrogram_pair_heights(k, ia, ib, mw, qi, qj)
    _, s = oracle.pairs(seqs, offsets, perm_ref[qi], perm_ref[qj])
    bad = np.flatnonzero(~(s <= h * (1 + 1e-6)))
    assert bad.size == 0, (qi[bad[:5]], qj[bad[:5]], s[bad[:5]], h[bad[:5]])
