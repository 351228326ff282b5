"""Out-of-bounds WRITE detection without a sanitizer (compute-sanitizer is closed on this GPU pool): every
output of the C-ABI calls is placed in the middle of a larger device buffer whose margins hold a canary pattern; after
the call the margins must be untouched and the payload must equal the result of the plain call.  Covers the register
and the blocked sweep paths, both CTA shapes, LCS-only / similarity-only, ragged row ranges, the sequence-versus-profile
batch (scores, paths, path lengths, workspace) and the static-scratch variant."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GUARD = 8192          # elements on each side


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def guarded(n, dtype, canary):
    """(whole buffer, payload view of n elements) with GUARD canary elements before and after the payload."""
    import torch
    whole = torch.full((n + 2 * GUARD,), canary, dtype=dtype, device="cuda")
    return whole, whole[GUARD:GUARD + n]


def guards_intact(whole, n, canary):
    import torch
    ref = torch.full((GUARD,), canary, dtype=whole.dtype, device="cuda")
    return bool(torch.equal(whole[:GUARD], ref)) and bool(torch.equal(whole[GUARD + n:], ref))


@pytest.mark.parametrize("cfg,k,seed", [(1, 900, 71), (2, 230, 72), (4, 700, 73)])
def test_sweep_outputs_stay_inside_their_buffers(F, cfg, k, seed):
    import torch
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(cfg, k=k, seed=seed)
    rng = np.random.default_rng(seed)
    with F.famsa_pack(seqs, offsets) as ctx:
        n_all = F.famsa_rows_pairs(0, k)
        ref_l = torch.zeros(n_all, dtype=torch.int16, device="cuda")
        ref_s = torch.zeros(n_all, dtype=torch.float32, device="cuda")
        F.famsa_lcs_rows(ctx, 0, k, ref_l, ref_s)
        ranges = [(0, k), (0, 1), (1, 2), (k - 1, k)] + [tuple(sorted(rng.integers(0, k + 1, 2).tolist())) for _ in range(6)]
        for small in (0, 1):
            F.famsa_ctx_set_tuning(ctx, 0, small, 0)
            for i0, i1 in ranges:
                n = F.famsa_rows_pairs(i0, i1)
                if n == 0:
                    continue
                base = F.famsa_rows_pairs(0, i0)
                for want_l, want_s in ((True, True), (True, False), (False, True)):
                    wl, pl = guarded(n, torch.int16, 0x5A5A)
                    ws, ps = guarded(n, torch.float32, -12345.0)
                    F.famsa_lcs_rows(ctx, i0, i1, pl if want_l else None, ps if want_s else None)
                    torch.cuda.synchronize()
                    assert guards_intact(wl, n, 0x5A5A) and guards_intact(ws, n, -12345.0), (cfg, small, i0, i1)
                    if want_l:
                        assert torch.equal(pl, ref_l[base:base + n])
                    else:
                        assert bool((pl == 0x5A5A).all())                      # an output that was not asked for is not touched
                    if want_s:
                        assert torch.equal(ps, ref_s[base:base + n])
                    else:
                        assert bool((ps == -12345.0).all())
                ck_w, ck = guarded(2, torch.int64, 77)
                ck.zero_()
                wl, pl = guarded(n, torch.int16, 0x5A5A)
                F.famsa_lcs_rows_checksum(ctx, i0, i1, pl, None, ck)
                torch.cuda.synchronize()
                assert guards_intact(ck_w, 2, 77) and guards_intact(wl, n, 0x5A5A)


def test_seqprof_outputs_stay_inside_their_buffers(F):
    import torch
    from paper_1603_06958_b200 import synth
    lengths = [(1, 1), (3, 1024), (700, 5), (64, 129), (200, 511), (90, 640), (33, 897)] + [(40 + 9 * q, 30 + 31 * q) for q in range(30)]
    counts, col_off, seq, seq_off, nseq = synth.profile_batch(len(lengths), seed=81, lengths=lengths)
    B = len(lengths)
    gaps = np.tile(np.array([0.66, 0.66, 14.85, 1.25], np.float32), (B, 1))
    d_counts = torch.from_numpy(counts.astype(np.int32)).cuda()
    d_subst = torch.from_numpy(synth.substitution_matrix()).cuda()
    cw, cost = guarded(counts.shape[0] * 32, torch.float32, -7.0)
    F.famsa_profile_costs(d_counts, d_subst, cost)
    torch.cuda.synchronize()
    assert guards_intact(cw, counts.shape[0] * 32, -7.0)
    d_seq, d_gaps, d_nseq = torch.from_numpy(seq).cuda(), torch.from_numpy(gaps).cuda(), torch.from_numpy(nseq).cuda()
    n_path = int(col_off[-1] + seq_off[-1])
    n_ws = F.famsa_seqprof_workspace(col_off, seq_off)
    sw, score = guarded(B, torch.float32, -5.0)
    pw, path = guarded(n_path, torch.uint8, 0xEE)
    lw, plen = guarded(B, torch.int32, -3)
    ww, ws = guarded(n_ws, torch.uint8, 0xC3)
    F.famsa_seqprof_align(cost, col_off, d_seq, seq_off, d_gaps, d_nseq, score, path, plen, ws)
    torch.cuda.synchronize()
    assert guards_intact(sw, B, -5.0) and guards_intact(pw, n_path, 0xEE) and guards_intact(lw, B, -3) and guards_intact(ww, n_ws, 0xC3)
    lens = plen.cpu().numpy()
    n1, n2 = np.diff(col_off), np.diff(seq_off)
    assert np.all(lens >= np.maximum(n1, n2)) and np.all(lens <= n1 + n2)
    # the unused head of every path segment keeps the canary: paths are right-aligned and never start early
    hp = path.cpu().numpy()
    for b in range(B):
        a, e = int(col_off[b] + seq_off[b]), int(col_off[b + 1] + seq_off[b + 1])
        assert np.all(hp[a:e - lens[b]] == 0xEE) and np.all(hp[e - lens[b]:e] <= 2)
    # score-only mode and the static-scratch variant write the scores and nothing else
    for call in ("align", "static"):
        sw2, score2 = guarded(B, torch.float32, -5.0)
        if call == "align":
            F.famsa_seqprof_align(cost, col_off, d_seq, seq_off, d_gaps, d_nseq, score2)
        else:
            F.famsa_seqprof_scores_static(cost, col_off, d_seq, seq_off, d_gaps, d_nseq, score2)
        torch.cuda.synchronize()
        assert guards_intact(sw2, B, -5.0) and torch.equal(score2, score)
