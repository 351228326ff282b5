"""GPU parity of SURVEY.md 8(f) NEXT-4 (sequence-versus-profile DP, include/famsa_profile.h) against
oracle/profile_oracle.c, through the C ABI.  The kernel computes in fp32; the oracle's float64 score is the
reference within a tolerance derived from the arithmetic (one rounding per addition along a path of at most
n1 + n2 steps: (n1 + n2) * 2^-24 relative to the largest partial score), and where floating point decides an
integer -- the traceback -- both sides decide in fp32 (the oracle's f32 mode), so paths are compared exactly."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

BASE_GAPS = np.array([0.66, 0.66, 14.85, 1.25], np.float32)     # magnitudes only: terminal gaps cheap, opens dear


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def run_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst, want_path=True):
    import torch
    dev = "cuda"
    B = col_off.size - 1
    d_counts = torch.from_numpy(counts.astype(np.int32)).to(dev)
    d_subst = torch.from_numpy(subst).to(dev)
    d_cost = torch.empty((counts.shape[0], 32), dtype=torch.float32, device=dev)
    F.famsa_profile_costs(d_counts, d_subst, d_cost)
    d_seq = torch.from_numpy(seq).to(dev)
    d_gaps = torch.from_numpy(np.ascontiguousarray(gaps, dtype=np.float32)).to(dev)
    d_nseq = torch.from_numpy(nseq).to(dev)
    score = torch.full((B,), float("nan"), dtype=torch.float32, device=dev)
    path = plen = ws = None
    if want_path:
        path = torch.full((int(col_off[-1] + seq_off[-1]),), 9, dtype=torch.uint8, device=dev)
        plen = torch.zeros(B, dtype=torch.int32, device=dev)
        ws = torch.empty(F.famsa_seqprof_workspace(col_off, seq_off), dtype=torch.uint8, device=dev)
    F.famsa_seqprof_align(d_cost, col_off, d_seq, seq_off, d_gaps, d_nseq, score, path, plen, ws)
    torch.cuda.synchronize()
    out = [d_cost.cpu().numpy(), score.cpu().numpy()]
    if want_path:
        out += [path.cpu().numpy(), plen.cpu().numpy()]
    return out


def check_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst):
    from oracle import profile_oracle as po
    cost, score, path, plen = run_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst)
    assert np.array_equal(cost, po.profile_costs(counts, subst))               # a1: counts x matrix, exact
    for b in range(col_off.size - 1):
        c = cost[col_off[b]:col_off[b + 1]]
        y = seq[seq_off[b]:seq_off[b + 1]]
        n1, n2 = c.shape[0], y.size
        s64 = po.align(c, y, gaps[b], int(nseq[b]))
        s32, p32 = po.align(c, y, gaps[b], int(nseq[b]), want_path=True, precision="f32")
        assert score[b] == np.float32(s32), (b, n1, n2, score[b], s32)          # same precision: bit-exact
        scale = max(abs(s64), float(np.abs(c).max()) * min(n1, n2), 1.0)
        assert abs(float(score[b]) - s64) <= (n1 + n2) * 2.0 ** -24 * scale * 4, (b, n1, n2, score[b], s64)
        end = int(col_off[b + 1] + seq_off[b + 1])
        got = path[end - plen[b]:end]
        assert np.array_equal(got, p32), (b, n1, n2)                            # decisions taken in fp32 on both sides
        assert (got == 0).sum() + (got == 1).sum() == n1 and (got == 0).sum() + (got == 2).sum() == n2
        assert abs(po.path_score(c, y, gaps[b], int(nseq[b]), got) - s64) <= (n1 + n2) * 2.0 ** -24 * scale * 8


def test_batch_against_oracle(F):
    from paper_1603_06958_b200 import synth
    from oracle import profile_oracle as po
    subst = synth.substitution_matrix()
    counts, col_off, seq, seq_off, nseq = synth.profile_batch(48, seed=401)
    gaps = np.stack([BASE_GAPS * np.float32(po.gap_scale(200 + 50 * b)) for b in range(48)])
    assert np.float32(F.famsa_gap_scale(415519)) == np.float32(po.gap_scale(415519))
    check_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst)


def test_every_lane_width_and_the_edges(F):
    """n2 at both sides of every residues-per-lane boundary (multiples of 64 up to 1024), the smallest inputs, long and short profiles."""
    from paper_1603_06958_b200 import synth
    subst = synth.substitution_matrix()
    lengths = [(1, 1), (1, 5), (7, 1), (2, 2), (20, 63), (20, 64), (20, 65), (25, 191), (25, 192), (25, 193), (30, 320), (30, 321), (30, 448),
               (30, 449), (30, 576), (30, 577), (30, 704), (30, 705), (30, 832), (30, 833), (30, 960), (30, 961), (40, 127), (40, 128), (40, 129), (33, 256), (33, 257), (35, 384), (35, 385), (90, 511),
               (90, 512), (90, 513), (50, 640), (50, 641), (45, 768), (45, 769), (45, 896), (45, 897), (60, 1023), (60, 1024),
               (1500, 31), (900, 300), (5, 700), (31, 32), (32, 33), (64, 4)]
    counts, col_off, seq, seq_off, nseq = synth.profile_batch(len(lengths), seed=402, lengths=lengths)
    rng = np.random.default_rng(403)
    gaps = np.stack([BASE_GAPS * np.float32(rng.uniform(0.5, 2.0)) for _ in lengths])
    gaps[3] = 0.0                                                               # free gaps
    gaps[5] = [9.0, 3.0, 1.0, 0.5]                                              # terminal gaps dearer than internal ones
    check_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst)


def test_exact_inputs_ties_and_score_only(F):
    """Small-integer inputs (many ties): the fp32 path equals the float64 oracle's path; score-only mode agrees."""
    from oracle import profile_oracle as po
    rng = np.random.default_rng(404)
    B = 24
    n1s, n2s = rng.integers(1, 200, B), rng.integers(1, 300, B)
    col_off = np.concatenate([[0], np.cumsum(n1s)]).astype(np.int64)
    seq_off = np.concatenate([[0], np.cumsum(n2s)]).astype(np.int64)
    counts = rng.integers(0, 3, (int(col_off[-1]), 32)).astype(np.uint32)
    subst = rng.integers(-2, 4, (32, 32)).astype(np.float32)
    seq = rng.integers(0, 25, int(seq_off[-1])).astype(np.uint8)
    nseq = rng.integers(1, 4, B).astype(np.int32)
    gaps = rng.integers(0, 6, (B, 4)).astype(np.float32)
    cost, score, path, plen = run_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst)
    only = run_batch(F, counts, col_off, seq, seq_off, nseq, gaps, subst, want_path=False)[1]
    assert np.array_equal(score, only)
    for b in range(B):
        c = cost[col_off[b]:col_off[b + 1]]; y = seq[seq_off[b]:seq_off[b + 1]]
        s64, p64 = po.align(c, y, gaps[b], int(nseq[b]), want_path=True)
        end = int(col_off[b + 1] + seq_off[b + 1])
        assert float(score[b]) == s64 and np.array_equal(path[end - plen[b]:end], p64)


def test_back_to_back_calls_without_synchronisation(F):
    """Three batches enqueued on one stream with no host synchronisation in between (the call stages its descriptors
    through two pinned buffers): every batch's scores and paths equal the oracle's fp32 mode."""
    import torch
    from paper_1603_06958_b200 import synth
    from oracle import profile_oracle as po
    subst = synth.substitution_matrix()
    d_subst = torch.from_numpy(subst).cuda()
    jobs = []
    for n, seed in ((9, 411), (17, 412), (5, 413)):
        counts, col_off, seq, seq_off, nseq = synth.profile_batch(n, seed=seed, n1_range=(20, 300))
        gaps = np.tile(BASE_GAPS, (n, 1))
        cost = torch.empty((counts.shape[0], 32), dtype=torch.float32, device="cuda")
        bufs = dict(cost=cost, counts=torch.from_numpy(counts.astype(np.int32)).cuda(), seq=torch.from_numpy(seq).cuda(),
                    gaps=torch.from_numpy(gaps).cuda(), nseq=torch.from_numpy(nseq).cuda(),
                    score=torch.empty(n, dtype=torch.float32, device="cuda"),
                    path=torch.empty(int(col_off[-1] + seq_off[-1]), dtype=torch.uint8, device="cuda"),
                    plen=torch.empty(n, dtype=torch.int32, device="cuda"),
                    ws=torch.empty(F.famsa_seqprof_workspace(col_off, seq_off), dtype=torch.uint8, device="cuda"))
        jobs.append((col_off, seq, seq_off, nseq, gaps, bufs))
    for col_off, seq, seq_off, nseq, gaps, b in jobs:           # enqueue everything first
        F.famsa_profile_costs(b["counts"], d_subst, b["cost"])
        F.famsa_seqprof_align(b["cost"], col_off, b["seq"], seq_off, b["gaps"], b["nseq"], b["score"], b["path"], b["plen"], b["ws"])
    torch.cuda.synchronize()
    for col_off, seq, seq_off, nseq, gaps, b in jobs:
        cost, score, path, plen = b["cost"].cpu().numpy(), b["score"].cpu().numpy(), b["path"].cpu().numpy(), b["plen"].cpu().numpy()
        for q in range(col_off.size - 1):
            s32, p32 = po.align(cost[col_off[q]:col_off[q + 1]], seq[seq_off[q]:seq_off[q + 1]], gaps[q], int(nseq[q]), want_path=True, precision="f32")
            end = int(col_off[q + 1] + seq_off[q + 1])
            assert score[q] == np.float32(s32) and np.array_equal(path[end - plen[q]:end], p32)


def test_errors(F):
    import torch
    z = torch.zeros(64, dtype=torch.float32, device="cuda")
    s = torch.zeros(2048, dtype=torch.uint8, device="cuda")
    n = torch.ones(1, dtype=torch.int32, device="cuda")
    for col_off, seq_off in (([0, 2], [0, 0]), ([0, 0], [0, 2]), ([0, 2], [0, 1025])):
        with pytest.raises(F.FamsaError) as e:
            F.famsa_seqprof_align(z, col_off, s, seq_off, z, n, z)
        assert e.value.code == F.FAMSA_ELENGTH
