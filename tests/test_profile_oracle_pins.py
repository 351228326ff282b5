"""Pins of the NEXT-4 oracle (oracle/profile_oracle.c: sequence-versus-profile DP, PAPER.md:71-79, 111-116,
133-139) against things other than itself: brute-force enumeration of every alignment path scored from the
gap-run definition, the pinned LCS oracle (zero gap costs, 0/1 scores), a textbook single-matrix
Needleman-Wunsch (linear gaps), closed forms for terminal / internal / profile-side gaps, g_scale values."""
import math

import numpy as np

from oracle import profile_oracle as po


def one_seq_profile(a, match=1.0, mismatch=0.0):
    cost = np.full((len(a), po.SYMS), mismatch, np.float32)
    cost[np.arange(len(a)), a] = match
    return cost


def test_brute_force_all_paths():
    """max over ALL paths of the run-based path score == the DP score, and the DP's own path attains it."""
    rng = np.random.default_rng(5)
    n_cases = 0
    for n1 in range(1, 5):
        for n2 in range(1, 5):
            paths = po.all_paths(n1, n2)
            for trial in range(6):
                if trial % 2 == 0:
                    cost = rng.integers(-4, 9, (n1, po.SYMS)).astype(np.float32)
                    gaps = rng.integers(0, 7, 4).astype(np.float32)
                else:
                    cost = rng.normal(0, 3, (n1, po.SYMS)).astype(np.float32)
                    gaps = rng.uniform(0, 6, 4).astype(np.float32)
                y = rng.integers(0, 25, n2).astype(np.uint8)
                nseq = int(rng.integers(1, 4))
                best = max(po.path_score(cost, y, gaps, nseq, p) for p in paths)
                score, path = po.align(cost, y, gaps, nseq, want_path=True)
                assert abs(score - best) <= 1e-9 * max(1.0, abs(best)), (n1, n2, trial, score, best)
                assert abs(po.path_score(cost, y, gaps, nseq, path) - best) <= 1e-9 * max(1.0, abs(best))
                assert (path == po.OP_M).sum() + (path == po.OP_X).sum() == n1
                assert (path == po.OP_M).sum() + (path == po.OP_Y).sum() == n2
                n_cases += 1
    assert n_cases == 96
    assert len(po.all_paths(3, 3)) == 63                      # Delannoy number D(3, 3)


def test_reduces_to_lcs(oracle):
    """0/1 column scores of a one-sequence profile and free gaps: the score is the LCS length (pinned oracle)."""
    rng = np.random.default_rng(6)
    for _ in range(40):
        a = rng.integers(0, 6, int(rng.integers(1, 60))).astype(np.uint8)
        y = rng.integers(0, 6, int(rng.integers(1, 60))).astype(np.uint8)
        s = po.align(one_seq_profile(a), y, (0, 0, 0, 0), 1)
        assert s == oracle.lcs_len(a, y)


def test_reduces_to_textbook_needleman_wunsch():
    """open == extension everywhere, one sequence: the single-matrix recurrence H = max(diag + s, up - g, left - g)."""
    rng = np.random.default_rng(7)
    for _ in range(25):
        n1, n2 = int(rng.integers(1, 40)), int(rng.integers(1, 40))
        cost = rng.integers(-3, 6, (n1, po.SYMS)).astype(np.float32)
        y = rng.integers(0, 25, n2).astype(np.uint8)
        g = float(rng.integers(0, 5))
        H = np.zeros((n1 + 1, n2 + 1))
        H[:, 0] = -g * np.arange(n1 + 1); H[0, :] = -g * np.arange(n2 + 1)
        for i in range(1, n1 + 1):
            for j in range(1, n2 + 1):
                H[i, j] = max(H[i - 1, j - 1] + cost[i - 1, y[j - 1]], H[i - 1, j] - g, H[i, j - 1] - g)
        assert po.align(cost, y, (g, g, g, g), 1) == H[n1, n2]


def test_closed_forms_for_the_four_gap_types():
    """terminal open/extension at the ends, open/extension inside, x nseq for gap columns."""
    rng = np.random.default_rng(8)
    a = rng.permutation(25)[:20].astype(np.uint8)             # 20 distinct symbols: the optimal alignment is forced
    cost = one_seq_profile(a, match=10.0, mismatch=-10.0)
    To, Te, Go, Ge = 3.0, 0.5, 7.0, 1.0
    g = (To, Te, Go, Ge)
    assert po.align(cost, a, g, 1) == 200.0                                            # identical: no gap
    assert po.align(cost, a[5:], g, 1) == 150.0 - (To + 4 * Te)                        # 5 columns before the first residue
    assert po.align(cost, a[:14], g, 1) == 140.0 - (To + 5 * Te)                       # 6 columns after the last residue
    assert po.align(cost, np.concatenate([a[:8], a[11:]]), g, 1) == 170.0 - (Go + 2 * Ge)   # 3 columns inside
    ins = np.array([25, 26, 27, 28], np.uint8)                                         # symbols no column likes
    for nseq in (1, 3):
        y = np.concatenate([a[:8], ins, a[8:]])
        assert po.align(cost, y, g, nseq) == 200.0 - nseq * (Go + 3 * Ge)              # 4 gap columns inside the profile
        y = np.concatenate([ins[:2], a])
        assert po.align(cost, y, g, nseq) == 200.0 - nseq * (To + Te)                  # 2 gap columns before column 0
        y = np.concatenate([a, ins[:3]])
        assert po.align(cost, y, g, nseq) == 200.0 - nseq * (To + 2 * Te)              # 3 gap columns after the last column
    # consecutive gap columns in BOTH inputs may be optimal: X directly followed by Y
    cost2 = one_seq_profile(np.array([1, 2, 3], np.uint8), match=5.0, mismatch=-50.0)
    s, path = po.align(cost2, np.array([1, 9, 3], np.uint8), (1, 1, 1, 1), 1, want_path=True)
    assert s == 10.0 - 2.0 and sorted(path.tolist()) == [0, 0, 1, 2]


def test_gap_scale_values():
    """g_scale = 1 + ln(k / 45) / 7."""
    assert po.gap_scale(45) == 1.0
    assert abs(po.gap_scale(45 * math.e ** 7) - 2.0) < 1e-12
    assert abs(po.gap_scale(415519) - (1 + math.log(415519 / 45) / 7)) < 1e-12
    assert po.gap_scale(10) < 1.0 < po.gap_scale(1000)


def test_profile_costs_is_counts_times_matrix():
    rng = np.random.default_rng(9)
    counts = rng.integers(0, 50, (37, po.SYMS)).astype(np.uint32)
    subst = rng.integers(-4, 12, (po.SYMS, po.SYMS)).astype(np.float32)
    ref = counts.astype(np.float64) @ subst.astype(np.float64)
    assert np.array_equal(po.profile_costs(counts, subst), ref.astype(np.float32))
    one = np.zeros((5, po.SYMS), np.uint32); one[np.arange(5), [3, 1, 4, 1, 5]] = 1
    assert np.array_equal(po.profile_costs(one, subst), subst[[3, 1, 4, 1, 5]])       # one sequence: rows of the matrix


def test_f32_mode_equals_f64_on_exact_inputs():
    """Small-integer inputs are exact in both precisions: same score, same path (same tie rule)."""
    rng = np.random.default_rng(10)
    for _ in range(20):
        n1, n2 = int(rng.integers(1, 80)), int(rng.integers(1, 80))
        cost = rng.integers(-4, 9, (n1, po.SYMS)).astype(np.float32)
        y = rng.integers(0, 25, n2).astype(np.uint8)
        gaps = rng.integers(0, 7, 4).astype(np.float32)
        s64, p64 = po.align(cost, y, gaps, 2, want_path=True)
        s32, p32 = po.align(cost, y, gaps, 2, want_path=True, precision="f32")
        assert s64 == s32 and np.array_equal(p64, p32)
