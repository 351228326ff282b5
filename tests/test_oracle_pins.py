"""Pins for the CPU oracle (oracle/): it is checked against things OTHER than itself --
brute force, closed forms, invariants, an independent second DP, planted structure and
hand values from the paper's formulas.  A dropped term, a wrong sign or
index, or a transposed operand in oracle/lcs_oracle.c fails at least one of these."""
import itertools
import math
import os

import numpy as np
import pytest

LETTERS = "ACDEFGHIKLMNPQRSTVWYBZXUO"
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def brute_lcs(a, b):
    """Definition: the longest string that is a subsequence of both."""
    def is_subseq(s, t):
        it = iter(t)
        return all(c in it for c in s)
    for n in range(min(len(a), len(b)), 0, -1):
        seen = set()
        for idx in itertools.combinations(range(len(a)), n):
            s = tuple(a[i] for i in idx)
            if s in seen:
                continue
            seen.add(s)
            if is_subseq(s, b):
                return n
    return 0


def indel_distance_dp(a, b):
    """Independent second DP: the number of single-symbol insertions and deletions needed to
    transform a into b (in words) -- edit distance without substitutions."""
    la, lb = len(a), len(b)
    E = [[0] * (lb + 1) for _ in range(la + 1)]
    for i in range(la + 1):
        E[i][0] = i
    for j in range(lb + 1):
        E[0][j] = j
    for i in range(1, la + 1):
        for j in range(1, lb + 1):
            best = min(E[i - 1][j] + 1, E[i][j - 1] + 1)
            if a[i - 1] == b[j - 1]:
                best = min(best, E[i - 1][j - 1])
            E[i][j] = best
    return E[la][lb]


def rand_seq(rng, n, sigma):
    return "".join(LETTERS[c] for c in rng.integers(0, sigma, n))


@pytest.mark.parametrize("sigma", [2, 4, 25])
def test_brute_force_tiny(oracle, sigma):
    rng = np.random.default_rng(100 + sigma)
    for _ in range(400):
        a = rand_seq(rng, int(rng.integers(1, 11)), sigma)
        b = rand_seq(rng, int(rng.integers(1, 11)), sigma)
        assert oracle.lcs_len(a, b) == brute_lcs(a, b), (a, b)


def test_invariants(oracle):
    rng = np.random.default_rng(7)
    for _ in range(200):
        sigma = int(rng.choice([2, 4, 20, 25]))
        a = rand_seq(rng, int(rng.integers(1, 200)), sigma)
        b = rand_seq(rng, int(rng.integers(1, 200)), sigma)
        l = oracle.lcs_len(a, b)
        assert oracle.lcs_len(a, a) == len(a)
        assert l == oracle.lcs_len(b, a)                       # symmetry
        assert 0 <= l <= min(len(a), len(b))
        assert l == oracle.lcs_len(a[::-1], b[::-1])           # reversal
        c = LETTERS[int(rng.integers(0, sigma))]
        assert oracle.lcs_len(a, b + c) - l in (0, 1)          # monotone, unit steps
        it = iter(b)
        is_sub = all(ch in it for ch in a)
        assert (l == len(a)) == is_sub                         # greedy subsequence scan


def test_closed_forms(oracle):
    for m, n in [(1, 1), (3, 8), (64, 33), (100, 257)]:
        assert oracle.lcs_len("A" * m, "A" * n) == min(m, n)
    for n in range(1, 30):
        assert oracle.lcs_len("AC" * n, "CA" * n) == 2 * n - 1
    assert oracle.lcs_len("ACDEFGHIKL", "MNPQRSTVWY") == 0     # disjoint symbol sets
    rng = np.random.default_rng(11)
    for _ in range(50):
        a = rand_seq(rng, int(rng.integers(5, 300)), 19)       # symbols 0..18: 'W' (18)... use Y as foreign
        a = a.replace("Y", "A")
        p = int(rng.integers(0, len(a)))
        assert oracle.lcs_len(a, a[:p] + a[p + 1:]) == len(a) - 1   # one deletion
        r = int(rng.integers(1, min(5, len(a)) + 1))
        pos = rng.choice(len(a), r, replace=False)
        b = list(a)
        for q in pos:
            b[q] = "Y"                                          # symbol absent from a
        assert oracle.lcs_len(a, "".join(b)) == len(a) - r


def test_indel_is_insert_delete_distance(oracle):
    rng = np.random.default_rng(13)
    for _ in range(150):
        sigma = int(rng.choice([2, 4, 25]))
        a = rand_seq(rng, int(rng.integers(1, 60)), sigma)
        b = rand_seq(rng, int(rng.integers(1, 60)), sigma)
        l = oracle.lcs_len(a, b)
        assert oracle.indel(len(a), len(b), l) == indel_distance_dp(a, b)
        assert oracle.indel(len(a), len(b), l) == len(a) + len(b) - 2 * l


def test_similarity_hand_values(oracle):
    n = 0
    with open(os.path.join(GOLDEN, "similarity_hand_values.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            a, b, lcs, ind, sim = line.split()[:5]
            l = oracle.lcs_len(a, b)
            assert l == int(lcs), (a, b)
            assert oracle.indel(len(a), len(b), l) == int(ind)
            s = oracle.similarity(len(a), len(b), l)
            if sim == "inf":
                assert math.isinf(s) and s > 0
            else:
                assert s == pytest.approx(float(sim), rel=1e-15)
            n += 1
    assert n >= 8


def test_similarity_range(oracle):
    rng = np.random.default_rng(17)
    for _ in range(200):
        la, lb = int(rng.integers(1, 500)), int(rng.integers(1, 500))
        l = int(rng.integers(1, min(la, lb) + 1))
        if la + lb - 2 * l == 0:
            continue
        s = oracle.similarity(la, lb, l)
        assert 1.0 / (la + lb - 2) ** 2 <= s <= min(la, lb)


def test_planted_subsequence(oracle):
    """B shares with A exactly a planted common subsequence; filler alphabets are disjoint.
    Reaches 4 000 residues (the long multi-word path) where brute force cannot."""
    rng = np.random.default_rng(19)
    for la, lb, p in [(300, 350, 120), (1000, 64, 33), (4000, 3500, 1500), (31, 33, 31)]:
        common = rng.integers(0, 8, p)                       # symbols 0..7
        def embed(n, lo, hi):
            out = rng.integers(lo, hi, n)
            pos = np.sort(rng.choice(n, p, replace=False))
            out[pos] = common
            return np.asarray(out, dtype=np.uint8)
        a = embed(la, 8, 16)                                 # filler 8..15
        b = embed(lb, 16, 24)                                # filler 16..23
        assert oracle.lcs_len(a, b) == p


def test_random_band(oracle):
    """Gross-error smoke test only (band NOT from the paper -- unpinned): two independent
    background sequences of length 1000."""
    from paper_1603_06958_b200 import synth
    rng = np.random.default_rng(23)
    for _ in range(5):
        a, b = synth._draw_bg(rng, 1000), synth._draw_bg(rng, 1000)
        assert 0.25 <= oracle.lcs_len(a, b) / 1000.0 <= 0.50


def test_encode_table(oracle):
    assert list(oracle.encode(LETTERS)) == list(range(25))
    assert list(oracle.encode(LETTERS.lower())) == list(range(25))
    assert list(oracle.encode("Jj")) == [22, 22]              # J -> X (R9)
    assert list(oracle.encode(bytes(range(25)))) == list(range(25))   # codes pass through (R10)
    for bad in ["*", "-", ".", "1", " ", "@", "[", "{", bytes([25]), bytes([31]), bytes([200])]:
        with pytest.raises(ValueError):
            oracle.encode(bad)
    assert oracle.lcs_len("acde", "ACDE") == 4                # X matches X, case folded (R11)
    assert oracle.lcs_len("XXBZ", "XBZ") == 3


def test_sort_perm_and_rows_layout(oracle):
    lens = [5, 9, 5, 2, 9, 7]
    offsets = np.concatenate([[0], np.cumsum(lens)])
    perm = oracle.sort_perm(offsets)
    assert list(perm) == [1, 4, 5, 0, 2, 3]                   # descending, ties by index (R15)
    rng = np.random.default_rng(29)
    seqs = rng.integers(0, 4, offsets[-1]).astype(np.uint8)
    lcs, sim = oracle.rows(seqs, offsets, 0, 6)
    assert lcs.size == 15 == oracle.rows_pairs(0, 6)
    part, _ = oracle.rows(seqs, offsets, 2, 5)
    assert part.size == oracle.rows_pairs(2, 5) == 2 + 3 + 4
    assert list(part) == list(lcs[1:10])                      # rows 2,3,4 of the full triangle
    def seq(t):
        return seqs[offsets[perm[t]]:offsets[perm[t] + 1]]
    assert lcs[4 * 3 // 2 + 1] == oracle.lcs_len(seq(4), seq(1))      # entry (4,1) at i(i-1)/2+j


@pytest.mark.parametrize("isa", [0, 2, 4, 8, -1])
def test_bitparallel_cpu_baseline_matches_dp(oracle, isa):
    """oracle/bitpar_cpu.c is bench.py's context baseline (the paper's own 64-bit multi-pair CPU design,
    PAPER.md:54-56), not an oracle: every lane count (a = 1, 2, 4, 8; the wide ones through the generic code
    path when the host lacks AVX2 / AVX-512, and natively with isa = -1) must agree with the plain-DP oracle,
    including 64-bit word boundaries, ragged column lengths inside one vector and partial last vectors."""
    rng = np.random.default_rng(43)
    lens = [1, 2, 63, 64, 65, 127, 128, 129, 300, 1000, 1025] + [int(x) for x in rng.integers(1, 400, 40)]
    seqs = [rng.integers(0, int(rng.choice([2, 4, 25])), n).astype(np.uint8) for n in lens]
    offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    flat = np.concatenate(seqs)
    k = len(lens)
    pi, pj = [a.ravel() for a in np.meshgrid(np.arange(k), np.arange(k))]       # 51 columns per row: 51 mod 2, 4, 8 != 0
    fast = oracle.bitpar_pairs(flat, offsets, pi, pj, isa=isa, n_threads=3)
    slow, _ = oracle.pairs(flat, offsets, pi, pj, want_sim=False, n_threads=3)
    assert np.array_equal(fast, slow)
    assert oracle.bitpar_best_isa() in oracle.BITPAR_ISA_NAMES


def test_oracle_digests_are_stable(oracle):
    """The oracle + the seeded generator still reproduce the stored digests (tests/golden/oracle_digests.txt,
    written by tests/golden/make_goldens.py from oracle/ only): guards against silent drift of either."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_goldens", os.path.join(GOLDEN, "make_goldens.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = [l.strip() for l in open(os.path.join(GOLDEN, "oracle_digests.txt")) if l.strip() and not l.startswith("#")]
    assert len(stored) == len(mg.CASES)
    for case, line in zip(mg.CASES, stored):
        got = mg.digest(*case).split()
        want = line.split()
        assert got[:7] == want[:7], case
        assert float(got[7]) == pytest.approx(float(want[7]), rel=1e-12)


def test_indel_is_a_metric(oracle):
    """indel(A,B) = |A| + |B| - 2 LCS is the insertion/deletion edit distance, hence a metric:
    zero iff equal, symmetric, triangle inequality.  A wrong LCS (too long or too short) breaks one of them."""
    rng = np.random.default_rng(47)
    for _ in range(120):
        sigma = int(rng.choice([2, 3, 20]))
        a, b, c = (rand_seq(rng, int(rng.integers(1, 80)), sigma) for _ in range(3))
        d = lambda x, y: oracle.indel(len(x), len(y), oracle.lcs_len(x, y))
        assert d(a, a) == 0 and (d(a, b) == 0) == (a == b)
        assert d(a, b) == d(b, a)
        assert d(a, c) <= d(a, b) + d(b, c)
        assert (d(a, b) - (len(a) + len(b))) % 2 == 0 and abs(len(a) - len(b)) <= d(a, b) <= len(a) + len(b)


def test_lcs_of_concatenations(oracle):
    """LCS(A1+A2, B1+B2) >= LCS(A1,B1) + LCS(A2,B2) (superadditivity), with equality when the halves use
    disjoint alphabets; and LCS(A+X, B+X) = LCS(A,B) + |X| for a common suffix X."""
    rng = np.random.default_rng(53)
    for _ in range(60):
        a1, b1 = rand_seq(rng, int(rng.integers(1, 60)), 4), rand_seq(rng, int(rng.integers(1, 60)), 4)      # ACDE
        a2 = "".join("FGHI"[i] for i in rng.integers(0, 4, int(rng.integers(1, 60))))
        b2 = "".join("FGHI"[i] for i in rng.integers(0, 4, int(rng.integers(1, 60))))
        l1, l2 = oracle.lcs_len(a1, b1), oracle.lcs_len(a2, b2)
        assert oracle.lcs_len(a1 + a2, b1 + b2) == l1 + l2                                              # disjoint halves
        m1, m2 = rand_seq(rng, 30, 4), rand_seq(rng, 30, 4)
        assert oracle.lcs_len(a1 + m1, b1 + m2) >= l1 + oracle.lcs_len(m1, m2)
        x = rand_seq(rng, int(rng.integers(1, 40)), 20)
        assert oracle.lcs_len(a1 + x, b1 + x) == l1 + len(x)
