"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Bar: uint16 LCS bit-exact; fp32 similarity within 1e-6 relative of the
oracle's float64 (inf == inf) -- BASELINE.json north_star."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SIM_RTOL = 1e-6
LETTERS = "ACDEFGHIKLMNPQRSTVWYBZXUO"


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1603_06958_b200 import build, famsa
    build.build()
    famsa.lib()              # raises if the extension is missing: no fallback
    return famsa


def gpu_rows(F, ctx, i0, i1, want_lcs=True, want_sim=True):
    import torch
    n = F.famsa_rows_pairs(i0, i1)
    lcs = torch.full((max(n, 1),), 0xFFFF, dtype=torch.uint16, device="cuda") if want_lcs else None
    sim = torch.full((max(n, 1),), -1.0, dtype=torch.float32, device="cuda") if want_sim else None
    F.famsa_lcs_rows(ctx, i0, i1, lcs, sim)
    torch.cuda.synchronize()
    return (lcs.cpu().numpy()[:n].astype(np.int64) if want_lcs else None,
            sim.cpu().numpy()[:n] if want_sim else None)


def assert_match(lcs_gpu, sim_gpu, lcs_ref, sim_ref):
    if lcs_gpu is not None:
        bad = np.flatnonzero(lcs_gpu != lcs_ref)
        assert bad.size == 0, "LCS mismatch at %s: gpu %s oracle %s" % (bad[:5], lcs_gpu[bad[:5]], lcs_ref[bad[:5]])
    if sim_gpu is not None:
        inf_ref = np.isinf(sim_ref)
        assert np.array_equal(np.isinf(sim_gpu) & (sim_gpu > 0), inf_ref)
        fin = ~inf_ref
        err = np.abs(sim_gpu[fin].astype(np.float64) - sim_ref[fin])
        assert np.all(err <= SIM_RTOL * np.abs(sim_ref[fin])), float((err / np.maximum(np.abs(sim_ref[fin]), 1e-300)).max())


def check_all_rows(F, oracle, seqs, offsets, i0=0, i1=None):
    k = len(offsets) - 1
    i1 = k if i1 is None else i1
    with F.famsa_pack(seqs, offsets) as ctx:
        lcs, sim = gpu_rows(F, ctx, i0, i1)
    lref, sref = oracle.rows(seqs, offsets, i0, i1)
    assert_match(lcs, sim, lref, sref)
    return lcs, sim


def make_set(seq_list):
    arrs = [np.frombuffer(s.encode(), np.uint8) if isinstance(s, str) else np.asarray(s, np.uint8) for s in seq_list]
    offsets = np.concatenate([[0], np.cumsum([a.size for a in arrs])]).astype(np.int64)
    return (np.concatenate(arrs) if arrs else np.zeros(0, np.uint8)), offsets


# ---- a1-a3: what pack builds ----------------------------------------------------------------
def test_pack_roundtrip(F, oracle):
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(2, k=200, seed=5)          # short + long sequences (blocked tables)
    with F.famsa_pack(seqs, offsets) as ctx:
        assert F.famsa_k(ctx) == 200
        perm = F.famsa_perm(ctx)
        lens = F.famsa_lengths(ctx)
        assert np.array_equal(perm, oracle.sort_perm(offsets))           # descending, stable (R15)
        assert np.array_equal(lens, np.diff(offsets)[perm])
        cells = F.famsa_rows_cells(ctx, 0, 200)
        L = lens.astype(np.float64)
        assert cells == pytest.approx(sum(L[i] * L[:i].sum() for i in range(200)), rel=1e-12)
        for s in [0, 1, 19, 20, 31, 32, 100, 199]:
            ref = oracle.encode(seqs[offsets[perm[s]]:offsets[perm[s] + 1]])
            assert np.array_equal(F.famsa_codes(ctx, s, lens[s]), ref)
            for c in [0, 9, 24, 25, 31]:
                bits = np.zeros(((lens[s] + 31) // 32) * 32, np.uint8)
                bits[:lens[s]] = ref == c                                # bit i of M[c] = (S[i] == c)
                words = np.packbits(bits.reshape(-1, 32), axis=1, bitorder="little").view(np.uint32).ravel()
                assert np.array_equal(F.famsa_match(ctx, s, c, lens[s]), words), (s, c)


def test_letters_and_bad_symbols(F, oracle):
    seqs, offsets = make_set(["ACDEFGHIKLMNPQRSTVWY", "acdefghiklmnpqrstvwy", "BZXUOJ", "bzxuoj", "MKVLAAGIVGL"])
    lcs, sim = check_all_rows(F, oracle, seqs, offsets)
    assert 20 in lcs and np.isinf(sim).sum() == 2        # case folded: two identical pairs
    for bad in ["ACD*F", "ACD-F", "ACD F", "ACD1F", "ACD@F", "ACD[F", "ACD{F"]:
        s, o = make_set(["ACDEF", bad])
        with pytest.raises(F.FamsaError) as e:
            F.famsa_pack(s, o)
        assert e.value.code == F.FAMSA_ESYMBOL and "position 8" in str(e.value)
    s, o = make_set([np.array([0, 1, 25], np.uint8)])
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(s, o)
    assert e.value.code == F.FAMSA_ESYMBOL


# ---- a4-a7: the sweep -------------------------------------------------------------------------
def test_config0_all_pairs(F, oracle):
    """BASELINE.json configs[0]: k = 500, all 124 750 pairs."""
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(0)
    lcs, sim = check_all_rows(F, oracle, seqs, offsets)
    assert lcs.size == 124750
    assert np.isinf(sim).sum() >= 3                      # the planted duplicates (R12)


def test_degenerate_sizes(F, oracle):
    import torch
    for seq_list in ([], ["ACD"], ["ACD", "AC"], ["A", "A"], ["A", "C"]):
        seqs, offsets = make_set(seq_list)
        check_all_rows(F, oracle, seqs, offsets)
    seqs, offsets = make_set(["ACDEF", "ACD", "AC"])
    with F.famsa_pack(seqs, offsets) as ctx:
        buf = torch.zeros(8, dtype=torch.uint16, device="cuda")
        F.famsa_lcs_rows(ctx, 1, 1, buf, None)           # empty range: legal, writes nothing
        F.famsa_lcs_rows(ctx, 0, 1, buf, None)           # row 0 is empty
        assert int(buf.cpu().numpy().astype(np.int64).sum()) == 0
        for i0, i1 in [(2, 1), (0, 4), (-1, 2)]:
            with pytest.raises(F.FamsaError) as e:
                F.famsa_lcs_rows(ctx, i0, i1, buf, None)
            assert e.value.code == F.FAMSA_ERANGE
        with pytest.raises(F.FamsaError) as e:
            F.famsa_lcs_rows(ctx, 0, 3, None, None)
        assert e.value.code == F.FAMSA_EINVAL


def test_word_boundaries(F, oracle):
    """|A| = 0, 1, 31 mod 32 and every register-path word count 1..32, plus the first blocked sizes."""
    rng = np.random.default_rng(31)
    lens = [1, 2, 31, 32, 33, 63, 64, 65, 95, 96, 97, 127, 128, 129, 255, 256, 257, 511, 512, 513,
            991, 992, 993, 1023, 1024, 1025, 1055, 1056, 1057, 2047, 2048, 2049] + list(range(40, 1030, 32))
    seq_list = [rng.integers(0, 4, n).astype(np.uint8) for n in lens]     # 4 letters: LCS is long, carries are busy
    seqs, offsets = make_set(seq_list)
    check_all_rows(F, oracle, seqs, offsets)


def test_closed_forms_on_gpu(F, oracle):
    """Inputs whose answer is known in closed form, independent of the oracle."""
    n = 700
    seq_list = ["A" * 1500, "A" * 64, "AC" * n, "CA" * n, "D" * 33, "W" * 1024, "W" * 1025]
    seqs, offsets = make_set(seq_list)
    with F.famsa_pack(seqs, offsets) as ctx:
        perm = F.famsa_perm(ctx)
        lcs, _ = gpu_rows(F, ctx, 0, len(seq_list))
    inv = np.argsort(perm)
    def get(a, b):
        i, j = max(inv[a], inv[b]), min(inv[a], inv[b])
        return lcs[i * (i - 1) // 2 + j]
    assert get(0, 1) == 64 and get(2, 3) == 2 * n - 1 and get(0, 4) == 0
    assert get(5, 6) == 1024 and get(0, 2) == n and get(1, 3) == 64


def test_row_block_independence(F, oracle):
    """(i, j) does not depend on block boundaries, tile shape or co-launched pairs."""
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(1, k=1300, seed=77)
    k = 1300
    with F.famsa_pack(seqs, offsets) as ctx:
        full_lcs, full_sim = gpu_rows(F, ctx, 0, k)
        for block in (1, 7, 1024):
            lo = 1100 if block == 1 else (900 if block == 7 else 0)
            for i0 in range(lo, k, block):
                i1 = min(i0 + block, k)
                l, s = gpu_rows(F, ctx, i0, i1)
                a, b = F.famsa_rows_pairs(0, i0), F.famsa_rows_pairs(0, i1)
                assert np.array_equal(l, full_lcs[a:b]) and np.array_equal(s, full_sim[a:b])
        for ta, small, l2mb in ((1, -1, 0), (3, 0, 1), (12, 0, 0), (8, 0, 4096), (0, 1, 0), (0, 1, 1)):
            F.famsa_ctx_set_tuning(ctx, ta, small, l2mb)        # tile shapes, one-warp CTAs, L2 column groups
            l, s = gpu_rows(F, ctx, 0, k)
            assert np.array_equal(l, full_lcs) and np.array_equal(s, full_sim)
        F.famsa_ctx_set_tuning(ctx)                             # back to the shipped defaults (the knobs are per ctx)
        l, _ = gpu_rows(F, ctx, 100, 300, want_sim=False)       # LCS only (configs[3])
        _, s = gpu_rows(F, ctx, 100, 300, want_lcs=False)       # similarity only
        a, b = F.famsa_rows_pairs(0, 100), F.famsa_rows_pairs(0, 300)
        assert np.array_equal(l, full_lcs[a:b]) and np.array_equal(s, full_sim[a:b])
        hl = np.empty(F.famsa_rows_pairs(0, k), np.uint16)
        hs = np.empty(F.famsa_rows_pairs(0, k), np.float32)
        F.famsa_lcs_rows_host(ctx, 0, k, hl, hs)                # the HOST-buffer entry point
        assert np.array_equal(hl.astype(np.int64), full_lcs) and np.array_equal(hs, full_sim)
    sel = np.arange(0, full_lcs.size, 97)
    lref, sref = oracle.rows(seqs, offsets, 0, k)
    assert_match(full_lcs, full_sim, lref, sref)
    assert sel.size > 0


def test_config2_long_path(F, oracle):
    """BASELINE.json configs[2] recipe at k = 320: 1 500-4 000-residue sequences (blocked carry path)."""
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(2, k=320, seed=91)
    assert np.diff(offsets).max() > 1500
    check_all_rows(F, oracle, seqs, offsets)


def test_config3_fragments_lcs_only(F, oracle):
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(3, k=600, seed=93)
    with F.famsa_pack(seqs, offsets) as ctx:
        lcs, _ = gpu_rows(F, ctx, 0, 600, want_sim=False)
    lref, _ = oracle.rows(seqs, offsets, 0, 600, want_sim=False)
    assert_match(lcs, None, lref, None)


def test_maximum_lengths(F, oracle):
    """FAMSA_MAX_LEN = 65535 and the large carry-vector variant (|B| > 4096)."""
    rng = np.random.default_rng(37)
    lens = [65535, 30000, 6000, 4097, 4096, 1025, 300, 1]
    seq_list = [rng.integers(0, 20, n).astype(np.uint8) for n in lens]
    seq_list.append(seq_list[2].copy())                           # a long duplicate: LCS = 6000, +inf
    seqs, offsets = make_set(seq_list)
    lcs, sim = check_all_rows(F, oracle, seqs, offsets)
    assert 6000 in lcs and np.isinf(sim).sum() == 1


def test_planted_long(F):
    """Planted common subsequence between disjoint-alphabet fillers: LCS known exactly, no oracle."""
    rng = np.random.default_rng(41)
    p = 1700
    common = rng.integers(0, 8, p)
    def embed(n, lo, hi):
        out = rng.integers(lo, hi, n)
        out[np.sort(rng.choice(n, p, replace=False))] = common
        return out.astype(np.uint8)
    seqs, offsets = make_set([embed(3900, 8, 16), embed(3500, 16, 24)])
    with F.famsa_pack(seqs, offsets) as ctx:
        lcs, sim = gpu_rows(F, ctx, 0, 2)
    assert lcs[0] == p
    assert sim[0] == pytest.approx(p / float(3900 + 3500 - 2 * p) ** 2, rel=1e-6)


def test_random_sets(F, oracle):
    """Seeded random sets: ragged lengths 1..1300 (register path, every rows-per-thread variant, and the
    blocked path), alphabets of 2-25 letters, set sizes that leave partial warps and partial row steps."""
    rng = np.random.default_rng(101)
    for trial in range(6):
        k = int(rng.integers(2, 140))
        sigma = int(rng.choice([2, 4, 20, 25]))
        hi = int(rng.choice([40, 300, 700, 1300]))
        seq_list = [rng.integers(0, sigma, int(rng.integers(1, hi + 1))).astype(np.uint8) for _ in range(k)]
        if trial % 2:
            seq_list[int(rng.integers(0, k))] = seq_list[0].copy()        # an exact duplicate
        seqs, offsets = make_set(seq_list)
        check_all_rows(F, oracle, seqs, offsets)


def test_random_long_sets(F, oracle):
    """Seeded random sets with sequences of up to 9 000 residues: the blocked path with 2-9 table blocks per row,
    both carry-vector sizes (|B| <= 4096 and above), mixed with short rows in the same set."""
    rng = np.random.default_rng(202)
    for hi, k in ((4096, 14), (9000, 10), (2500, 24)):
        lens = [int(x) for x in rng.integers(1025, hi + 1, k // 2)] + [int(x) for x in rng.integers(1, 1200, k - k // 2)]
        seq_list = [rng.integers(0, int(rng.choice([4, 20])), n).astype(np.uint8) for n in lens]
        seqs, offsets = make_set(seq_list)
        check_all_rows(F, oracle, seqs, offsets)


def test_two_streams_one_ctx(F, oracle):
    """One ctx serves concurrent famsa_lcs_rows calls on different streams (it is read-only after pack)."""
    import torch
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(1, k=900, seed=55)
    k = 900
    with F.famsa_pack(seqs, offsets) as ctx:
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        n1, n2 = F.famsa_rows_pairs(0, 600), F.famsa_rows_pairs(600, k)
        l1 = torch.zeros(n1, dtype=torch.uint16, device="cuda"); f1 = torch.zeros(n1, dtype=torch.float32, device="cuda")
        l2 = torch.zeros(n2, dtype=torch.uint16, device="cuda"); f2 = torch.zeros(n2, dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        for _ in range(3):
            F.famsa_lcs_rows(ctx, 0, 600, l1, f1, s1)
            F.famsa_lcs_rows(ctx, 600, k, l2, f2, s2)
        torch.cuda.synchronize()
        lcs = np.concatenate([l1.cpu().numpy(), l2.cpu().numpy()]).astype(np.int64)
        sim = np.concatenate([f1.cpu().numpy(), f2.cpu().numpy()])
    lref, sref = oracle.rows(seqs, offsets, 0, k)
    assert_match(lcs, sim, lref, sref)


def test_alu_peak_is_sane(F):
    """The roofline denominator: the ALU pipe issues 64 thread-instructions per clock per SM on sm_100."""
    p = F.famsa_alu_peak(0)
    assert 55.0 < p["instr_per_clk_sm"] <= 64.5
    assert 1000.0 < p["sm_mhz"] < 2300.0
    assert p["instr_per_s"] == pytest.approx(p["instr_per_clk_sm"] * p["sm_mhz"] * 1e6 * 148, rel=0.05)


def test_checksum_epilogue_against_the_oracle(F, oracle):
    """famsa_lcs_rows_checksum ("a 64-bit checksum per block ... to prove the work was done"): the sums
    the kernels' epilogue accumulates equal the ORACLE's sum of LCS lengths and the sum of the stored fp32 bit patterns,
    for the register path in both CTA shapes and for the blocked long path; the call ADDS to what is there."""
    import torch
    from paper_1603_06958_b200 import synth
    for cfg, k, seed in ((1, 700, 55), (2, 260, 56)):
        seqs, offsets = synth.family(cfg, k=k, seed=seed)
        lref, _ = oracle.rows(seqs, offsets, 0, k)
        n = F.famsa_rows_pairs(0, k)
        with F.famsa_pack(seqs, offsets) as ctx:
            for small in (0, 1):
                F.famsa_ctx_set_tuning(ctx, 0, small, 0)
                lcs = torch.zeros(n, dtype=torch.uint16, device="cuda")
                sim = torch.zeros(n, dtype=torch.float32, device="cuda")
                ck = torch.tensor([5, 7], dtype=torch.int64, device="cuda")
                F.famsa_lcs_rows_checksum(ctx, 0, k // 2, lcs, sim, ck)
                half = F.famsa_rows_pairs(0, k // 2)
                F.famsa_lcs_rows_checksum(ctx, k // 2, k, lcs[half:], sim[half:], ck)
                torch.cuda.synchronize()
                c = ck.cpu().numpy()
                assert int(c[0]) - 5 == int(lref.sum())
                bits = int(sim.cpu().numpy().view(np.uint32).astype(np.uint64).sum())
                assert (int(c[1]) - 7) % 2 ** 64 == bits % 2 ** 64
                assert np.array_equal(lcs.cpu().numpy().astype(np.int64), lref)
                ck2 = torch.zeros(2, dtype=torch.int64, device="cuda")
                F.famsa_lcs_rows_checksum(ctx, 0, k, lcs, None, ck2)       # LCS only: [1] untouched
                torch.cuda.synchronize()
                assert ck2.cpu().numpy().tolist() == [int(lref.sum()), 0]


def test_profiling_getters(F):
    """famsa_mix_peak (the instruction-mix ceiling printed in every bench line), the per-phase timers of the host path
    in both modes, famsa_pack_profile, famsa_trim."""
    import torch
    from paper_1603_06958_b200 import synth
    m = F.famsa_mix_peak(0)
    assert 45.0 < m["alu_instr_per_clk_sm"] <= F.famsa_alu_peak(0)["instr_per_clk_sm"] + 0.5
    seqs, offsets = synth.family(1, k=900, seed=57)
    n = F.famsa_rows_pairs(0, 900)
    with F.famsa_pack(seqs, offsets) as ctx:
        pp = F.famsa_pack_profile(ctx)
        assert all(v >= 0.0 for v in pp.values()) and sum(pp.values()) > 0.0
        F.famsa_host_profile(ctx, True)
        hl = torch.empty(n, dtype=torch.uint16).pin_memory(); hs = torch.empty(n, dtype=torch.float32).pin_memory()
        F.famsa_lcs_rows_host(ctx, 0, 900, hl, hs)                          # pinned: direct stores
        p = F.famsa_host_profile_read(ctx)
        assert p["chunks"] == 1 and p["d2h_ms"] == 0.0 and p["sweep_ms"] > 0.0 and p["d2h_bytes"] == 6.0 * n
        nl = np.empty(n, np.uint16); nsim = np.empty(n, np.float32)
        F.famsa_lcs_rows_host(ctx, 0, 900, nl, nsim)                        # pageable: staged chunks + copies
        p = F.famsa_host_profile_read(ctx)
        assert p["chunks"] >= 1 and p["d2h_ms"] > 0.0 and p["sweep_ms"] > 0.0 and p["d2h_bytes"] == 6.0 * n
        assert np.array_equal(nl, hl.numpy().view(np.uint16)) and np.array_equal(nsim, hs.numpy())
    F.famsa_trim()


def test_gpu_matches_stored_oracle_digests(F):
    """The CUDA path against digests the oracle wrote earlier (tests/golden/oracle_digests.txt): the
    expected values do not come from this run, nor ever from the CUDA path."""
    import hashlib
    import os
    from paper_1603_06958_b200 import synth
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_digests.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        config, k, seed, residues, sha, total, n_inf, _ = line.split()
        seqs, offsets = synth.family(int(config), k=int(k), seed=None if seed == "default" else int(seed))
        assert seqs.size == int(residues)
        with F.famsa_pack(seqs, offsets) as ctx:
            lcs, sim = gpu_rows(F, ctx, 0, int(k))
        assert hashlib.sha256(np.ascontiguousarray(lcs, dtype="<i4").tobytes()).hexdigest() == sha
        assert int(lcs.sum()) == int(total) and int(np.isinf(sim).sum()) == int(n_inf)
        n += 1
    assert n == 5


def test_host_path_async(F, oracle):
    """famsa_lcs_rows_host_async + famsa_sync: row blocks streamed into two pinned host buffers give the
    same values as the synchronous host call."""
    import torch
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(1, k=1100, seed=61)
    k, block = 1100, 256
    with F.famsa_pack(seqs, offsets) as ctx:
        n_all = F.famsa_rows_pairs(0, k)
        ref_l = np.empty(n_all, np.uint16); ref_s = np.empty(n_all, np.float32)
        F.famsa_lcs_rows_host(ctx, 0, k, ref_l, ref_s)
        mp = F.famsa_rows_pairs(k - block, k)
        hl = [torch.empty(mp, dtype=torch.uint16).pin_memory() for _ in range(2)]
        hs = [torch.empty(mp, dtype=torch.float32).pin_memory() for _ in range(2)]
        blocks = [(a, min(a + block, k)) for a in range(0, k, block)]
        # pinned buffers: mode -1 / 1 = the kernels store into them directly, mode 0 = staged chunks + copies
        for mode in (-1, 0, 1):
            F.famsa_host_mode(ctx, mode)
            for n in range(0, len(blocks), 2):
                pair = blocks[n:n + 2]
                for q, (a, b) in enumerate(pair):
                    hl[q].zero_(); hs[q].zero_()
                    F.famsa_lcs_rows_host_async(ctx, a, b, hl[q], hs[q] if mode != 1 or n else None)
                F.famsa_sync(ctx)
                for q, (a, b) in enumerate(pair):
                    lo, hi = F.famsa_rows_pairs(0, a), F.famsa_rows_pairs(0, b)
                    assert np.array_equal(hl[q].numpy()[:hi - lo].view(np.uint16), ref_l[lo:hi])
                    if mode != 1 or n:
                        assert np.array_equal(hs[q].numpy()[:hi - lo], ref_s[lo:hi])
        with pytest.raises(F.FamsaError):                     # direct mode refuses pageable memory
            F.famsa_lcs_rows_host(ctx, 0, k, ref_l, ref_s)
        F.famsa_host_mode(ctx, -1)
    lref, sref = oracle.rows(seqs, offsets, 0, k)
    assert_match(ref_l.astype(np.int64), ref_s, lref, sref)
