"""famsa_seqprof_scores_static (include/famsa_profile.h): the score-only sequence-versus-profile batch that allocates
nothing -- its scratch is a file-scope static device array -- against the existing path, famsa_seqprof_align.
Collected LAST on purpose (the suite runs with pytest -x).  Self-contained: passes alone in a fresh process and after
the other GPU tests.  Both paths run the same kernels in fp32, so the tolerance is the one tests/test_gpu_profile.py
uses for same-precision results: bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

BASE_GAPS = np.array([0.66, 0.66, 14.85, 1.25], np.float32)


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def make_batch(F, n, seed, lengths=None):
    import torch
    from paper_1603_06958_b200 import synth
    counts, col_off, seq, seq_off, nseq = synth.profile_batch(n, seed=seed, n1_range=(20, 400), lengths=lengths)
    gaps = np.tile(BASE_GAPS, (n, 1)) * np.linspace(0.7, 1.6, n, dtype=np.float32)[:, None]
    cost = torch.empty((counts.shape[0], 32), dtype=torch.float32, device="cuda")
    F.famsa_profile_costs(torch.from_numpy(counts.astype(np.int32)).cuda(), torch.from_numpy(synth.substitution_matrix()).cuda(), cost)
    return dict(cost=cost, col_off=col_off, seq=torch.from_numpy(seq).cuda(), seq_off=seq_off,
                gaps=torch.from_numpy(np.ascontiguousarray(gaps, dtype=np.float32)).cuda(), nseq=torch.from_numpy(nseq).cuda(), n=n)


def existing_path(F, b):
    import torch
    score = torch.full((b["n"],), float("nan"), dtype=torch.float32, device="cuda")
    F.famsa_seqprof_align(b["cost"], b["col_off"], b["seq"], b["seq_off"], b["gaps"], b["nseq"], score)
    torch.cuda.synchronize()
    return score.cpu().numpy()


def test_static_scratch_entry_point_matches_existing_path_on_two_calls_in_a_row(F):
    import torch
    # every residues-per-lane class occurs in the first batch; the second is smaller and differently shaped, so
    # anything the shared array kept from the first call would show
    lengths = [(50 + 7 * q, 1 + (q * 37) % 1024) for q in range(96)]
    first = make_batch(F, 96, seed=901, lengths=lengths)
    second = make_batch(F, 41, seed=902)
    ref1, ref2 = existing_path(F, first), existing_path(F, second)
    assert np.all(np.isfinite(ref1)) and np.all(np.isfinite(ref2))
    s1 = torch.full((first["n"],), float("nan"), dtype=torch.float32, device="cuda")
    s2 = torch.full((second["n"],), float("nan"), dtype=torch.float32, device="cuda")
    # two calls in a row on one stream, no synchronisation in between
    F.famsa_seqprof_scores_static(first["cost"], first["col_off"], first["seq"], first["seq_off"], first["gaps"], first["nseq"], s1)
    F.famsa_seqprof_scores_static(second["cost"], second["col_off"], second["seq"], second["seq_off"], second["gaps"], second["nseq"], s2)
    torch.cuda.synchronize()
    assert np.array_equal(s1.cpu().numpy(), ref1)
    assert np.array_equal(s2.cpu().numpy(), ref2)
    # and once more, the first batch again after the smaller one
    s1.fill_(float("nan"))
    F.famsa_seqprof_scores_static(first["cost"], first["col_off"], first["seq"], first["seq_off"], first["gaps"], first["nseq"], s1)
    torch.cuda.synchronize()
    assert np.array_equal(s1.cpu().numpy(), ref1)


def test_static_scratch_entry_point_rejects_batches_beyond_its_maximum(F):
    import torch
    n = F.FAMSA_SEQPROF_STATIC_MAX + 1
    off = np.arange(n + 1, dtype=np.int64)
    z = torch.zeros(4 * n, dtype=torch.float32, device="cuda")
    with pytest.raises(F.FamsaError) as e:
        F.famsa_seqprof_scores_static(torch.zeros((n, 32), dtype=torch.float32, device="cuda"), off, torch.zeros(n, dtype=torch.uint8, device="cuda"), off,
                                      z, torch.ones(n, dtype=torch.int32, device="cuda"), z)
    assert e.value.code == F.FAMSA_ERANGE and "FAMSA_SEQPROF_STATIC_MAX" in str(e.value)
