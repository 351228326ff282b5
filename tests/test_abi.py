"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol that
include/famsa_lcs.h declares, and its host logic (argument validation, famsa_rows_pairs,
error texts) behaves as the header states.  No compute call is made without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def F():
    from paper_1603_06958_b200 import build, famsa
    build.build()
    return famsa


def test_exports_match_header(F):
    text = open(os.path.join(ROOT, "include", "famsa_lcs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(famsa_[a-z_]+)\s*\(", text)))
    assert declared == sorted(F.EXPORTS)
    L = F.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_profile_exports_match_header(F):
    text = open(os.path.join(ROOT, "include", "famsa_profile.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(famsa_[a-z_]+)\s*\(", text)))
    assert declared == sorted(F.EXPORTS_PROFILE)
    L = F.lib()
    for name in declared:
        assert hasattr(L, name), name
    # host logic of the NEXT-4 boundary (no GPU needed)
    assert F.famsa_gap_scale(45) == 1.0
    assert F.famsa_seqprof_workspace([0, 10, 30], [0, 100, 400]) == (10 + 15) * 16 * 8 + (20 + 31) * 32 * 12 + 2
    with pytest.raises(F.FamsaError) as e:
        F.famsa_seqprof_workspace([0, 10], [0, 2000])         # more than 1024 residues
    assert e.value.code == F.FAMSA_ELENGTH
    # argument validation happens before any CUDA call
    off = np.arange(F.FAMSA_SEQPROF_STATIC_MAX + 2, dtype=np.int64)
    assert L.famsa_seqprof_scores_static(None, off.ctypes.data, None, off.ctypes.data, None, None, F.FAMSA_SEQPROF_STATIC_MAX + 1, None, None) == F.FAMSA_ERANGE
    assert b"FAMSA_SEQPROF_STATIC_MAX" in L.famsa_last_error()
    assert L.famsa_seqprof_scores_static(None, off.ctypes.data, None, off.ctypes.data, None, None, 3, None, None) == F.FAMSA_EINVAL
    assert L.famsa_seqprof_align(None, off.ctypes.data, None, off.ctypes.data, None, None, 3, None, None, None, None, None) == F.FAMSA_EINVAL
    assert L.famsa_seqprof_align(None, None, None, None, None, None, 3, None, None, None, None, None) == F.FAMSA_EINVAL
    assert L.famsa_seqprof_align(None, off.ctypes.data, None, off.ctypes.data, None, None, 0, None, None, None, None, None) == F.FAMSA_OK
    assert L.famsa_profile_costs(None, None, 5, None, None) == F.FAMSA_EINVAL


def test_rows_pairs(F):
    assert F.famsa_rows_pairs(0, 0) == 0
    assert F.famsa_rows_pairs(0, 1) == 0            # row 0 is empty
    assert F.famsa_rows_pairs(0, 500) == 124750     # config 0 (BASELINE.json)
    assert F.famsa_rows_pairs(0, 415519) == 86327811921
    assert F.famsa_rows_pairs(7, 9) == 7 + 8
    assert F.famsa_rows_pairs(3, 2) == -1
    assert F.famsa_rows_pairs(-1, 2) == -1


def test_pack_validation_before_device(F):
    seqs = np.zeros(10, np.uint8)
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(seqs, np.array([1, 5, 10]))
    assert e.value.code == F.FAMSA_EINVAL            # offsets[0] != 0
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(seqs, np.array([0, 6, 5, 10]))
    assert e.value.code == F.FAMSA_EINVAL            # decreasing
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(seqs, np.array([0, 5, 5, 10]))
    assert e.value.code == F.FAMSA_ELENGTH           # empty sequence
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(np.zeros(70000, np.uint8), np.array([0, 70000]))
    assert e.value.code == F.FAMSA_ELENGTH           # longer than 65535
    out = ctypes.c_void_p()
    assert F.lib().famsa_pack(None, None, 0, 0, ctypes.byref(out)) == F.FAMSA_EINVAL
    assert F.lib().famsa_pack(seqs.ctypes.data, np.array([0, 10]).ctypes.data, 1, 0, None) == F.FAMSA_EINVAL


def test_no_cpu_fallback(F):
    """Without a CUDA device the product path fails loudly (FAMSA_ECUDA); it never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(F.FamsaError) as e:
        F.famsa_pack(np.zeros(10, np.uint8), np.array([0, 4, 10]))
    assert e.value.code == F.FAMSA_ECUDA
    with pytest.raises(F.FamsaError):
        F.famsa_alu_peak(0)


def test_null_ctx_and_strerror(F):
    L = F.lib()
    assert L.famsa_lcs_rows(None, 0, 0, None, None, None) == F.FAMSA_EINVAL
    assert L.famsa_lcs_rows_host(None, 0, 0, None, None) == F.FAMSA_EINVAL
    assert L.famsa_k(None, None) == F.FAMSA_EINVAL
    L.famsa_free(None)                               # no-op
    assert L.famsa_launch_count(None) == 0
    for code in range(0, -7, -1):
        assert L.famsa_strerror(code).decode() not in ("", "unknown error")
    assert L.famsa_strerror(-99).decode() == "unknown error"
    assert L.famsa_ctx_set_tuning(None, 0, -1, 0) == F.FAMSA_EINVAL      # the tuning knobs belong to a ctx
    assert L.famsa_lcs_rows_checksum(None, 0, 0, None, None, None, None) == F.FAMSA_EINVAL
    assert L.famsa_host_profile(None, 1) == F.FAMSA_EINVAL and L.famsa_host_profile_read(None, None) == F.FAMSA_EINVAL
    assert L.famsa_trim() == F.FAMSA_OK                                  # nothing pooled: a no-op


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code: neither imports or includes the other."""
    def code_lines(path):
        return [l.strip() for l in open(path) if re.match(r"\s*(import |from |#include)", l)]
    pkg = os.path.join(ROOT, "paper_1603_06958_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                for l in code_lines(os.path.join(dirpath, f)):
                    assert "oracle" not in l, (f, l)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            for l in code_lines(os.path.join(ROOT, "oracle", f)):
                assert "paper_1603_06958_b200" not in l and "famsa_lcs.h" not in l and "famsa_internal" not in l, (f, l)
