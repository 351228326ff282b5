"""Python face of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It imports nothing from paper_1603_06958_b200 (the CUDA path)
and the CUDA path imports nothing from here.

What it computes (arxiv 1603.06958, readings in DESIGN.md):
  encode      residue bytes -> 25-letter codes                       (R9, R10)
  sort_perm   descending length, ties by ascending original index    (R15)
  lcs_len     textbook DP LCS length
  indel       |A| + |B| - 2 LCS
  similarity  LCS / indel^2 in float64
  rows        the packed-triangular row block [i0, i1) in sorted index space:
              entry (i, j<i) at i(i-1)/2 - i0(i0-1)/2 + j            (R16)
"""
import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        u8p = ctypes.POINTER(ctypes.c_uint8)
        i64p = ctypes.POINTER(ctypes.c_int64)
        lib.oracle_encode.restype = ctypes.c_int64
        lib.oracle_encode.argtypes = [u8p, ctypes.c_int64, u8p]
        lib.oracle_lcs_len.restype = ctypes.c_int32
        lib.oracle_lcs_len.argtypes = [u8p, ctypes.c_int32, u8p, ctypes.c_int32]
        lib.oracle_indel.restype = ctypes.c_int64
        lib.oracle_indel.argtypes = [ctypes.c_int64] * 3
        lib.oracle_similarity.restype = ctypes.c_double
        lib.oracle_similarity.argtypes = [ctypes.c_int64] * 3
        lib.oracle_pairs.restype = ctypes.c_int
        lib.oracle_pairs.argtypes = [u8p, i64p, i64p, i64p, ctypes.c_int64,
                                     ctypes.POINTER(ctypes.c_int32),
                                     ctypes.POINTER(ctypes.c_double), ctypes.c_int32]
        lib.bitpar_rowsets.restype = ctypes.c_int
        lib.bitpar_rowsets.argtypes = [u8p, i64p, i64p, i64p, i64p, ctypes.c_int64, ctypes.c_int32,
                                       ctypes.POINTER(ctypes.c_int32), ctypes.c_int32, ctypes.c_int]
        lib.bitpar_best_isa.restype = ctypes.c_int
        lib.bitpar_best_isa.argtypes = []
        _lib = lib
    return _lib


def _u8(a):
    a = np.ascontiguousarray(a, dtype=np.uint8)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


def _i64(a):
    a = np.ascontiguousarray(a, dtype=np.int64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def as_bytes(seq):
    """str / bytes / array -> uint8 array (no encoding)."""
    if isinstance(seq, str):
        seq = seq.encode("ascii")
    if isinstance(seq, (bytes, bytearray)):
        return np.frombuffer(bytes(seq), dtype=np.uint8).copy()
    return np.ascontiguousarray(seq, dtype=np.uint8)


def encode(seq):
    """Residue bytes -> codes 0..24.  Raises ValueError at the first bad symbol."""
    raw, rp = _u8(as_bytes(seq))
    out = np.empty_like(raw)
    bad = _load().oracle_encode(rp, raw.size, out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)))
    if bad >= 0:
        raise ValueError("bad residue byte %d at position %d" % (int(raw[bad]), bad))
    return out


def lcs_len(a, b):
    """LCS length of two sequences (encoded first, so 'a' == 'A' == code 0)."""
    ea, pa = _u8(encode(a))
    eb, pb = _u8(encode(b))
    return int(_load().oracle_lcs_len(pa, ea.size, pb, eb.size))


def indel(la, lb, lcs):
    return int(_load().oracle_indel(int(la), int(lb), int(lcs)))


def similarity(la, lb, lcs):
    return float(_load().oracle_similarity(int(la), int(lb), int(lcs)))


def sort_perm(offsets):
    """perm[sorted] = original index: descending length, ties by ascending index (R15)."""
    offsets = np.asarray(offsets, dtype=np.int64)
    lens = np.diff(offsets)
    return np.argsort(-lens, kind="stable").astype(np.int64)


def n_threads_default():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def pairs(seqs, offsets, pi, pj, want_sim=True, n_threads=None):
    """LCS (int32) and similarity (float64) for pairs (pi[p], pj[p]) in ORIGINAL index space."""
    codes, cp = _u8(encode(seqs))
    offsets, op = _i64(offsets)
    pi, pip = _i64(pi)
    pj, pjp = _i64(pj)
    n = pi.size
    lcs = np.empty(n, dtype=np.int32)
    sim = np.empty(n, dtype=np.float64) if want_sim else None
    if n_threads is None:
        n_threads = n_threads_default()
    _load().oracle_pairs(cp, op, pip, pjp, n,
                         lcs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                         sim.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if want_sim else None,
                         int(n_threads))
    return lcs, sim


def rows_pairs(i0, i1):
    """Number of entries of row block [i0, i1): sum_{i=i0}^{i1-1} i."""
    return i1 * (i1 - 1) // 2 - i0 * (i0 - 1) // 2


def rows(seqs, offsets, i0, i1, want_sim=True, n_threads=None):
    """Row block [i0, i1) in SORTED index space, packed triangular by rows (R16)."""
    perm = sort_perm(offsets)
    ii = np.repeat(np.arange(i0, i1, dtype=np.int64), np.arange(i0, i1, dtype=np.int64))
    row_start = ii * (ii - 1) // 2 - i0 * (i0 - 1) // 2
    jj = np.arange(ii.size, dtype=np.int64) - row_start
    return pairs(seqs, offsets, perm[ii], perm[jj], want_sim, n_threads)


BITPAR_ISA_NAMES = {0: "scalar (1 pair per step)", 2: "generic 128-bit vectors (a = 2)", 4: "generic 256-bit vectors (a = 4)",
                    8: "generic 512-bit vectors (a = 8)", 14: "AVX2 (a = 4)", 18: "AVX-512 (a = 8)"}


def bitpar_best_isa():
    """The widest multi-pair variant of oracle/bitpar_cpu.c this host runs natively (an ISA code)."""
    return int(_load().bitpar_best_isa())


def bitpar_rowsets(seqs, offsets, row_i, col_ptr, col_j, isa=-1, n_threads=None):
    """CONTEXT BASELINE, not an oracle: the paper's own CPU design (oracle/bitpar_cpu.c):
    64-bit bit-parallel LCS, one task per row sequence (match table built once), its columns taken `a` per
    SIMD register, tasks over threads.  Row r = sequence row_i[r] against col_j[col_ptr[r]:col_ptr[r+1]]
    (ORIGINAL indices).  Returns LCS (int32) parallel to col_j."""
    codes, cp = _u8(encode(seqs))
    offsets, op = _i64(offsets)
    row_i, rp = _i64(row_i)
    col_ptr, pp = _i64(col_ptr)
    col_j, jp = _i64(col_j)
    lcs = np.empty(col_j.size, dtype=np.int32)
    if n_threads is None:
        n_threads = n_threads_default()
    max_len = int(np.diff(offsets).max()) if offsets.size > 1 else 0
    rc = _load().bitpar_rowsets(cp, op, rp, pp, jp, row_i.size, max_len,
                                lcs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), int(n_threads), int(isa))
    if rc != 0:
        raise ValueError("bitpar_rowsets: ISA code %d is not supported on this host" % isa)
    return lcs


def bitpar_pairs(seqs, offsets, pi, pj, isa=-1, n_threads=None):
    """bitpar_rowsets for a flat pair list (ORIGINAL index space): pairs are grouped by pi, which carries
    the bit-vectors.  LCS (int32) in the order of the input pairs."""
    pi = np.asarray(pi, dtype=np.int64)
    pj = np.asarray(pj, dtype=np.int64)
    order = np.argsort(pi, kind="stable")
    rows, counts = np.unique(pi[order], return_counts=True)
    col_ptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    out = np.empty(pi.size, dtype=np.int32)
    out[order] = bitpar_rowsets(seqs, offsets, rows, col_ptr, pj[order], isa, n_threads)
    return out
