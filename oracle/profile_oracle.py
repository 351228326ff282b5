"""Python face of oracle/profile_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The sequence-versus-profile DP of FAMSA's stage III (PAPER.md:71-79, 111-116,
133-139; readings P1-P9 in DESIGN.md).  Imports nothing from paper_1603_06958_b200 and is imported by
nothing there.

  profile_costs(counts, subst)          cost[i][c] = sum_d counts[i][d] * subst[d][c]
  gap_scale(k)                          1 + ln(k / 45) / 7
  align(cost, y, gaps, nseq, ...)       global affine-gap alignment score (+ path), float64, or float32 when
                                        the traceback of the fp32 kernel is compared (same-precision decisions)
  path_score(cost, y, gaps, nseq, path) the score of a GIVEN path, computed from the gap RUNS of the path, not
                                        by the recurrence: the independent check used by the brute-force pin
"""
import ctypes

import numpy as np

from . import build as _build

SYMS = 32
OP_M, OP_X, OP_Y = 0, 1, 2      # column~residue, column~gap in the sequence, residue~gap column in the profile
_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        fp = ctypes.POINTER(ctypes.c_float)
        u8p = ctypes.POINTER(ctypes.c_uint8)
        for name in ("oracle_seqprof_align_f64", "oracle_seqprof_align_f32"):
            f = getattr(lib, name)
            f.restype = ctypes.c_int
            f.argtypes = [fp, ctypes.c_int32, u8p, ctypes.c_int32, fp, ctypes.c_int32,
                          ctypes.POINTER(ctypes.c_double), u8p, ctypes.POINTER(ctypes.c_int32)]
        lib.oracle_profile_costs.restype = None
        lib.oracle_profile_costs.argtypes = [ctypes.POINTER(ctypes.c_uint32), fp, ctypes.c_int32, fp]
        lib.oracle_gap_scale.restype = ctypes.c_double
        lib.oracle_gap_scale.argtypes = [ctypes.c_double] * 3
        _lib = lib
    return _lib


def profile_costs(counts, subst):
    counts = np.ascontiguousarray(counts, dtype=np.uint32)
    subst = np.ascontiguousarray(subst, dtype=np.float32)
    assert counts.ndim == 2 and counts.shape[1] == SYMS and subst.shape == (SYMS, SYMS)
    out = np.empty((counts.shape[0], SYMS), np.float32)
    _load().oracle_profile_costs(counts.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
                                 subst.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), counts.shape[0],
                                 out.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    return out


def gap_scale(k, g_l=45.0, g_d=7.0):
    return float(_load().oracle_gap_scale(float(k), float(g_l), float(g_d)))


def align(cost, y, gaps, nseq=1, want_path=False, precision="f64"):
    """Returns score (float) or (score, path uint8 array).  cost: float32 [n1][32]; y: codes; gaps: (T_o, T_e, G_o, G_e)."""
    cost = np.ascontiguousarray(cost, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.uint8)
    g = np.ascontiguousarray(gaps, dtype=np.float32)
    assert cost.ndim == 2 and cost.shape[1] == SYMS and g.size == 4 and cost.shape[0] >= 1 and y.size >= 1
    n1, n2 = cost.shape[0], y.size
    score = ctypes.c_double()
    path = np.zeros(n1 + n2, np.uint8) if want_path else None
    plen = ctypes.c_int32(0)
    f = getattr(_load(), "oracle_seqprof_align_" + precision)
    rc = f(cost.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), n1, y.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), n2,
           g.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), int(nseq), ctypes.byref(score),
           path.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)) if want_path else None, ctypes.byref(plen))
    if rc != 0:
        raise MemoryError("oracle_seqprof_align")
    if want_path:
        return score.value, path[:plen.value].copy()
    return score.value


def path_score(cost, y, gaps, nseq, path):
    """Score of one alignment path from its definition, NOT from the recurrence: the sum of
    the column scores of the matched (column, residue) pairs minus, for every maximal RUN of equal gap
    operations of length L, open + (L - 1) * extension -- terminal costs when the run lies before the first
    or after the last residue (X runs) / column (Y runs); a Y run costs nseq times as much."""
    cost = np.asarray(cost, dtype=np.float64)
    To, Te, Go, Ge = (float(np.float32(v)) for v in gaps)
    n1, n2 = cost.shape[0], len(y)
    i = j = 0
    total = 0.0
    p = 0
    path = list(path)
    while p < len(path):
        op = path[p]
        if op == OP_M:
            total += cost[i][y[j]]; i += 1; j += 1; p += 1
            continue
        q = p
        while q < len(path) and path[q] == op:
            q += 1
        L = q - p
        if op == OP_X:                              # L profile columns against gaps placed after residue j
            term = j == 0 or j == n2
            total -= (To if term else Go) + (L - 1) * (Te if term else Ge)
            i += L
        else:                                       # L residues against gap columns placed after column i
            term = i == 0 or i == n1
            total -= nseq * ((To if term else Go) + (L - 1) * (Te if term else Ge))
            j += L
        p = q
    assert i == n1 and j == n2, "not a complete path"
    return total


def all_paths(n1, n2):
    """Every monotone path from (0, 0) to (n1, n2) over the operations M, X, Y (tiny inputs only)."""
    out = []

    def rec(i, j, acc):
        if i == n1 and j == n2:
            out.append(tuple(acc)); return
        if i < n1 and j < n2:
            rec(i + 1, j + 1, acc + [OP_M])
        if i < n1:
            rec(i + 1, j, acc + [OP_X])
        if j < n2:
            rec(i, j + 1, acc + [OP_Y])
    rec(0, 0, [])
    return out
