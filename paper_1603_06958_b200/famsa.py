"""Thin binding over libfamsa_lcs.so (include/famsa_lcs.h): argument marshalling only.

Same names as the C ABI.  Every step of the path runs in the library's CUDA kernels; torch
supplies device memory and streams.  There is NO CPU fallback: if the library is missing or
no sm_100 device is present, the calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfamsa_lcs.so")

FAMSA_OK, FAMSA_EINVAL, FAMSA_ESYMBOL, FAMSA_ELENGTH, FAMSA_ERANGE, FAMSA_ENOMEM, FAMSA_ECUDA = 0, -1, -2, -3, -4, -5, -6
FAMSA_MAX_LEN = 65535

EXPORTS = ["famsa_pack", "famsa_lcs_rows", "famsa_lcs_rows_host", "famsa_lcs_rows_host_async", "famsa_sync", "famsa_host_mode",
           "famsa_lcs_rows_checksum", "famsa_host_profile", "famsa_host_profile_read", "famsa_pack_profile", "famsa_trim",
           "famsa_rows_pairs", "famsa_rows_cells",
           "famsa_k", "famsa_perm", "famsa_lengths", "famsa_codes", "famsa_match", "famsa_launch_count",
           "famsa_alu_peak", "famsa_mix_peak", "famsa_ctx_set_tuning", "famsa_free", "famsa_strerror", "famsa_last_error",
           "famsa_tree_create", "famsa_tree_update", "famsa_tree_merge_edges", "famsa_tree_edge_count",
           "famsa_tree_edges", "famsa_tree_finish", "famsa_tree_free",
           "famsa_guide_tree", "famsa_guide_forest"]
# include/famsa_profile.h
EXPORTS_PROFILE = ["famsa_profile_costs", "famsa_gap_scale", "famsa_seqprof_workspace", "famsa_seqprof_align",
                   "famsa_seqprof_scores_static"]
FAMSA_SEQPROF_STATIC_MAX = 16384


class FamsaError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("famsa error %d: %s" % (code, text))
        self.code = code


_lib = None


def lib():
    """The loaded C-ABI library.  Raises (never falls back) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libfamsa_lcs.so is not built (run `python -m paper_1603_06958_b200.build`); "
                              "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        L.famsa_pack.restype = i32
        L.famsa_pack.argtypes = [vp, vp, i64, i32, ctypes.POINTER(vp)]
        L.famsa_lcs_rows.restype = i32
        L.famsa_lcs_rows.argtypes = [vp, i64, i64, vp, vp, vp]
        L.famsa_lcs_rows_host.restype = i32
        L.famsa_lcs_rows_host.argtypes = [vp, i64, i64, vp, vp]
        L.famsa_lcs_rows_host_async.restype = i32
        L.famsa_lcs_rows_host_async.argtypes = [vp, i64, i64, vp, vp]
        L.famsa_sync.restype = i32
        L.famsa_sync.argtypes = [vp]
        L.famsa_host_mode.restype = i32
        L.famsa_host_mode.argtypes = [vp, i32]
        L.famsa_rows_pairs.restype = i64
        L.famsa_rows_pairs.argtypes = [i64, i64]
        L.famsa_rows_cells.restype = i32
        L.famsa_rows_cells.argtypes = [vp, i64, i64, ctypes.POINTER(ctypes.c_double)]
        L.famsa_k.restype = i32
        L.famsa_k.argtypes = [vp, ctypes.POINTER(i64)]
        L.famsa_perm.restype = i32
        L.famsa_perm.argtypes = [vp, vp]
        L.famsa_lengths.restype = i32
        L.famsa_lengths.argtypes = [vp, vp]
        L.famsa_codes.restype = i32
        L.famsa_codes.argtypes = [vp, i64, vp]
        L.famsa_match.restype = i32
        L.famsa_match.argtypes = [vp, i64, i32, vp]
        L.famsa_launch_count.restype = i64
        L.famsa_launch_count.argtypes = [vp]
        L.famsa_alu_peak.restype = i32
        L.famsa_alu_peak.argtypes = [i32] + [ctypes.POINTER(ctypes.c_double)] * 3
        L.famsa_mix_peak.restype = i32
        L.famsa_mix_peak.argtypes = [i32] + [ctypes.POINTER(ctypes.c_double)] * 2
        L.famsa_ctx_set_tuning.restype = i32
        L.famsa_ctx_set_tuning.argtypes = [vp, i32, i32, i32]
        L.famsa_lcs_rows_checksum.restype = i32
        L.famsa_lcs_rows_checksum.argtypes = [vp, i64, i64, vp, vp, vp, vp]
        L.famsa_host_profile.restype = i32
        L.famsa_host_profile.argtypes = [vp, i32]
        L.famsa_host_profile_read.restype = i32
        L.famsa_host_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        L.famsa_pack_profile.restype = i32
        L.famsa_pack_profile.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        L.famsa_trim.restype = i32
        L.famsa_trim.argtypes = []
        L.famsa_free.restype = None
        L.famsa_free.argtypes = [vp]
        L.famsa_tree_create.restype = i32
        L.famsa_tree_create.argtypes = [i64, i32, ctypes.POINTER(vp)]
        L.famsa_tree_update.restype = i32
        L.famsa_tree_update.argtypes = [vp, i64, i64, vp, vp]
        L.famsa_tree_merge_edges.restype = i32
        L.famsa_tree_merge_edges.argtypes = [vp, vp, vp, vp, i64]
        L.famsa_tree_edge_count.restype = i64
        L.famsa_tree_edge_count.argtypes = [vp]
        L.famsa_tree_edges.restype = i32
        L.famsa_tree_edges.argtypes = [vp, vp, vp, vp]
        L.famsa_tree_finish.restype = i32
        L.famsa_tree_finish.argtypes = [vp, vp, vp, vp, vp]
        L.famsa_tree_free.restype = None
        L.famsa_tree_free.argtypes = [vp]
        L.famsa_guide_forest.restype = i32
        L.famsa_guide_forest.argtypes = [vp, i64, i64, i64, ctypes.POINTER(vp)]
        L.famsa_guide_tree.restype = i32
        L.famsa_guide_tree.argtypes = [vp, i64, vp, vp, vp, vp]
        L.famsa_profile_costs.restype = i32
        L.famsa_profile_costs.argtypes = [vp, vp, i64, vp, vp]
        L.famsa_gap_scale.restype = ctypes.c_double
        L.famsa_gap_scale.argtypes = [ctypes.c_double] * 3
        L.famsa_seqprof_workspace.restype = i64
        L.famsa_seqprof_workspace.argtypes = [vp, vp, i64]
        L.famsa_seqprof_align.restype = i32
        L.famsa_seqprof_align.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp]
        L.famsa_seqprof_scores_static.restype = i32
        L.famsa_seqprof_scores_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp]
        L.famsa_strerror.restype = ctypes.c_char_p
        L.famsa_strerror.argtypes = [i32]
        L.famsa_last_error.restype = ctypes.c_char_p
        L.famsa_last_error.argtypes = []
        _lib = L
    return _lib


def _check(rc):
    if rc != FAMSA_OK:
        L = lib()
        detail = L.famsa_last_error().decode() or L.famsa_strerror(rc).decode()
        raise FamsaError(rc, detail)


def _ptr(t):
    """Raw pointer of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


class Ctx:
    """Owns a famsa_ctx*.  Use as a context manager or call free()."""

    def __init__(self, handle):
        self.handle = handle

    def free(self):
        if self.handle:
            lib().famsa_free(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.free()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def famsa_pack(seqs, offsets, device=0):
    """seqs: uint8 numpy array / bytes (HOST); offsets: int64[k+1] (HOST).  Returns Ctx."""
    if isinstance(seqs, (bytes, bytearray, str)):
        seqs = np.frombuffer(seqs.encode("ascii") if isinstance(seqs, str) else bytes(seqs), dtype=np.uint8)
    seqs = np.ascontiguousarray(seqs, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    k = offsets.size - 1
    out = ctypes.c_void_p()
    _check(lib().famsa_pack(seqs.ctypes.data if seqs.size else None, offsets.ctypes.data, k, int(device),
                            ctypes.byref(out)))
    return Ctx(out.value)


def famsa_rows_pairs(i0, i1):
    return int(lib().famsa_rows_pairs(int(i0), int(i1)))


def _stream(cuda_stream):
    if cuda_stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return cuda_stream.cuda_stream if hasattr(cuda_stream, "cuda_stream") else cuda_stream


def _check_device_outputs(i0, i1, lcs_out, sim_out):
    n = famsa_rows_pairs(i0, i1)
    for t, size in ((lcs_out, 2), (sim_out, 4)):
        if t is not None:
            assert t.is_cuda and t.is_contiguous() and t.element_size() == size and t.numel() >= n


def famsa_lcs_rows(ctx, i0, i1, lcs_out, sim_out, cuda_stream=None):
    """lcs_out: torch.uint16/int16 CUDA tensor or None; sim_out: torch.float32 CUDA tensor or None
    (each with >= famsa_rows_pairs(i0, i1) elements).  Work is enqueued on cuda_stream (an int
    cudaStream_t, a torch.cuda.Stream, or None = torch's current stream)."""
    _check_device_outputs(i0, i1, lcs_out, sim_out)
    _check(lib().famsa_lcs_rows(ctx.handle, int(i0), int(i1), _ptr(lcs_out), _ptr(sim_out), _stream(cuda_stream)))


def famsa_lcs_rows_checksum(ctx, i0, i1, lcs_out, sim_out, checksum, cuda_stream=None):
    """As famsa_lcs_rows; `checksum` is a CUDA int64/uint64 tensor of >= 2 elements that the call ADDS to:
    [0] += sum of LCS, [1] += sum of the similarities' fp32 bit patterns."""
    _check_device_outputs(i0, i1, lcs_out, sim_out)
    assert checksum.is_cuda and checksum.is_contiguous() and checksum.element_size() == 8 and checksum.numel() >= 2
    _check(lib().famsa_lcs_rows_checksum(ctx.handle, int(i0), int(i1), _ptr(lcs_out), _ptr(sim_out), _ptr(checksum),
                                         _stream(cuda_stream)))


def famsa_lcs_rows_host(ctx, i0, i1, lcs_host, sim_host):
    """HOST outputs: numpy arrays or CPU torch tensors (pinned or pageable), or None."""
    n = famsa_rows_pairs(i0, i1)
    for t, size in ((lcs_host, 2), (sim_host, 4)):
        if t is not None:
            if isinstance(t, np.ndarray):
                assert t.flags.c_contiguous and t.itemsize == size and t.size >= n
            else:
                assert (not t.is_cuda) and t.is_contiguous() and t.element_size() == size and t.numel() >= n
    _check(lib().famsa_lcs_rows_host(ctx.handle, int(i0), int(i1), _ptr(lcs_host), _ptr(sim_host)))


def famsa_lcs_rows_host_async(ctx, i0, i1, lcs_host, sim_host):
    """As famsa_lcs_rows_host, but only enqueues (pinned CPU torch tensors / numpy views of pinned memory);
    results are in the buffers after famsa_sync(ctx)."""
    n = famsa_rows_pairs(i0, i1)
    for t, size in ((lcs_host, 2), (sim_host, 4)):
        if t is None:
            continue
        if isinstance(t, np.ndarray):                     # a numpy VIEW of pinned memory: size-checked like the sync call;
            assert t.flags.c_contiguous and t.itemsize == size and t.size >= n    # pageable memory makes the copies synchronous
        else:
            assert (not t.is_cuda) and t.is_contiguous() and t.element_size() == size and t.numel() >= n
            assert t.is_pinned(), "famsa_lcs_rows_host_async needs pinned host tensors (pageable memory makes the copies synchronous)"
    _check(lib().famsa_lcs_rows_host_async(ctx.handle, int(i0), int(i1), _ptr(lcs_host), _ptr(sim_host)))


def famsa_sync(ctx):
    _check(lib().famsa_sync(ctx.handle))


def famsa_host_mode(ctx, mode=-1):
    """-1 auto (pinned outputs are stored by the kernels directly), 0 always staged, 1 direct or fail."""
    _check(lib().famsa_host_mode(ctx.handle, int(mode)))


def famsa_rows_cells(ctx, i0, i1):
    c = ctypes.c_double()
    _check(lib().famsa_rows_cells(ctx.handle, int(i0), int(i1), ctypes.byref(c)))
    return c.value


def famsa_k(ctx):
    k = ctypes.c_int64()
    _check(lib().famsa_k(ctx.handle, ctypes.byref(k)))
    return k.value


def famsa_perm(ctx):
    out = np.empty(famsa_k(ctx), dtype=np.int64)
    _check(lib().famsa_perm(ctx.handle, out.ctypes.data))
    return out


def famsa_lengths(ctx):
    out = np.empty(famsa_k(ctx), dtype=np.uint32)
    _check(lib().famsa_lengths(ctx.handle, out.ctypes.data))
    return out


def famsa_codes(ctx, s, length):
    out = np.empty(int(length), dtype=np.uint8)
    _check(lib().famsa_codes(ctx.handle, int(s), out.ctypes.data))
    return out


def famsa_match(ctx, s, c, length):
    out = np.empty((int(length) + 31) // 32, dtype=np.uint32)
    _check(lib().famsa_match(ctx.handle, int(s), int(c), out.ctypes.data))
    return out


def famsa_launch_count(ctx):
    return int(lib().famsa_launch_count(ctx.handle))


def famsa_alu_peak(device=0):
    """Returns dict(instr_per_s, instr_per_clk_sm, sm_mhz): the measured INT32 ALU-pipe rate."""
    a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(lib().famsa_alu_peak(int(device), ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return {"instr_per_s": a.value, "instr_per_clk_sm": b.value, "sm_mhz": c.value}


def famsa_mix_peak(device=0):
    """Returns dict(alu_instr_per_clk_sm, sm_mhz): the ceiling of the sweep's instruction mix (3 ALU + 1 LDS)."""
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(lib().famsa_mix_peak(int(device), ctypes.byref(a), ctypes.byref(b)))
    return {"alu_instr_per_clk_sm": a.value, "sm_mhz": b.value}


def famsa_ctx_set_tuning(ctx, rows_per_cta=0, small_job_mode=-1, l2_group_mb=0):
    """Per-ctx tuning knobs (0 / -1 = default); results never depend on them."""
    _check(lib().famsa_ctx_set_tuning(ctx.handle, int(rows_per_cta), int(small_job_mode), int(l2_group_mb)))


def famsa_host_profile(ctx, enable=True):
    _check(lib().famsa_host_profile(ctx.handle, 1 if enable else 0))


def famsa_host_profile_read(ctx):
    out = (ctypes.c_double * 5)()
    _check(lib().famsa_host_profile_read(ctx.handle, out))
    return {"sweep_ms": out[0], "d2h_ms": out[1], "d2h_bytes": out[2], "span_ms": out[3], "chunks": int(out[4])}


def famsa_pack_profile(ctx):
    out = (ctypes.c_double * 4)()
    _check(lib().famsa_pack_profile(ctx.handle, out))
    return {"h2d_encode_ms": out[0], "sort_ms": out[1], "plan_ms": out[2], "build_ms": out[3]}


def famsa_trim():
    _check(lib().famsa_trim())


# ---- stage II consumer: single-linkage guide tree (include/famsa_lcs.h) ----------------------------
class Tree:
    """Owns a famsa_tree*."""

    def __init__(self, handle, k):
        self.handle, self.k, self.rows = handle, int(k), 0

    def free(self):
        if self.handle:
            lib().famsa_tree_free(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.free()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def famsa_tree_create(k, device=0):
    out = ctypes.c_void_p()
    _check(lib().famsa_tree_create(int(k), int(device), ctypes.byref(out)))
    return Tree(out.value, k)


def famsa_tree_update(tree, i0, i1, sim_block, cuda_stream=None):
    """sim_block: float32 CUDA tensor in the famsa_lcs_rows layout for rows [i0, i1)."""
    if cuda_stream is None:
        import torch
        cuda_stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(cuda_stream, "cuda_stream"):
        cuda_stream = cuda_stream.cuda_stream
    if sim_block is not None:
        assert sim_block.is_cuda and sim_block.is_contiguous() and sim_block.element_size() == 4
        assert sim_block.numel() >= famsa_rows_pairs(i0, i1)
    _check(lib().famsa_tree_update(tree.handle, int(i0), int(i1), _ptr(sim_block), cuda_stream))
    tree.rows += int(i1) - int(i0)
    tree._last_block = sim_block          # the call only enqueues: keep the block alive until the next one / a query


def famsa_tree_merge_edges(tree, a, b, sim):
    """HOST arrays: leaves a[e], b[e] (int64) and similarities sim[e] (float32) of the edges to merge in."""
    a = np.ascontiguousarray(a, dtype=np.int64)
    b = np.ascontiguousarray(b, dtype=np.int64)
    sim = np.ascontiguousarray(sim, dtype=np.float32)
    assert a.size == b.size == sim.size
    _check(lib().famsa_tree_merge_edges(tree.handle, a.ctypes.data, b.ctypes.data, sim.ctypes.data, a.size))


def famsa_tree_edge_count(tree):
    return int(lib().famsa_tree_edge_count(tree.handle))


def famsa_tree_edges(tree):
    m = famsa_tree_edge_count(tree)
    a, b, w = np.empty(m, np.int64), np.empty(m, np.int64), np.empty(m, np.float32)
    _check(lib().famsa_tree_edges(tree.handle, a.ctypes.data, b.ctypes.data, w.ctypes.data))
    return a, b, w


def famsa_tree_finish(tree):
    m = max(tree.k - 1, 0)
    a, b, w, s = np.empty(m, np.int64), np.empty(m, np.int64), np.empty(m, np.float32), np.empty(m, np.int64)
    _check(lib().famsa_tree_finish(tree.handle, a.ctypes.data, b.ctypes.data, w.ctypes.data, s.ctypes.data))
    return a, b, w, s


def famsa_guide_tree(ctx, block_rows=0):
    m = max(famsa_k(ctx) - 1, 0)
    a, b, w, s = np.empty(m, np.int64), np.empty(m, np.int64), np.empty(m, np.float32), np.empty(m, np.int64)
    _check(lib().famsa_guide_tree(ctx.handle, int(block_rows), a.ctypes.data, b.ctypes.data, w.ctypes.data, s.ctypes.data))
    return a, b, w, s


def famsa_guide_forest(ctx, block_rows=0, part=0, parts=1):
    """Stages I + II over row blocks part, part + parts, ...: returns the Tree (a forest unless parts == 1)."""
    out = ctypes.c_void_p()
    _check(lib().famsa_guide_forest(ctx.handle, int(block_rows), int(part), int(parts), ctypes.byref(out)))
    t = Tree(out.value, famsa_k(ctx))
    return t


# ---- stage III specialisation: sequence-versus-profile DP (include/famsa_profile.h) ----------------
def famsa_profile_costs(counts, subst, cost, cuda_stream=None):
    """counts: uint32/int32 CUDA tensor [n][32]; subst: float32 CUDA [32][32]; cost: float32 CUDA [n][32] (output)."""
    n = counts.shape[0]
    assert counts.is_cuda and counts.is_contiguous() and counts.element_size() == 4 and counts.shape[1] == 32
    assert subst.is_cuda and subst.is_contiguous() and subst.element_size() == 4 and subst.numel() == 1024
    assert cost.is_cuda and cost.is_contiguous() and cost.element_size() == 4 and cost.numel() >= n * 32
    _check(lib().famsa_profile_costs(_ptr(counts), _ptr(subst), int(n), _ptr(cost), _stream(cuda_stream)))


def famsa_gap_scale(k, g_l=45.0, g_d=7.0):
    return float(lib().famsa_gap_scale(float(k), float(g_l), float(g_d)))


def famsa_seqprof_workspace(col_off, seq_off):
    col_off = np.ascontiguousarray(col_off, dtype=np.int64)
    seq_off = np.ascontiguousarray(seq_off, dtype=np.int64)
    assert col_off.size == seq_off.size >= 1
    n = int(lib().famsa_seqprof_workspace(col_off.ctypes.data, seq_off.ctypes.data, col_off.size - 1))
    if n < 0:
        _check(FAMSA_ELENGTH if "residues" in lib().famsa_last_error().decode() else FAMSA_EINVAL)
    return n


def famsa_seqprof_align(cost, col_off, seq, seq_off, gaps, nseq, score, path=None, path_len=None, workspace=None, cuda_stream=None):
    """cost float32 CUDA [sum n1][32]; col_off / seq_off HOST int64 [B+1]; seq uint8 CUDA; gaps float32 CUDA [B][4];
    nseq int32 CUDA [B]; score float32 CUDA [B] (output); path uint8 CUDA [sum (n1+n2)] / path_len int32 CUDA [B] /
    workspace uint8 CUDA [famsa_seqprof_workspace] for the traceback (all three or none)."""
    col_off = np.ascontiguousarray(col_off, dtype=np.int64)
    seq_off = np.ascontiguousarray(seq_off, dtype=np.int64)
    B = col_off.size - 1
    assert seq_off.size == B + 1
    for t, size in ((cost, 4), (seq, 1), (gaps, 4), (nseq, 4), (score, 4), (path, 1), (path_len, 4), (workspace, 1)):
        assert t is None or (t.is_cuda and t.is_contiguous() and t.element_size() == size)
    assert gaps.numel() >= 4 * B and nseq.numel() >= B and score.numel() >= B
    if path is not None:
        assert path.numel() >= int(col_off[-1] + seq_off[-1]) and path_len.numel() >= B
        assert workspace.numel() >= famsa_seqprof_workspace(col_off, seq_off)
    _check(lib().famsa_seqprof_align(_ptr(cost), col_off.ctypes.data, _ptr(seq), seq_off.ctypes.data, _ptr(gaps), _ptr(nseq), B,
                                     _ptr(score), _ptr(path), _ptr(path_len), _ptr(workspace), _stream(cuda_stream)))


def famsa_seqprof_scores_static(cost, col_off, seq, seq_off, gaps, nseq, score, cuda_stream=None):
    """Score-only famsa_seqprof_align that allocates nothing (scratch in a static device array; at most
    FAMSA_SEQPROF_STATIC_MAX alignments per call; overlapping calls on one GPU race: see include/famsa_profile.h)."""
    col_off = np.ascontiguousarray(col_off, dtype=np.int64)
    seq_off = np.ascontiguousarray(seq_off, dtype=np.int64)
    B = col_off.size - 1
    assert seq_off.size == B + 1
    for t, size in ((cost, 4), (seq, 1), (gaps, 4), (nseq, 4), (score, 4)):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == size
    assert gaps.numel() >= 4 * B and nseq.numel() >= B and score.numel() >= B
    _check(lib().famsa_seqprof_scores_static(_ptr(cost), col_off.ctypes.data, _ptr(seq), seq_off.ctypes.data, _ptr(gaps), _ptr(nseq), B,
                                             _ptr(score), _stream(cuda_stream)))
