"""Seeded synthetic protein families shaped like the paper's workloads.

This module serves BOTH the CUDA path's tests/bench and the oracle, and therefore holds
none of the method's arithmetic: no LCS, no similarity, no sorting, no bit-vectors, no
residue encoding.  It only draws residues (already as codes 0..24) and mutates them.

The paper measures on HomFam / extHomFam (headline ABC_tran with
k = 415 519).  Those datasets are not available; BASELINE.json's five
`configs` stand in for them and this is their generator (recipe: DESIGN.md "Input
recipe").  Seed = 160306958 + config index.

    seqs, offsets = family(config)          # uint8 codes (0..24), int64 offsets[k+1]
"""
import numpy as np

SEED_BASE = 160306958

# Background residue distribution over codes 0..19 (percent, normalised below); skewed like
# natural proteins: commonest ~10 %, rarest ~1 %.  Codes 20..24 at 2e-5 each.
_BG20 = np.array([8.3, 1.4, 5.5, 6.8, 3.9, 7.1, 2.3, 5.9, 5.8, 9.9,
                  2.4, 4.1, 4.7, 3.9, 5.5, 6.6, 5.3, 6.9, 1.1, 2.9])
_RARE = 2e-5
BACKGROUND = np.concatenate([_BG20 / _BG20.sum() * (1.0 - 5 * _RARE), np.full(5, _RARE)])
_BG_CDF = np.cumsum(BACKGROUND)
_BG_CDF[-1] = 1.0

INDEL_RATE = 0.05      # indel events per site
INDEL_MEAN = 3.0       # geometric length, support >= 1

K = [500, 10_000, 50_000, 100_000, 415_519]


def _draw_bg(rng, n):
    return np.searchsorted(_BG_CDF, rng.random(n), side="right").astype(np.uint8)


def _draw_bg_not(rng, orig):
    """Background residues, each different from orig[i]."""
    out = _draw_bg(rng, orig.size)
    bad = np.flatnonzero(out == orig)
    while bad.size:
        out[bad] = _draw_bg(rng, bad.size)
        bad = bad[out[bad] == orig[bad]]
    return out


def _mutate_batch(rng, parent, d):
    """Mutate `parent` (uint8[n]) once per entry of d (float[m]): m members.

    Walk the parent left to right; at each site, with probability INDEL_RATE start an indel
    event (insertion before the site or deletion from the site on, equal probability, length
    geometric with mean INDEL_MEAN).  Surviving sites are substituted with probability d by
    a background residue different from the original.  Returns (flat codes, lengths[m]).
    """
    m, n = d.size, parent.size
    event = rng.random((m, n)) < INDEL_RATE
    is_del = rng.random((m, n)) < 0.5
    glen = rng.geometric(1.0 / INDEL_MEAN, size=(m, n)).astype(np.int32)
    # deletions: difference array, +1 at s, -1 at s+g
    dstart = event & is_del
    diff = np.zeros((m, n + 1), dtype=np.int32)
    rr, ss = np.nonzero(dstart)
    np.add.at(diff, (rr, ss), 1)
    np.add.at(diff, (rr, np.minimum(ss + glen[rr, ss], n)), -1)
    keep = np.cumsum(diff[:, :n], axis=1) == 0
    ins = np.where(event & ~is_del, glen, 0)
    counts = ins + keep                      # output residues produced at each site
    lengths = counts.sum(axis=1).astype(np.int64)
    total = int(lengths.sum())
    out = _draw_bg(rng, total)               # inserted residues; kept sites overwritten below
    ends = np.cumsum(counts.ravel())         # exclusive end of each (member, site) group
    kflat = np.flatnonzero(keep.ravel())
    site_res = np.broadcast_to(parent, (m, n)).ravel()[kflat]
    sub = rng.random(kflat.size) < np.repeat(d, keep.sum(axis=1))
    site_res = site_res.copy()
    site_res[sub] = _draw_bg_not(rng, site_res[sub])
    out[ends[kflat] - 1] = site_res
    return out, lengths


def _split(flat, lengths):
    offs = np.concatenate([[0], np.cumsum(lengths)])
    return [flat[offs[i]:offs[i + 1]] for i in range(lengths.size)]


def _fit(rng, s, lo, hi):
    """Clip one member to [lo, hi]: truncate if too long, pad with background if too short
    (the bounded-retry redraw happens in the caller; this is its fallback)."""
    if s.size > hi:
        return s[:hi]
    if s.size < lo:
        return np.concatenate([s, _draw_bg(rng, lo - s.size)])
    return s


def _members(rng, parent, d, lo, hi, batch=4096):
    """Members of one family, each clipped to [lo, hi] (redraw up to 4 times if too short)."""
    res = [None] * d.size
    todo = np.arange(d.size)
    for _ in range(5):
        if todo.size == 0:
            break
        redo = []
        for b0 in range(0, todo.size, batch):
            idx = todo[b0:b0 + batch]
            flat, lens = _mutate_batch(rng, parent, d[idx])
            for t, s in zip(idx, _split(flat, lens)):
                if s.size < lo:
                    redo.append(t)
                    res[t] = s
                else:
                    res[t] = s[:hi]
        todo = np.array(redo, dtype=np.int64)
    for t in todo:
        res[t] = _fit(rng, res[t], lo, hi)
    return res


def _resize_segments(rng, s, target):
    """Reach `target` length by 1-3 contiguous segment insertions (background) or deletions
    at random positions (config 4: a 0.05/site indel process alone gives +-5 % spread)."""
    diff = int(target) - s.size
    if diff == 0:
        return s
    nseg = int(rng.integers(1, 4))
    nseg = min(nseg, abs(diff))
    cuts = np.sort(rng.choice(np.arange(1, abs(diff)), size=nseg - 1, replace=False)) if nseg > 1 else np.array([], dtype=np.int64)
    parts = np.diff(np.concatenate([[0], cuts, [abs(diff)]])).astype(np.int64)
    if diff > 0:
        pos = np.sort(rng.integers(0, s.size + 1, size=nseg))
        pieces, prev = [], 0
        for p, g in zip(pos, parts):
            pieces.append(s[prev:p])
            pieces.append(_draw_bg(rng, int(g)))
            prev = p
        pieces.append(s[prev:])
        return np.concatenate(pieces)
    keep = np.ones(s.size, dtype=bool)
    for g in parts:
        p = int(rng.integers(0, max(1, s.size - int(g) + 1)))
        keep[p:p + int(g)] = False
    return s[keep]


def _finish(rng, members):
    """Plant 3 exact duplicate pairs (similarity at indel = 0), shuffle, concatenate."""
    k = len(members)
    if k >= 8:
        picks = rng.choice(k, size=6, replace=False)
        for a, b in picks.reshape(3, 2):
            members[b] = members[a].copy()
    order = rng.permutation(k)
    members = [members[t] for t in order]
    lens = np.array([s.size for s in members], dtype=np.int64)
    offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    seqs = np.concatenate(members).astype(np.uint8) if k else np.zeros(0, np.uint8)
    return seqs, offsets


def family(config, k=None, seed=None):
    """Synthetic family for BASELINE.json config index 0..4.  `k` overrides the member count
    (same recipe, smaller set: parity tests); `seed` overrides SEED_BASE + config."""
    if config not in range(5):
        raise ValueError("config must be 0..4")
    k = K[config] if k is None else int(k)
    rng = np.random.default_rng(SEED_BASE + config if seed is None else seed)
    if config == 0:
        # one ancestor of length 300, d = 0.30 for all, lengths clipped 50-600
        anc = _draw_bg(rng, 300)
        members = _members(rng, anc, np.full(k, 0.30), 50, 600)
    elif config == 1:
        # 20 ancestors, lengths N(350, 80) clipped 50-1000; family d ~ U[0.10, 0.50]
        alen = np.clip(np.rint(rng.normal(350, 80, 20)), 50, 1000).astype(int)
        ancs = [_draw_bg(rng, n) for n in alen]
        fd = rng.uniform(0.10, 0.50, 20)
        fam = rng.integers(0, 20, k)
        members = [None] * k
        for f in range(20):
            idx = np.flatnonzero(fam == f)
            for t, s in zip(idx, _members(rng, ancs[f], np.full(idx.size, fd[f]), 50, 1000)):
                members[t] = s
    elif config == 2:
        # 90 % short (100-400), 10 % long (1500-4000); 90 short + 10 long ancestors
        alen = np.concatenate([rng.integers(100, 401, 90), rng.integers(1500, 4001, 10)])
        ancs = [_draw_bg(rng, int(n)) for n in alen]
        fd = rng.uniform(0.10, 0.50, 100)
        is_long = rng.random(k) < 0.10
        fam = np.where(is_long, rng.integers(90, 100, k), rng.integers(0, 90, k))
        members = [None] * k
        for f in range(100):
            idx = np.flatnonzero(fam == f)
            lo, hi = (1500, 4000) if f >= 90 else (100, 400)
            for t, s in zip(idx, _members(rng, ancs[f], np.full(idx.size, fd[f]), lo, hi)):
                members[t] = s
    elif config == 3:
        # one ancestor of length 250, per-member d ~ U[0.20, 0.60]; 2 % fragments
        anc = _draw_bg(rng, 250)
        members = _members(rng, anc, rng.uniform(0.20, 0.60, k), 10, 65535)
        frag = np.flatnonzero(rng.random(k) < 0.02)
        for t in frag:
            s = members[t]
            n = max(10, int(round(s.size * rng.uniform(0.20, 0.40))))
            n = min(n, s.size)
            p = int(rng.integers(0, s.size - n + 1))
            members[t] = s[p:p + n].copy()
    else:
        # one ancestor of length 300, per-member d ~ U[0.10, 0.70]; target length lognormal
        # (mu = ln 300 - sigma^2/2, sigma = 0.35) clipped 30-3000, reached by segment indels
        anc = _draw_bg(rng, 300)
        members = _members(rng, anc, rng.uniform(0.10, 0.70, k), 1, 65535)
        sigma = 0.35
        tgt = np.clip(np.rint(rng.lognormal(np.log(300) - sigma * sigma / 2, sigma, k)), 30, 3000)
        members = [_fit(rng, _resize_segments(rng, s, t), 30, 3000) for s, t in zip(members, tgt)]
    return _finish(rng, members)


def sample_pairs(k, n, seed, lengths_sorted=None, block_rows=1024):
    """Seeded pair sample (i, j < i) in SORTED index space: n uniform pairs plus the strata a
    uniform sample would miss: longest x longest (top-left corner), shortest
    (bottom rows), pairs on row-block boundary rows, and -- if `lengths_sorted` is given --
    rows whose length is 0, 1 or 31 mod 32.  Returns unique (i, j) int64 arrays."""
    rng = np.random.default_rng(seed)
    if k < 2:
        z = np.zeros(0, np.int64)
        return z, z
    i = rng.integers(1, k, n)
    j = (rng.random(n) * i).astype(np.int64)
    extra_i, extra_j = [i], [j]
    m = min(k, 46)                                   # ~1000 longest x longest pairs
    a, b = np.tril_indices(m, -1)
    extra_i.append(a.astype(np.int64)); extra_j.append(b.astype(np.int64))
    extra_i.append(k - 1 - b.astype(np.int64)); extra_j.append(k - 1 - a.astype(np.int64))
    for r in range(block_rows - 1, k, block_rows):   # boundary rows r and r+1
        for rr in (r, r + 1):
            if 1 <= rr < k:
                jj = rng.integers(0, rr, 8)
                extra_i.append(np.full(8, rr, np.int64)); extra_j.append(jj)
    if lengths_sorted is not None:
        ls = np.asarray(lengths_sorted)
        for res in (0, 1, 31):
            rows = np.flatnonzero((ls % 32 == res) & (np.arange(k) > 0))
            if rows.size:
                rows = rng.choice(rows, size=min(rows.size, 64), replace=False)
                extra_i.append(rows.astype(np.int64))
                extra_j.append((rng.random(rows.size) * rows).astype(np.int64))
    i = np.concatenate(extra_i); j = np.concatenate(extra_j)
    key = np.unique(i * k + j)
    return key // k, key % k


# ---- inputs of the sequence-versus-profile DP ---------------------------------
def substitution_matrix(seed=SEED_BASE + 40):
    """A seeded 32 x 32 float32 stand-in for the paper's MIQS matrix (its values are not in
    the paper): symmetric, diagonal 4..9 in quarter steps, off-diagonal -4..2, symbols >= 25 score -1
    against everything.  Only its shape and magnitudes matter here."""
    rng = np.random.default_rng(seed)
    a = rng.integers(-16, 9, (32, 32)).astype(np.float32) / 4.0
    s = np.minimum(a, a.T)
    s[np.arange(32), np.arange(32)] = rng.integers(16, 37, 32).astype(np.float32) / 4.0
    s[25:, :] = -1.0
    s[:, 25:] = -1.0
    return np.ascontiguousarray(s, dtype=np.float32)


def profile_batch(n_align, seed, n1_range=(30, 700), nseq_max=40, lengths=None):
    """n_align independent (profile, sequence) inputs: per alignment an ancestor of n1 residues, a profile of
    nseq members that differ from it by substitutions (and 5 % gap cells), and one more member with
    substitutions AND indels as the sequence (<= 1024 residues).
    `lengths`: optional list of (n1, n2) to force (n2 by cutting / padding the sequence).
    Returns counts uint32 [sum n1][32], col_off int64, seq uint8, seq_off int64, nseq int32, k_total int."""
    rng = np.random.default_rng(seed)
    counts, seqs, col_off, seq_off, nseq = [], [], [0], [0], []
    for b in range(n_align):
        n1 = int(lengths[b][0]) if lengths is not None else int(rng.integers(n1_range[0], n1_range[1] + 1))
        ns = int(rng.integers(1, nseq_max + 1))
        anc = _draw_bg(rng, n1)
        d = float(rng.uniform(0.1, 0.4))
        c = np.zeros((n1, 32), np.uint32)
        for _ in range(ns):                              # profile members: substitutions only, so columns are aligned;
            m = anc.copy()                               # 5 % of the cells are gaps (no symbol counted)
            sub = rng.random(n1) < d
            m[sub] = _draw_bg(rng, int(sub.sum()))
            keep = np.flatnonzero(rng.random(n1) >= 0.05)
            np.add.at(c, (keep, m[keep]), 1)
        flat, lens = _mutate_batch(rng, anc, np.array([d]))   # the sequence: substitutions and indels
        y = flat
        n2 = int(lengths[b][1]) if lengths is not None else int(min(max(y.size, 1), 1024))
        y = np.concatenate([y, _draw_bg(rng, max(0, n2 - y.size))])[:n2]
        counts.append(c); seqs.append(y.astype(np.uint8)); nseq.append(ns)
        col_off.append(col_off[-1] + n1); seq_off.append(seq_off[-1] + n2)
    return (np.concatenate(counts), np.array(col_off, np.int64), np.concatenate(seqs), np.array(seq_off, np.int64),
            np.array(nseq, np.int32))
