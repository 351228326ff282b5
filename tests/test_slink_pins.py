"""Pins for the single-linkage oracle (oracle/slink_oracle.py): a library routine on a special
case (scipy single linkage on rank-transformed distances), brute force (max-min path similarity
over all simple paths on tiny graphs), a hand example and invariants."""
import itertools

import numpy as np
import pytest

from oracle import slink_oracle as so


def random_sim(rng, k, levels=None):
    """Symmetric similarity matrix; `levels` forces many exact ties."""
    tri = rng.random(k * (k - 1) // 2) if levels is None else rng.integers(1, levels + 1, k * (k - 1) // 2) / 4.0
    return so.full_matrix(k, tri)


def join_similarity(merges, k):
    """J[x, y] = similarity of the merge at which leaves x and y first share a cluster."""
    members = {i: [i] for i in range(k)}
    J = np.full((k, k), np.nan)
    for t, (a, b, s, size) in enumerate(merges):
        for x in members[a]:
            for y in members[b]:
                J[x, y] = J[y, x] = s
        members[k + t] = members.pop(a) + members.pop(b)
        assert len(members[k + t]) == size
    return J


def maximin_bruteforce(S):
    """Max over all simple paths x -> y of the smallest similarity on the path."""
    k = S.shape[0]
    B = np.full((k, k), np.nan)
    for x in range(k):
        for y in range(x + 1, k):
            others = [z for z in range(k) if z not in (x, y)]
            best = -np.inf
            for n in range(len(others) + 1):
                for mid in itertools.permutations(others, n):
                    path = (x,) + mid + (y,)
                    best = max(best, min(S[path[i], path[i + 1]] for i in range(len(path) - 1)))
            B[x, y] = B[y, x] = best
    return B


def test_hand_example():
    # sims: (1,0)=0.9 (2,0)=0.1 (2,1)=0.5 (3,0)=0.2 (3,1)=0.3 (3,2)=0.8
    S = so.full_matrix(4, np.array([0.9, 0.1, 0.5, 0.2, 0.3, 0.8]))
    m = so.single_linkage(S)
    assert m == [(0, 1, 0.9, 2), (2, 3, 0.8, 2), (4, 5, 0.5, 4)]     # {0,1}, {2,3}, then joined through (2,1)
    assert list(so.cut(m, 4, 0.6)) == [0, 0, 2, 2]


@pytest.mark.parametrize("levels", [None, 3])
def test_bruteforce_maximin(levels):
    rng = np.random.default_rng(5)
    for k in (2, 3, 5, 6):
        for _ in range(4):
            S = random_sim(rng, k, levels)
            J = join_similarity(so.single_linkage(S), k)
            B = maximin_bruteforce(S)
            iu = np.triu_indices(k, 1)
            assert np.array_equal(J[iu], B[iu])


@pytest.mark.parametrize("levels", [None, 5])
def test_against_scipy_single_linkage(levels):
    from scipy.cluster.hierarchy import fcluster, linkage
    from scipy.spatial.distance import squareform
    rng = np.random.default_rng(9)
    for k in (2, 7, 40, 90):
        S = random_sim(rng, k, levels)
        vals = np.unique(S[np.triu_indices(k, 1)])                  # ascending similarities
        rank = {v: float(len(vals) - n) for n, v in enumerate(vals)}  # highest similarity -> distance 1
        D = np.zeros((k, k))
        for x in range(k):
            for y in range(k):
                if x != y:
                    D[x, y] = rank[S[x, y]]
        Z = linkage(squareform(D), method="single")
        m = so.single_linkage(S)
        back = {d: v for v, d in rank.items()}
        assert np.array_equal(so.merge_heights(m), np.array([back[d] for d in Z[:, 2]]))   # Z is ascending in distance
        nv = len(vals)
        for r in sorted({1, max(1, nv // 2), max(1, nv - 1)}):         # cut between two adjacent similarity values
            lab_scipy = fcluster(Z, t=r + 0.5, criterion="distance")   # merges at distance <= r, i.e. similarity >= back[r]
            thr_sim = back[r + 1] if r + 1 in back else -np.inf        # ... i.e. similarity > the next lower value
            lab = so.cut(m, k, thr_sim)
            assert np.array_equal(lab_scipy[:, None] == lab_scipy[None, :], lab[:, None] == lab[None, :])


def test_invariants():
    rng = np.random.default_rng(13)
    S = random_sim(rng, 60, 4)
    m = so.single_linkage(S)
    assert len(m) == 59 and m[-1][3] == 60
    h = np.array([x[2] for x in m])
    assert np.all(h[:-1] >= h[1:])                                    # single linkage is monotone
    used = [x for t in m for x in t[:2]]
    assert sorted(used) == list(range(2 * 60 - 2))                    # every cluster merged exactly once
    # the merge similarities are the edge weights of a maximum spanning tree: compare with Kruskal
    edges = sorted(((S[a, b], a, b) for a in range(60) for b in range(a)), reverse=True)
    parent = list(range(60))
    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]; x = parent[x]
        return x
    w = []
    for s, a, b in edges:
        ra, rb = find(a), find(b)
        if ra != rb:
            parent[ra] = rb; w.append(s)
    assert np.array_equal(so.merge_heights(m), np.array(w))


def test_dendrogram_pair_heights_vs_replaying_the_merges():
    """oracle.slink_oracle.dendrogram_pair_heights (binary-lifting LCA, used by the full-size guide-tree check)
    against the plain definition: replay the merges in order and note when the two leaves first meet."""
    from oracle import slink_oracle as so
    rng = np.random.default_rng(5)
    for k in (2, 3, 9, 40, 130):
        n = k * (k - 1) // 2
        tri = rng.integers(1, 9, n) / 8.0 if k % 2 else rng.random(n)
        merges = so.single_linkage(so.full_matrix(k, tri))
        ia = np.array([m[0] for m in merges]); ib = np.array([m[1] for m in merges]); w = np.array([m[2] for m in merges])
        qi, qj = np.tril_indices(k, -1)
        got = so.dendrogram_pair_heights(k, ia, ib, w, qi, qj)
        cluster = {v: {v} for v in range(k)}
        want = np.full((k, k), np.nan)
        for t, (a, b, s, _) in enumerate(merges):
            for x in cluster[a]:
                for y in cluster[b]:
                    want[x, y] = want[y, x] = s
            cluster[k + t] = cluster.pop(a) | cluster.pop(b)
        assert np.array_equal(got, want[qi, qj])
        # and the single-linkage property itself: every pair's similarity is at most its merge height
        S = so.full_matrix(k, tri)
        assert np.all(S[qi, qj] <= got)
