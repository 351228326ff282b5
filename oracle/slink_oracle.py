"""Single-linkage guide tree oracle (stage II) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The paper builds the guide tree by single linkage over the stage-I similarities, computed
incrementally with SLINK so that rows can be discarded as they are consumed.
SLINK itself is not printed in the paper; it reaches exactly the single-linkage dendrogram, which
has a plain definition, so the oracle is that definition written out:

    start with k singleton clusters; k-1 times, merge the two clusters X, Y whose linkage
    similarity  max_{x in X, y in Y} similarity(x, y)  is highest.

Plain numpy, O(k^3); for small k only.  Shares nothing with paper_1603_06958_b200/csrc.
What is unique when similarities tie is the sequence of merge similarities (sorted descending) and
the partition into clusters at any threshold that is not itself a tie value; the merge order among
equal similarities is not (R19).  Ties here are broken by lowest cluster index.

Pins (tests/test_slink_pins.py): scipy.cluster.hierarchy.linkage(method="single") on rank-transformed
distances, brute-force bottleneck (max-min path) similarities on tiny graphs, a hand example.
"""
import numpy as np


def full_matrix(k, lcs_rows_sim):
    """Packed-triangular rows (entry (i, j<i) at i(i-1)/2 + j) -> symmetric k x k matrix, diagonal -inf."""
    S = np.full((k, k), -np.inf, dtype=np.float64)
    ii, jj = np.tril_indices(k, -1)
    S[ii, jj] = lcs_rows_sim
    S[jj, ii] = lcs_rows_sim
    return S


def single_linkage(S):
    """S: symmetric k x k similarity matrix (diagonal ignored).  Returns merges as a list of
    (a, b, sim, size) with scipy-style ids: leaves 0..k-1, the t-th merge creates cluster k + t;
    a < b.  Highest similarity first; ties by lowest (a, b) among the current cluster ids."""
    S = np.array(S, dtype=np.float64, copy=True)
    k = S.shape[0]
    np.fill_diagonal(S, -np.inf)
    ids = list(range(k))            # current cluster id of each active slot
    size = [1] * k
    active = list(range(k))         # slots still alive
    merges = []
    for t in range(k - 1):
        best, bi, bj = None, -1, -1
        for x in range(len(active)):
            for y in range(x + 1, len(active)):
                s = S[active[x], active[y]]
                key = (-s, min(ids[active[x]], ids[active[y]]), max(ids[active[x]], ids[active[y]]))
                if best is None or key < best:
                    best, bi, bj = key, active[x], active[y]
        s = S[bi, bj]
        a, b = sorted((ids[bi], ids[bj]))
        merges.append((a, b, float(s), size[bi] + size[bj]))
        # linkage similarity of the union to every other cluster: the max of the two (single linkage)
        S[bi, :] = np.maximum(S[bi, :], S[bj, :])
        S[:, bi] = S[bi, :]
        S[bi, bi] = -np.inf
        size[bi] += size[bj]
        ids[bi] = k + t
        active.remove(bj)
    return merges


def merge_heights(merges):
    """The unique part under ties: merge similarities, sorted descending."""
    return np.array(sorted((m[2] for m in merges), reverse=True), dtype=np.float64)


def cut(merges, k, threshold):
    """Partition of the k leaves after applying every merge with similarity > threshold, as a
    canonical label array (label = smallest leaf of the cluster)."""
    parent = list(range(2 * k - 1))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x
    for t, (a, b, s, _) in enumerate(merges):
        if s > threshold:
            parent[find(a)] = k + t
            parent[find(b)] = k + t
    roots = {}
    labels = np.zeros(k, dtype=np.int64)
    for leaf in range(k):
        r = find(leaf)
        roots.setdefault(r, leaf)
        labels[leaf] = roots[r]
    return labels


def dendrogram_pair_heights(k, id_a, id_b, sim, qi, qj):
    """For leaf pairs (qi[q], qj[q]), qi != qj: the merge similarity at which the two leaves first share a
    cluster, i.e. the similarity of their lowest common ancestor in the dendrogram given as k-1 merges
    (merge t joins clusters id_a[t], id_b[t] into cluster k + t; scipy ids).  For a single-linkage dendrogram
    this is the bottleneck (smallest edge) of the path between the leaves in the spanning tree it came from,
    which is what the cycle property of a maximum spanning tree bounds: similarity(i, j) <= height(i, j) for
    EVERY pair.  Plain binary lifting over the 2k-1 nodes, vectorised over the queries; any k.
    Pinned in tests/test_slink_pins.py against replaying the merges one by one."""
    k = int(k)
    n = 2 * k - 1
    id_a = np.asarray(id_a, dtype=np.int64)
    id_b = np.asarray(id_b, dtype=np.int64)
    sim = np.asarray(sim, dtype=np.float64)
    parent = np.arange(n, dtype=np.int64)                     # the root is its own parent
    parent[id_a] = k + np.arange(k - 1)
    parent[id_b] = k + np.arange(k - 1)
    depth = np.zeros(n, dtype=np.int64)
    dl, pl = depth.tolist(), parent.tolist()
    for v in range(n - 2, -1, -1):                            # a parent's id is larger than its children's
        dl[v] = dl[pl[v]] + 1
    depth = np.asarray(dl, dtype=np.int64)
    levels = max(1, int(depth.max()).bit_length())
    up = [parent]
    for _ in range(1, levels):
        up.append(up[-1][up[-1]])
    a = np.asarray(qi, dtype=np.int64).copy()
    b = np.asarray(qj, dtype=np.int64).copy()
    swap = depth[a] < depth[b]
    a[swap], b[swap] = b[swap], a[swap]                       # a is the deeper one
    diff = depth[a] - depth[b]
    for j in range(levels):
        m = ((diff >> j) & 1).astype(bool)
        a[m] = up[j][a[m]]
    for j in range(levels - 1, -1, -1):
        m = up[j][a] != up[j][b]
        a[m] = up[j][a[m]]
        b[m] = up[j][b[m]]
    lca = np.where(a == b, a, parent[a])
    assert np.all(lca >= k), "a query pair with qi == qj"
    return sim[lca - k]
