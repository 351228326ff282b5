"""Command line: FASTA in, single-linkage guide tree out (stages I + II of FAMSA).

    python -m paper_1603_06958_b200.cli family.fasta -o tree.nwk [--device 0] [--block-rows 1024] [--merges merges.tsv]

File handling and the Newick writer are host-side conveniences; every similarity and every merge is
computed by the CUDA library (famsa_pack -> famsa_guide_tree).  There is no CPU fallback.
The paper defines no branch lengths for the guide tree; with --similarities every internal node carries
its merge similarity in Newick's length field.
"""
import argparse
import sys

import numpy as np


def read_fasta(path):
    """Returns (names, seqs uint8 array of residue letters, offsets int64[k+1]).  Whitespace inside
    sequences is dropped; '*' terminators are dropped; anything else is passed to famsa_pack as is."""
    names, chunks, lens = [], [], []
    cur = []
    with open(path, "rb") as f:
        for line in f:
            line = line.strip()
            if not line:
                continue
            if line.startswith(b">"):
                if names:
                    s = b"".join(cur).replace(b"*", b"")
                    chunks.append(s); lens.append(len(s))
                names.append(line[1:].split()[0].decode("ascii", "replace") if len(line) > 1 else "seq%d" % len(names))
                cur = []
            else:
                if not names:
                    raise ValueError("%s: sequence data before the first '>' header" % path)
                cur.append(bytes(line.translate(None, b" \t\r")))
    if names:
        s = b"".join(cur).replace(b"*", b"")
        chunks.append(s); lens.append(len(s))
    seqs = np.frombuffer(b"".join(chunks), dtype=np.uint8).copy()
    offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    return names, seqs, offsets


def newick(k, id_a, id_b, sim, leaf_names, with_similarity=False):
    """scipy-style merges (cluster k + t = id_a[t] + id_b[t]) -> Newick string.  Iterative (no recursion)."""
    if k == 0:
        return ";"
    if k == 1:
        return leaf_names[0] + ";"
    text = {}
    for t in range(k - 1):
        parts = []
        for c in (int(id_a[t]), int(id_b[t])):
            parts.append(leaf_names[c] if c < k else text.pop(c))
        node = "(" + ",".join(parts) + ")"
        if with_similarity:
            node += ":%.6g" % float(sim[t])
        text[k + t] = node
    return text[2 * k - 2] + ";"


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("fasta")
    ap.add_argument("-o", "--out", default="-", help="Newick file ('-' = stdout)")
    ap.add_argument("--merges", default=None, help="also write the merges as TSV: id_a id_b similarity size")
    ap.add_argument("--device", type=int, default=0)
    ap.add_argument("--block-rows", type=int, default=1024)
    ap.add_argument("--similarities", action="store_true", help="append ':similarity' to every internal node")
    args = ap.parse_args(argv)

    from . import famsa
    names, seqs, offsets = read_fasta(args.fasta)
    k = len(names)
    with famsa.famsa_pack(seqs, offsets, device=args.device) as ctx:
        perm = famsa.famsa_perm(ctx)
        id_a, id_b, sim, size = famsa.famsa_guide_tree(ctx, args.block_rows)
    leaf_names = [names[int(perm[s])].replace("(", "_").replace(")", "_").replace(",", "_").replace(":", "_").replace(";", "_")
                  for s in range(k)]                      # leaves of the tree are SORTED indices: map back through perm
    nwk = newick(k, id_a, id_b, sim, leaf_names, args.similarities)
    if args.out == "-":
        sys.stdout.write(nwk + "\n")
    else:
        with open(args.out, "w") as f:
            f.write(nwk + "\n")
    if args.merges:
        with open(args.merges, "w") as f:
            for t in range(max(k - 1, 0)):
                f.write("%d\t%d\t%.9g\t%d\n" % (id_a[t], id_b[t], sim[t], size[t]))
    return 0


if __name__ == "__main__":
    sys.exit(main())
