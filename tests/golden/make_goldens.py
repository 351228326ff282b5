"""Writes tests/golden/oracle_digests.txt: digests of what the ORACLE computes on the seeded synthetic
sets (calls only oracle/ and the shared input generator; never the CUDA path).  Re-run by hand only when
the generator recipe or a reading of the paper changes, and say why in the commit message.

    python tests/golden/make_goldens.py
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

CASES = [(0, 500, None), (1, 300, 77), (2, 120, 91), (3, 250, 93), (4, 200, 5)]   # (config, k, seed)


def digest(config, k, seed):
    from oracle import famsa_oracle
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(config, k=k, seed=seed)
    lcs, sim = famsa_oracle.rows(seqs, offsets, 0, k)
    h = hashlib.sha256(np.ascontiguousarray(lcs, dtype="<i4").tobytes()).hexdigest()
    fin = np.isfinite(sim)
    return "%d %d %s %d %s %d %d %.12e" % (config, k, "default" if seed is None else seed, int(seqs.size), h,
                                           int(lcs.sum()), int((~fin).sum()), float(sim[fin].sum()))


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_digests.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_goldens.py from oracle/ only (plain-DP LCS, PAPER.md:40-46)\n")
        f.write("# config k seed residues sha256(int32 LCS rows, packed triangular, sorted index space) sum(LCS) n_inf sum(finite similarity)\n")
        for c in CASES:
            f.write(digest(*c) + "\n")
    print(open(out).read())
