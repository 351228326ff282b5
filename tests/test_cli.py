"""The FASTA -> guide tree command line: host-side pieces on CPU, the whole thing on the GPU."""
import os
import re

import numpy as np
import pytest

FASTA = """>s1 first
ACDEFGHIKL
MNPQ
>s2
acdefghikl mnpq*
>s3 third one
WWWWYYYY

>s4
ACDEFGHIKLMNPQRSTVWY
"""


def test_read_fasta_and_newick(tmp_path):
    from paper_1603_06958_b200 import cli
    p = tmp_path / "x.fasta"
    p.write_text(FASTA)
    names, seqs, offsets = cli.read_fasta(str(p))
    assert names == ["s1", "s2", "s3", "s4"]
    assert list(np.diff(offsets)) == [14, 14, 8, 20]
    assert bytes(seqs[offsets[1]:offsets[2]]) == b"acdefghiklmnpq"          # blanks and the '*' terminator dropped
    # merges for 4 leaves: (0,1) -> 4, (2,3) -> 5, (4,5) -> 6
    nwk = cli.newick(4, [0, 2, 4], [1, 3, 5], [0.9, 0.5, 0.1], ["a", "b", "c", "d"])
    assert nwk == "((a,b),(c,d));"
    assert cli.newick(4, [0, 2, 4], [1, 3, 5], [0.9, 0.5, 0.1], ["a", "b", "c", "d"], True) == "((a,b):0.9,(c,d):0.5):0.1;"
    assert cli.newick(1, [], [], [], ["only"]) == "only;" and cli.newick(0, [], [], [], []) == ";"
    with pytest.raises(ValueError):
        (tmp_path / "bad.fasta").write_text("ACDE\n>s\nAC\n")
        cli.read_fasta(str(tmp_path / "bad.fasta"))


@pytest.mark.gpu
def test_cli_end_to_end(tmp_path):
    from paper_1603_06958_b200 import build, cli
    build.build()
    p = tmp_path / "x.fasta"
    p.write_text(FASTA)
    out, merges = tmp_path / "t.nwk", tmp_path / "m.tsv"
    assert cli.main([str(p), "-o", str(out), "--merges", str(merges), "--similarities"]) == 0
    nwk = out.read_text().strip()
    assert sorted(re.findall(r"s\d", nwk)) == ["s1", "s2", "s3", "s4"] and nwk.endswith(";")
    assert "(s1,s2):inf" in nwk or "(s2,s1):inf" in nwk                        # s1 == s2 after case folding: merged first
    rows = [l.split("\t") for l in merges.read_text().splitlines()]
    assert len(rows) == 3 and rows[0][2] == "inf" and rows[-1][3] == "4"
