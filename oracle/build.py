"""Build the C oracle (TEST INFRASTRUCTURE).  gcc -O2, never tuned.

Called by __graft_entry__.build() ("building the checker is not using it") and lazily by
oracle/famsa_oracle.py.  Output: oracle/libfamsa_oracle.so (git-ignored).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lcs_oracle.c")
SRC_BITPAR = os.path.join(HERE, "bitpar_cpu.c")   # context baseline, not an oracle (see its header)
SRC_PROFILE = os.path.join(HERE, "profile_oracle.c")   # NEXT-4: sequence-vs-profile DP
LIB = os.path.join(HERE, "libfamsa_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(SRC_BITPAR), os.path.getmtime(SRC_PROFILE))):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-O2", "-std=gnu99", "-Wall", "-shared", "-fPIC",
                           "-ffp-contract=off",
                           "-pthread", SRC, SRC_BITPAR, SRC_PROFILE, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
