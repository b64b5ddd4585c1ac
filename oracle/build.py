"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liboracle.so with gcc.

Plain C + libquadmath + OpenMP; no CUDA, nothing shared with the product path.
Usage: python -m oracle.build   (also called by __graft_entry__.build()).
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "emugemm_oracle.c")
OUT = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-Wall", "-Wextra",
           "-o", OUT, SRC, "-lquadmath", "-lm"]
    # rebuilt when the SHA-256 of the source + command differs from the recorded one (content, not mtime)
    with open(SRC, "rb") as f:
        want = hashlib.sha256(f.read() + " ".join(cmd).encode()).hexdigest()
    stamp = OUT + ".sha256"
    try:
        with open(stamp) as f:
            have = f.read().strip()
    except OSError:
        have = ""
    if not force and os.path.exists(OUT) and have == want:
        return OUT
    subprocess.run(cmd, check=True)
    with open(stamp, "w") as f:
        f.write(want)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
