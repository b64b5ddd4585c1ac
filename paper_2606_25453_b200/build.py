"""Build the sm_100a C-ABI libraries in-tree.

  paper_2606_25453_b200/libemugemm.so         the product (no experiment switches, no probe kernels)
  paper_2606_25453_b200/libemugemm_probes.so  the same sources with -DEMUGEMM_PROBES: adds emugemm_dbg_set_flags and the
                                              tensor-pipe probes that bench.py's probe leg uses (include/emugemm.h)

nvcc cross-compiles without a GPU.  An object is rebuilt when the SHA-256 of its source, the headers and the flags
differs from the one recorded beside it (content, not mtime: a fresh checkout or a copied tree rebuilds correctly and a
prebuilt library that does not match the sources is never reused).
Usage: python -m paper_2606_25453_b200.build [--force] [--verbose] [--no-probes]
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libemugemm.so")
OUT_PROBES = os.path.join(HERE, "libemugemm_probes.so")
SOURCES = ["api.cu", "prepass.cu", "gemm_oz1.cu", "gemm_oz2.cu", "crt.cu", "static_ws.cu"]
HEADERS = ["common.cuh", "ptx.cuh", "gemm_common.cuh", "crt_dev.cuh", os.path.join("..", "..", "include", "emugemm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]


def _digest(paths, extra):
    h = hashlib.sha256()
    for p in paths:
        h.update(os.path.basename(p).encode())
        with open(p, "rb") as f:
            h.update(f.read())
    h.update(" ".join(extra).encode())
    return h.hexdigest()


def _read(path):
    try:
        with open(path) as f:
            return f.read().strip()
    except OSError:
        return ""


def _build_variant(out, tag, defines, force, verbose):
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    hdrs = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS if os.path.exists(os.path.join(CSRC, h))]
    flags = NVCC_FLAGS + defines + (["-Xptxas", "-v"] if verbose else [])
    objdir = os.path.join(OBJ, tag)
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src) + ".o")
        want = _digest([src] + hdrs, NVCC_FLAGS + defines)
        if not force and os.path.exists(obj) and _read(obj + ".sha256") == want:
            return obj, False
        r = subprocess.run(["nvcc", *flags, "-c", src, "-o", obj], capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        with open(obj + ".sha256", "w") as f:
            f.write(want)
        return obj, True

    with ThreadPoolExecutor(max_workers=len(srcs)) as ex:
        res = list(ex.map(compile_one, srcs))
    objs = [o for o, _ in res]
    link_want = _digest(objs, ["link"])
    if force or any(c for _, c in res) or not os.path.exists(out) or _read(out + ".sha256") != link_want:
        r = subprocess.run(["nvcc", "-shared", "-o", out, *objs, "-gencode", "arch=compute_100a,code=sm_100a"],
                           capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
        with open(out + ".sha256", "w") as f:
            f.write(link_want)
    return out


def build(force: bool = False, verbose: bool = False, probes: bool = True) -> str:
    with ThreadPoolExecutor(max_workers=2) as ex:
        jobs = [ex.submit(_build_variant, OUT, "product", [], force, verbose)]
        if probes:
            jobs.append(ex.submit(_build_variant, OUT_PROBES, "probes", ["-DEMUGEMM_PROBES"], force, verbose))
        for j in jobs:
            j.result()
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, probes="--no-probes" not in sys.argv))
