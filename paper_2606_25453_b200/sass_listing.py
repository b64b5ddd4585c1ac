"""SASS listing of the hot kernels of libemugemm.so (north_star: "a committed SASS listing").

    python -m paper_2606_25453_b200.sass_listing > profiles/r2_sass_listing.txt

Runs `cuobjdump -sass` on the in-tree library (no GPU needed), keeps the kernels named in HOT, drops the hexadecimal
encodings and prints, per kernel, an opcode histogram (tcgen05.mma = UTCIMMA, TMA = UTMALDG / UTMASTG, tcgen05.ld =
LDTM, tcgen05.commit = UTCBAR, dp4a / dp2a = IDP, ...) followed by the instruction stream.
"""
import collections
import os
import re
import subprocess
import sys

from .build import OUT, build

# (label, regex on the demangled name)
HOT = [
    ("fused Scheme I GEMM, p = 8 (N-concatenated, A multicast)", r"oz1_gemm_kernel<8, 0, false, true>"),
    ("fused Scheme I GEMM, p = 3 (cta_group::2 pairs)", r"oz1_gemm_kernel<3, 0, true, false>"),
    ("fused Scheme I GEMM, FP32 output, p = 4", r"oz1_gemm_kernel<4, 1, false, true>"),
    ("Scheme II per-modulus GEMM + mod epilogue (real)", r"oz2_gemm_kernel<1, 0>"),
    ("Scheme II 3M GEMM", r"oz2_gemm_kernel<3, 0>"),
    ("Scheme II GEMM with fused reconstruction, N = 15 / 16", r"oz2_gemm_kernel<1, 8>"),
    ("exact FP64 CRT, N = 15 / 16, real", r"crt_kernel<8, 0>"),
    ("exact FP64 CRT, N = 17 / 18, complex", r"crt_kernel<9, 1>"),
    ("Scheme I row pre-pass, p = 8, default two's-complement digits (register-resident row)", r"planes_rows_reg_kernel<double, 1, 0, 40, 256>"),
    ("Scheme I column pre-pass, p = 8, default two's-complement digits", r"planes_cols_kernel<double, 1, 0, 40, 128>"),
    ("Scheme II row pre-pass (residues, 2 words)", r"planes_rows_kernel<double, 1, 1, 2>"),
    ("Scheme II column pre-pass (residues, 2 words)", r"planes_cols_kernel<double, 1, 1, 2, 128>"),
    ("column maxima", r"colmax_kernel<double, 1>"),
]


def main():
    build()
    names = subprocess.run(["cuobjdump", "-sass", OUT], capture_output=True, text=True).stdout
    mangled = re.findall(r"Function : (\S+)", names)
    dem = subprocess.run(["c++filt"], input="\n".join(mangled), capture_output=True, text=True).stdout.splitlines()
    table = dict(zip(mangled, dem))
    blocks = re.split(r"(?=\s+Function : )", names)
    by_name = {}
    for b in blocks:
        m = re.search(r"Function : (\S+)", b)
        if m:
            by_name[m.group(1)] = b
    print(f"# SASS listing of {os.path.relpath(OUT)} (cuobjdump -sass, sm_100a), hot kernels only; encodings removed")
    print("# command: python -m paper_2606_25453_b200.sass_listing > profiles/r2_sass_listing.txt")
    for label, pat in HOT:
        rx = re.compile(r"\b" + re.escape(pat).replace(r"\ ", r"\s*").replace("bool\\)", "") + r"\(")
        hits = [k for k, v in table.items() if re.search(re.escape(pat).replace(r"\ ", r"\s*"), re.sub(r"\((bool|int)\)", "", v))]
        if not hits:
            print(f"\n## {label}: {pat} -- NOT FOUND")
            continue
        k = hits[0]
        lines = []
        for ln in by_name[k].splitlines():
            m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);\s*/\*", ln)
            if m:
                lines.append((m.group(1), m.group(2).strip()))
        ops = collections.Counter()
        for _, ins in lines:
            t = ins.split()
            op = t[1] if t[0].startswith("@") else t[0]
            ops[op.split(".")[0]] += 1
        print(f"\n## {label}\n## {table[k]}\n## {len(lines)} instructions; opcode histogram:")
        print("## " + ", ".join(f"{o} {c}" for o, c in ops.most_common()))
        ev = {o: c for o, c in ops.items() if o.startswith(("UTC", "UTMA", "LDTM", "STTM", "UBLKCP", "IDP", "DFMA", "SYNCS", "ELECT", "UTCBAR"))}
        print("## Blackwell evidence: " + (", ".join(f"{o} x{c}" for o, c in sorted(ev.items())) or "none (plain CUDA-core kernel)"))
        for addr, ins in lines:
            print(f"{addr}  {ins}")
    return 0


if __name__ == "__main__":
    sys.exit(main())
