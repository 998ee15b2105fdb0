"""Per-kernel opcode histogram of the built library, from `cuobjdump -sass` (SURVEY.md §4 tier 2: the compile-time check
that the kernels are what DESIGN.md says they are — FFMA2 chains without MUFU, TMA loads, tcgen05 MMAs with TMEM loads).

    python -m paper_2606_29629_b200.sass_summary > profiles/r3_sass_summary.txt

No GPU needed: cuobjdump reads the sm_100a cubin embedded in libtriroof.so.  tests/test_sass.py asserts on the same
histograms.
"""
from __future__ import annotations

import collections
import re
import shutil
import subprocess
import sys

_INSN = re.compile(r"^\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P[0-9T]+\s+)?([A-Z][A-Z0-9_]*(?:\.[A-Za-z0-9_]+)*)")


def _tool(name: str) -> str:
    exe = shutil.which(name) or f"/usr/local/cuda/bin/{name}"
    return exe


def histograms(lib_path: str | None = None) -> dict:
    """-> {demangled kernel name: Counter(mnemonic with modifiers -> count)}"""
    if lib_path is None:
        from . import library_path, lib
        lib()                                            # builds if missing or stale
        lib_path = library_path()
    text = subprocess.run([_tool("cuobjdump"), "-sass", lib_path], check=True, capture_output=True, text=True).stdout
    out, cur = {}, None
    for line in text.splitlines():
        if "Function :" in line:
            cur = line.split("Function :", 1)[1].strip()
            out[cur] = collections.Counter()
            continue
        m = _INSN.match(line)
        if m and cur is not None:
            out[cur][m.group(1)] += 1
    names = list(out)
    dem = subprocess.run([_tool("c++filt")] + names, check=True, capture_output=True, text=True).stdout.splitlines() if names else []
    return {d.strip(): out[n] for n, d in zip(names, dem)}


def families(h: collections.Counter, prefix: str) -> int:
    """Instructions whose mnemonic (modifiers included) starts with `prefix`."""
    return sum(c for op, c in h.items() if op.startswith(prefix))


# what is worth a column: the instructions the design claims (or excludes) per kernel
COLUMNS = ["FFMA2", "FFMA", "FMUL", "FADD", "MUFU", "FHFMA", "HMMA", "UTMALDG", "UTMASTG", "UTCHMMA", "LDTM", "UTCBAR", "SYNCS", "LDG", "STG", "LDS", "STS"]


def main() -> int:
    hs = histograms()
    print("# Opcode histogram per kernel of paper_2606_29629_b200/libtriroof.so (sm_100a SASS)")
    print("# command: python -m paper_2606_29629_b200.sass_summary > profiles/r3_sass_summary.txt   (cuobjdump -sass, no GPU)")
    print("# columns count instructions whose mnemonic starts with the name (FFMA excludes FFMA2); `total` = all instructions")
    print("kernel\ttotal\t" + "\t".join(COLUMNS))
    for name in sorted(hs):
        h = hs[name]
        row = []
        for c in COLUMNS:
            v = families(h, c)
            if c == "FFMA":
                v -= families(h, "FFMA2")
            row.append(str(v))
        short = re.sub(r"\(.*", "", name).replace("void ", "")
        print(f"{short}\t{sum(h.values())}\t" + "\t".join(row))
    print("\n# tcgen05 / TMA mnemonics in full, per kernel that has any")
    for name in sorted(hs):
        ops = {op: c for op, c in hs[name].items() if op.startswith(("UTC", "UTMA", "LDTM", "STTM", "UTCBAR"))}
        if ops:
            short = re.sub(r"\(.*", "", name).replace("void ", "")
            print(short + ": " + ", ".join(f"{op} x{c}" for op, c in sorted(ops.items())))
    return 0


if __name__ == "__main__":
    sys.exit(main())
