"""Count the Blackwell-specific SASS mnemonics per kernel family of libcoarseop.so (evidence that the hot
kernels are sm_100a-native: tcgen05 / TMEM / TMA, no legacy HMMA), as a Markdown table under profiles/.

    python -m paper_2212_12559_b200.sass_counts --out profiles/r02_sass_counts.md

Needs `cuobjdump` (CUDA toolkit; no GPU).  PTX -> SASS names (B200_PROFILING.md): tcgen05.mma -> UTC*MMA
(UTCHMMA for kind::tf32, UTCIMMA for kind::i8), tcgen05.commit -> UTCBAR, tcgen05.ld / st -> LDTM / STTM,
cp.async.bulk.tensor -> UTMALDG, cp.async.bulk -> UBLKCP, mbarrier -> SYNCS, fma.rn.f32x2 -> FFMA2.
"""
from __future__ import annotations

import argparse
import collections
import re
import subprocess

from . import build as cuda_build

COLS = ["UTCHMMA", "UTCIMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UBLKCP", "SYNCS", "FFMA2", "HMMA"]
PAT = re.compile(r"\b(" + "|".join(COLS) + r")\b")


def family(mangled: str) -> str:
    m = re.search(r"coarse\d+(coarse_apply_[a-z0-9_]+?)I", mangled)
    if m:
        return m.group(1)
    m = re.search(r"coarse\d+([a-z_0-9]+kernel)", mangled)
    return m.group(1) if m else mangled[:40]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    args = ap.parse_args()
    lib = cuda_build.build_library()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    fam = collections.defaultdict(collections.Counter)
    nk = collections.Counter()
    arch = collections.Counter()
    cur = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = family(m.group(1))
            nk[cur] += 1
            continue
        m = re.search(r"arch = (sm_\w+)", line)
        if m:
            arch[m.group(1)] += 1
        m = PAT.search(line)
        if m and cur:
            fam[cur][m.group(1)] += 1
    lines = ["# Round 2 — SASS mnemonic counts of `libcoarseop.so` per kernel family", "",
             "Command (here, no GPU needed): `python -m paper_2212_12559_b200.sass_counts --out profiles/r02_sass_counts.md`",
             "(= `cuobjdump -sass paper_2212_12559_b200/libcoarseop.so`, instructions counted per `Function :` block and summed",
             "over the template instantiations of a family).  Cubins in the library: " +
             ", ".join(f"{k} x {v}" for k, v in sorted(arch.items())) + ".", "",
             "| kernel family | instantiations | " + " | ".join(COLS) + " |", "|---|---|" + "---|" * len(COLS)]
    tot = collections.Counter()
    for k in sorted(nk, key=lambda k: -sum(fam[k].values())):
        lines.append(f"| `{k}` | {nk[k]} | " + " | ".join(str(fam[k][c]) for c in COLS) + " |")
        tot.update(fam[k])
    lines.append("| **total** | " + str(sum(nk.values())) + " | " + " | ".join(f"**{tot[c]}**" for c in COLS) + " |")
    lines += ["", "Reading: the two tensor-core families issue `tcgen05.mma` (UTCHMMA = kind::tf32 for complex64 links, UTCIMMA =",
              "kind::i8 for int16 links), keep operands and accumulators in tensor memory (STTM / LDTM) and are fed by 2-D TMA",
              "tensor copies (UTMALDG); every streaming family is fed by 1-D TMA bulk copies (UBLKCP) counted on mbarriers",
              "(SYNCS) and does its complex MACs with packed FFMA2.  No legacy `mma.sync` (HMMA) anywhere."]
    with open(args.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print(args.out)


if __name__ == "__main__":
    main()
