"""What the built library actually contains: per-kernel SASS opcode histograms and the hot loops.

    python -m paper_2606_15991_b200.sass_report                 # histogram table of every kernel
    python -m paper_2606_15991_b200.sass_report --loops REGEX   # + the loops around UTCHMMA / UTMALDG of matching kernels

Runs `cuobjdump -sass` on csrc/libtilegemm.so (no GPU needed).  The paper's central claim about its
kernels is that the hot loop carries no bounds checks ("no check in the kernel"; the
17 % cost of leaving them in): `--loops` prints the K loops so that this can be read
off the machine code -- the instructions between a backward branch and its target that contain the
tensor-core (UTCHMMA) or TMA (UTMALDG) instructions, with the watchdog's cold path (globaltimer ..
trap) folded away.
"""
from __future__ import annotations

import argparse
import collections
import re
import subprocess
import sys

from . import build as _build

BLACKWELL = ["UTCHMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UTMASTG", "UTMAPF", "UTMACCTL", "UBLKCP", "SYNCS", "UTCATOMSWS", "HMMA"]
INST = re.compile(r"^\s+/\*([0-9a-f]{4,})\*/\s+(.*?);\s*/\*")


def demangle_short(name: str) -> str:
    try:
        out = subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip()
    except OSError:
        out = name
    out = re.sub(r"\((?:int|bool|unsigned int)\)", "", out)      # (int)2 -> 2
    depth, cut = 0, len(out)
    for i, ch in enumerate(out):                                   # drop the parameter list: first '(' outside <...>
        depth += ch == "<"
        depth -= ch == ">"
        if ch == "(" and depth == 0:
            cut = i
            break
    return out[:cut].replace("void tg::", "").replace("tg::", "")


def parse(lib: str):
    """-> [(mangled name, [(address, instruction text)])]"""
    txt = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    kernels, cur = [], None
    for line in txt.splitlines():
        if "Function :" in line:
            cur = (line.split("Function :")[1].strip(), [])
            kernels.append(cur)
            continue
        m = INST.match(line)
        if m and cur is not None:
            cur[1].append((int(m.group(1), 16), m.group(2).strip()))
    return kernels


def opcode(text: str) -> str:
    t = text.split()
    op = t[1] if t[0].startswith("@") else t[0]
    return op.split(".")[0]


def histogram(insts):
    h = collections.Counter(opcode(t) for _, t in insts)
    pred = sum(1 for _, t in insts if t.startswith("@"))
    return h, pred


def loops_around(insts, needles):
    """Innermost backward-branch loops that contain an instruction whose opcode is in `needles`."""
    addr_index = {a: i for i, (a, _) in enumerate(insts)}
    spans = []
    for i, (a, t) in enumerate(insts):
        m = re.search(r"\bBRA(?:\.\w+)*\s+(?:!?U?P\d,\s*)?0x([0-9a-f]+)", t)
        if not m:
            continue
        tgt = int(m.group(1), 16)
        if tgt <= a and tgt in addr_index:
            j = addr_index[tgt]
            if any(opcode(x) in needles for _, x in insts[j:i + 1]):
                spans.append((j, i))
    # keep innermost spans only
    inner = [s for s in spans if not any(o != s and s[0] <= o[0] and o[1] <= s[1] for o in spans)]
    return inner


def fold_watchdog(body):
    """Replace the bounded-wait cold path (read globaltimer ... trap) by one line."""
    out, i = [], 0
    while i < len(body):
        a, t = body[i]
        if "SR_GLOBALTIMERLO" in t:
            j = i
            while j < len(body) and "BPT.TRAP" not in body[j][1]:
                j += 1
            if j < len(body):
                out.append((a, f"[... {j - i + 1} instructions: mbarrier retry with the 4 s watchdog (globaltimer compare, printf, trap) ...]"))
                i = j + 1
                continue
        out.append((a, t))
        i += 1
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--lib", default=_build.LIB)
    ap.add_argument("--loops", metavar="REGEX", help="print the UTCHMMA / UTMALDG loops of kernels whose demangled name matches")
    args = ap.parse_args(argv)
    kernels = parse(args.lib)
    cols = [c for c in BLACKWELL if any(histogram(i)[0].get(c) for _, i in kernels)]
    print("| kernel | instructions | predicated | " + " | ".join(cols) + " |")
    print("|---|---|---|" + "---|" * len(cols))
    total = collections.Counter()
    for name, insts in kernels:
        h, pred = histogram(insts)
        total.update({c: h.get(c, 0) for c in cols})
        print(f"| `{demangle_short(name)}` | {len(insts)} | {pred} | " + " | ".join(str(h.get(c, 0)) for c in cols) + " |")
    print(f"| **all {len(kernels)} kernels** | | | " + " | ".join(str(total[c]) for c in cols) + " |")
    if args.loops:
        rx = re.compile(args.loops)
        for name, insts in kernels:
            short = demangle_short(name)
            if not rx.search(short):
                continue
            for needle, title in ((("UTCHMMA",), "MMA issuer K loop"), (("UTMALDG",), "TMA producer K loop")):
                for (j, i) in loops_around(insts, needle):
                    body = fold_watchdog(insts[j:i + 1])
                    h = collections.Counter(opcode(t) for _, t in body if not t.startswith("[..."))
                    print(f"\n### `{short}`: {title}, 0x{insts[j][0]:04x}..0x{insts[i][0]:04x} "
                          f"({len(body)} lines; compares: {h.get('ISETP', 0)} ISETP, {h.get('UISETP', 0)} UISETP)\n")
                    print("```")
                    for a, t in body:
                        print(f"/*{a:04x}*/  {t}")
                    print("```")
    return 0


if __name__ == "__main__":
    sys.exit(main())
