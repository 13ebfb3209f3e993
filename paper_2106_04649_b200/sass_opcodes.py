"""Opcode histogram of every kernel in the built objects (cuobjdump -sass build/libmk/*.o): the evidence that the
contraction kernels use the instructions DESIGN.md says they use (UTCHMMA / LDTM / STTM / UTMALDG for tcgen05, TMEM and
TMA; 256-bit LDG for the streaming GEMV; RED for the accumulations of the fused pass).
`python -m paper_2106_04649_b200.sass_opcodes [object stems ...]` after `python -m paper_2106_04649_b200.build`."""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from .build import OBJ

ALWAYS = re.compile(r"UTC|LDTM|STTM|UTMA|SYNCS|RED|ATOM|LDG|STG|LDS|STS|LDGSTS|SETMAXREG|FENCE|NANOSLEEP|HMMA|ELECT|FFMA|MUFU|PREEXIT|ACQBULK|CCTL")
INSTR = re.compile(r"^\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Za-z0-9_.]*)")


def histogram(obj):
    out = subprocess.run(["cuobjdump", "-sass", str(obj)], capture_output=True, text=True, check=True).stdout
    fn, hists = None, collections.OrderedDict()
    for line in out.splitlines():
        if "Function :" in line:
            fn = line.split("Function :")[1].strip()
            hists[fn] = collections.Counter()
            continue
        m = INSTR.match(line)
        if m and fn:
            hists[fn][m.group(1)] += 1
    return hists


def demangle(name):
    try:
        return subprocess.run(["c++filt", "-p", name], capture_output=True, text=True, check=True).stdout.strip()
    except Exception:
        return name


def main(argv):
    stems = argv or sorted(p.stem for p in OBJ.glob("*.o"))
    for stem in stems:
        for fn, h in histogram(OBJ / (stem + ".o")).items():
            print(f"{stem}.o  {demangle(fn)}  ({sum(h.values())} instructions)")
            shown = [(op, c) for op, c in h.most_common() if c >= 12 or ALWAYS.search(op)]
            print("    " + ", ".join(f"{op} {c}" for op, c in shown))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
