"""Issue-cost estimate of a kernel's loops from its SASS (a diagnostic).

    python -m paper_2512_13403_b200.sass_cost --kernel stage_fused2_kernelIfLi0ELi0ELi7ELb1ELb0ELb0E [--lib path/to/libdh.so] [--top 3]

Disassembles the kernel with `cuobjdump -sass`, finds its loops (backward branches) and prints, for the largest ones, the
instruction count, the opcode histogram and the modelled issue cycles per trip under the rule that `dh_issue_probe`
(csrc/dh_probe.cu; `python bench.py --issue-probe`) measures on the B200:

    an instruction occupies a scheduler's issue port for max(1, r / 2) cycles, r = the 32-bit register source operands it
    reads that are not served by the operand-reuse cache (a packed .F32x2 operand counts 2, an immediate, constant-bank or
    uniform-register operand 0), and the half-rate ALU pipe (FMNMX, FSEL, LOP3, integer, compares, moves) for 2 cycles.

Loops are reported with the code they contain, branches not taken included: a bound from above on what one trip executes.
"""
from __future__ import annotations

import argparse
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))

ALU_PIPE = {"FMNMX", "FMNMX3", "FSEL", "LOP3", "FSETP", "ISETP", "IADD3", "MOV", "SEL", "LEA", "SHF", "PRMT", "IADD", "VIADD",
            "IABS", "PLOP3", "FSET", "ISET", "VIMNMX", "IMNMX", "LOP", "POPC", "FLO", "BREV", "SGXT", "BMSK"}
NO_DEST = {"STS", "STG", "ST", "STL", "BAR", "BRA", "LDGSTS", "BSYNC", "BSSY", "NOP", "WARPSYNC", "RED", "ATOMG", "EXIT", "RET",
           "DEPBAR", "LDGDEPBAR", "MEMBAR", "ERRBAR", "CCTL", "UTMALDG", "SYNCS", "ARRIVES"}


def disassemble(lib: str, kernel: str) -> list[tuple[int, str]]:
    """(address, text) of every instruction of the first function whose mangled name contains `kernel`."""
    names = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    full = next((m.group(1) for m in re.finditer(r"Function (\S+?):", names) if kernel in m.group(1)), None)
    if full is None:
        raise SystemExit(f"no function containing '{kernel}' in {lib}")
    out = subprocess.run(["cuobjdump", "-sass", "-fun", full, lib], capture_output=True, text=True).stdout
    ins: list[tuple[int, str]] = []
    for line in out.splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    if not ins:
        raise SystemExit(f"cuobjdump printed no SASS for {full}")
    return ins


def loops(ins: list[tuple[int, str]]) -> list[tuple[int, int]]:
    """(first, last) addresses of the loops, largest first: a branch to a lower address closes one.  The out-of-line blocks
    that BRA.DIV jumps to (divergent-shuffle handlers at the end of the function) return with a backward branch too: those
    are not loops."""
    div_targets = [int(m.group(1), 16) for _, t in ins for m in [re.search(r"\bBRA\.DIV\s+\S+\s+0x([0-9a-f]+)", t)] if m]
    outline = min(div_targets) if div_targets else 1 << 62
    found = []
    for addr, text in ins:
        m = re.search(r"\bBRA(?:\.\w+)*\s+(?:!?U?P\d+,\s*)?(?:UR\d+,\s*)?0x([0-9a-f]+)", text)
        if m and int(m.group(1), 16) < addr < outline:
            found.append((int(m.group(1), 16), addr))
    return sorted(set(found), key=lambda lh: lh[0] - lh[1])


def cost_of(text: str) -> tuple[str, float, bool]:
    """(opcode, issue cycles, runs on the half-rate ALU pipe) of one instruction under the rule in the module docstring."""
    text = re.sub(r"^@!?U?P\d+\s+", "", text)
    op = text.split()[0]
    base = op.split(".")[0]
    ops = [s.strip() for s in text[len(op):].split(",")]
    srcs = ops if base in NO_DEST else ops[1:]
    reads = 0
    for s in srcs:
        for m in re.finditer(r"(?<![U\w])R(\d+|Z)(\.reuse)?((?:\.[A-Za-z0-9_]+)*)", s):
            if m.group(1) == "Z" or m.group(2):
                continue
            wide = "F32x2" in (m.group(3) or "") or (".64" in s and "[" in s)
            reads += 2 if wide else 1
    if base in ("STS", "STG", "STL", "ST"):
        reads += 1 if ".64" in op else 3 if ".128" in op else 0
    return base, max(1.0, reads / 2.0), base in ALU_PIPE


def report(ins, lo: int, hi: int, show: int = 14) -> dict:
    n = 0
    cycles = 0.0
    alu = 0
    per_op: dict[str, list[float]] = collections.defaultdict(lambda: [0, 0.0])
    for addr, text in ins:
        if lo <= addr <= hi:
            base, c, is_alu = cost_of(text)
            n += 1
            cycles += c
            alu += is_alu
            per_op[base][0] += 1
            per_op[base][1] += c
    print(f"loop 0x{lo:x}-0x{hi:x}: {n} instructions ({(hi - lo + 16) / 1024:.1f} KiB), modelled issue cycles per trip {cycles:.1f} "
          f"({cycles / max(n, 1):.3f} per instruction), ALU-pipe instructions {alu} (pipe cycles {2 * alu})")
    for base, (k, c) in sorted(per_op.items(), key=lambda kv: -kv[1][1])[:show]:
        print(f"    {base:<10s} n = {k:4d}   issue cycles = {c:7.1f}")
    return {"instructions": n, "issue_cycles": cycles, "alu_instructions": alu}


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--lib", default=os.path.join(HERE, "libdh.so"))
    ap.add_argument("--kernel", required=True, help="substring of the mangled kernel name")
    ap.add_argument("--top", type=int, default=2, help="how many of the largest loops to report")
    a = ap.parse_args(argv)
    ins = disassemble(a.lib, a.kernel)
    print(f"{a.kernel}: {len(ins)} instructions")
    for lo, hi in loops(ins)[: a.top]:
        report(ins, lo, hi)


if __name__ == "__main__":
    main(sys.argv[1:])
