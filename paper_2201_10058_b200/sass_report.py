"""Reads the per-pair FP64 instruction and flop count of the dense pair loop off the SASS of the
built library (north_star: "a per-pair flop count read off the committed SASS").

    python -m paper_2201_10058_b200.sass_report > profiles/sass_pair_loop_r01.md

Dumps `kick_kernel<256, 2, 256, 2, STAGES>` (the level-0 pair loop) with cuobjdump, finds the innermost loops that
issue FP64 arithmetic (a backward branch whose body holds no other loop with FP64 instructions),
and prints for each the instruction mix, the pairs per trip (MUFU.RSQ64H count: one seed per
pair) and the listing.  No GPU needed.
"""
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libgenga_kick.so")
CUOBJDUMP = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")
FP64 = ("DADD", "DMUL", "DFMA")
FLOPS = {"DADD": 1, "DMUL": 1, "DFMA": 2}


def dense_kernel_sass():
    out = subprocess.run([CUOBJDUMP, "-sass", LIB], check=True, capture_output=True, text=True).stdout
    blocks = re.split(r"\n\s*Function : ", out)
    for b in blocks[1:]:
        name = b.split("\n", 1)[0].strip()
        if re.search(r"kick_kernelILi256ELi2ELi256ELi2ELi\d+EE", name):
            return name, b
    raise RuntimeError("kick_kernel<256, 2, 256, 2, STAGES> not found in " + LIB)


def parse(block):
    ins = []
    for line in block.splitlines():
        m = re.search(r"/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    return ins


def opcode(text):
    return re.sub(r"^@!?U?P\d+\s+", "", text).split()[0]


def innermost_loops(ins):
    back = []
    for addr, text in ins:
        m = re.search(r"\bBRA(?:\.\S+)?\s+(?:\S+,\s*)?(0x[0-9a-f]+)", text)
        if m and int(m.group(1), 16) <= addr:
            back.append((int(m.group(1), 16), addr))
    def n64(a, b):
        return sum(opcode(t) in FP64 for x, t in ins if a <= x <= b)
    loops = []
    for a, b in sorted(set(back)):
        inner = [(a2, b2) for a2, b2 in back if (a2, b2) != (a, b) and a <= a2 and b2 <= b]
        if n64(a, b) and not any(n64(a2, b2) for a2, b2 in inner):
            loops.append((a, b))
    return loops


def main():
    name, block = dense_kernel_sass()
    ins = parse(block)
    print("# SASS of the dense pair loop: FP64 instructions and flops per ordered pair\n")
    print("Written by `python -m paper_2201_10058_b200.sass_report` from `cuobjdump -sass` of the built")
    print("`libgenga_kick.so` (sm_100a).  Kernel: `" + name + "`.\n")
    for a, b in innermost_loops(ins):
        body = [(x, t) for x, t in ins if a <= x <= b]
        mix = collections.Counter(opcode(t) for _, t in body)
        n64 = sum(mix[o] for o in FP64)
        pairs = mix["MUFU.RSQ64H"]
        if n64 < 8 or pairs == 0:
            continue
        flops = sum(mix[o] * FLOPS[o] for o in FP64)
        checked = any(o.startswith(("VOTE", "REDUX")) for o in mix) or mix["ISETP.GE.AND"] + mix["ISETP.LT.AND"] > 2
        three = 0
        for _, t in body:
            if opcode(t) == "DFMA":
                regs = {r.lstrip("-|").split(".")[0].rstrip("|") for r in re.findall(r"[-|]?\bR\d+(?:\.reuse)?\|?", t.split(None, 1)[1])[1:]}
                three += len(regs) >= 3
        kind = "checked loop (groups the box test has not cleared: filter compare on the integer pipe)" if checked \
            else "bare loop (groups the box test has cleared: 98.8 % of the (warp, group) combinations of config 3)"
        print(f"## loop 0x{a:04x}..0x{b:04x}: {kind}\n")
        print(f"* {len(body)} instructions per trip, {pairs} ordered pairs per trip (one MUFU.RSQ64H each)")
        print(f"* FP64 pipe: DADD {mix['DADD']}, DMUL {mix['DMUL']}, DFMA {mix['DFMA']} = {n64} instructions, {flops} flops")
        print(f"* **per pair: {n64 / pairs:g} FP64-pipe instructions ({mix['DADD'] / pairs:g} DADD + {mix['DMUL'] / pairs:g} DMUL + "
              f"{mix['DFMA'] / pairs:g} DFMA), {flops / pairs:g} flops**")
        print(f"* DFMAs with three distinct register operands (3 issue cycles instead of 2 on this part): {three} "
              f"= {three / pairs:g} per pair")
        other = {o: c for o, c in sorted(mix.items()) if o not in FP64}
        print(f"* other pipes: {other}\n")
        print("```")
        for x, t in body:
            print(f"/*{x:04x}*/  {t}")
        print("```\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
