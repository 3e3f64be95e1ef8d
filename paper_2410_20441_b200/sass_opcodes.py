"""Per-kernel SASS opcode histogram of libdr.so: the evidence that the hot kernels are TMA / mbarrier code
(UTMALDG = cp.async.bulk.tensor, UBLKCP = cp.async.bulk, SYNCS = mbarrier ops, MUFU.RCP64H = fp64 reciprocal seed).

    python -m paper_2410_20441_b200.sass_opcodes > profiles/rN_sass_opcodes.txt
"""
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
WATCH = ("UTMALDG", "UTMASTG", "UBLKCP", "SYNCS", "DFMA", "DADD", "DMUL", "MUFU.RCP64H", "LDS", "STS", "LDG", "STG", "BAR", "ATOMG", "SHFL")


def main():
    lib = os.path.join(HERE, "libdr.so")
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    print("# command: cuobjdump -sass paper_2410_20441_b200/libdr.so | (per-function opcode count); python -m paper_2410_20441_b200.sass_opcodes")
    from paper_2410_20441_b200 import build
    print("# kernel source hash: %s" % build.source_hash())
    print("# columns: kernel, total SASS instructions, then counts of: " + " ".join(WATCH))
    name, counts, total = None, collections.Counter(), 0

    def flush():
        if name is not None:
            dem = subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip() or name
            cut = dem.rfind(">(")
            dem = (dem[:cut + 1] if cut >= 0 else dem.split("(")[0]).replace("void ", "").replace("(int)", "").replace("(bool)", "")
            print("%-58s %6d  " % (dem, total) + " ".join("%s=%d" % (w, counts[w]) for w in WATCH if counts[w]))

    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            flush()
            name, counts, total = m.group(1), collections.Counter(), 0
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m:
            op = m.group(1)
            total += 1
            for w in WATCH:
                if op == w or op.startswith(w + ".") or (w == "MUFU.RCP64H" and op.startswith("MUFU.RCP64H")):
                    counts[w] += 1
    flush()


if __name__ == "__main__":
    sys.exit(main())
