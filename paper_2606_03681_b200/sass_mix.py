"""Per-kernel SASS opcode histogram of libtabattn.so: the evidence that the shipped kernels use the Blackwell
paths (UTC*MMA = tcgen05.mma, LDTM/STTM = tcgen05.ld/st, UTMALDG/UTMASTG/UBLKCP = TMA; HMMA would be the legacy
mma.sync path).  Reads ``cuobjdump -sass`` text on stdin and prints a markdown table:

    cuobjdump -sass paper_2606_03681_b200/libtabattn.so | python -m paper_2606_03681_b200.sass_mix
"""
import collections
import re
import subprocess
import sys

OPS = ["UTCHMMA", "UTCBAR", "UTMALDG", "UTMASTG", "UBLKCP", "LDTM", "STTM", "HMMA", "MUFU.EX2", "MUFU.RCP", "FFMA2",
       "FADD2", "FMUL2", "F2FP", "LDGSTS", "STG", "LDG", "STS", "LDS", "SYNCS", "STL", "LDL"]


def demangle(name):
    try:
        d = subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip() or name
    except OSError:
        d = name
    d = re.sub(r"tabattn::(gemm::)?\(anonymous namespace\)::", "", d)
    return re.sub(r"\(.*", "", d).replace("void ", "")


def main():
    fn, counts = None, collections.OrderedDict()
    for line in sys.stdin:
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            fn = m.group(1)
            counts[fn] = collections.Counter()
            continue
        if fn is None:
            continue
        m = re.match(r"\s*/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if not m:
            continue
        op = m.group(1)
        counts[fn]["_total"] += 1
        for o in OPS:
            if op == o or op.startswith(o + ".") or (o.startswith("MUFU.") and op.startswith(o)):
                counts[fn][o] += 1
    print("| kernel | SASS instr | " + " | ".join(OPS) + " |")
    print("|---|---|" + "---|" * len(OPS))
    for fn, c in counts.items():
        print("| `%s` | %d | " % (demangle(fn), c["_total"]) + " | ".join(str(c[o]) for o in OPS) + " |")


if __name__ == "__main__":
    main()
