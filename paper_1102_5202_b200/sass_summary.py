"""Static summary of the built CUDA library: per kernel the registers, stack and SASS instruction counts that show
what the hardware is asked to do (UTMALDG = TMA tensor loads, SYNCS = mbarrier operations, DFMA/DMUL/DADD = fp64
pipe, FFMA2/FMUL2/FADD2 = packed fp32, LDL/STL = local-memory spills).  Needs no GPU:

    python -m paper_1102_5202_b200.sass_summary > profiles/r02_sass.txt
"""
import collections
import re
import subprocess
import sys

from .build import LIB, build

OPS = ["UTMALDG", "SYNCS", "DFMA", "DMUL", "DADD", "DSETP", "FFMA2", "FMUL2", "FADD2", "FFMA", "FMUL", "FADD", "MUFU",
       "LDS", "STS", "LDG", "STG", "LDL", "STL", "BAR"]


def demangle(name):
    out = subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip()
    if out == name:   # internal linkage (anonymous namespace): nvcc's _GLOBAL__N__<hash>_<file> prefix is not Itanium
        m = re.search(r"_cu_[0-9a-f]{8}\d+(k_[a-z_]+)(I[fd]E)?", name)
        return "(file-local) " + (m.group(1) + {"IfE": "<float>", "IdE": "<double>", None: ""}[m.group(2)] if m else name)
    out = out.replace("(anonymous namespace)::", "")
    return re.sub(r"\(.*", "", out) or name


def main():
    lib = build()
    res = subprocess.run(["cuobjdump", "--dump-resource-usage", lib], capture_output=True, text=True).stdout
    usage, cur = {}, None
    for line in res.splitlines():
        m = re.match(r"\s*Function (\S+):", line)
        if m:
            cur = m.group(1)
        elif cur and "REG:" in line:
            usage[cur] = dict(kv.split(":") for kv in line.split() if ":" in kv and not kv.startswith("CONSTANT"))
            cur = None
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    counts, total, cur = collections.defaultdict(collections.Counter), collections.Counter(), None
    for line in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", line)
        if m and cur:
            total[cur] += 1
            op = m.group(1)
            if op in OPS:
                counts[cur][op] += 1
    print(f"# {lib.split('/')[-1]}: cuobjdump --dump-resource-usage and cuobjdump -sass, instruction counts per kernel")
    print("# (static counts of the SASS text, not executed counts)")
    hdr = ["kernel", "REG", "STACK", "SASS"] + OPS
    print(" | ".join(hdr))
    for f in sorted(total, key=demangle):
        u = usage.get(f, {})
        row = [demangle(f), u.get("REG", "?"), u.get("STACK", "?"), str(total[f])] + [str(counts[f][o]) for o in OPS]
        print(" | ".join(row))
    return 0


if __name__ == "__main__":
    sys.exit(main())
