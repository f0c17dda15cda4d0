"""Count the arithmetic operations of one RK substep per zone with the CPU oracle built on an
operation-counting scalar (tests/opcount/counted_real.h).  Test infrastructure: calls only oracle/.

    python tests/opcount/count_ops.py [n]      (default n = 32: Kerr-Schild sweep at 32^3)

Prints adds, muls, divs, sqrts, compares and abs/min/max per zone and substep for each Runge-Kutta
stage, and the flop totals used in DESIGN.md section 5 (FMA not assumed: add and mul count 1 each).
"""
import ctypes as C
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)


def build_counting_oracle():
    out = os.path.join(tempfile.gettempdir(), "libhzo_count.so")
    cmd = ["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-DHZO_CUSTOM_REAL", "-DHZO_REAL=Counted",
           "-include", os.path.join(HERE, "counted_real.h"), "-I", os.path.join(ROOT, "oracle"),
           "-o", out, os.path.join(ROOT, "oracle", "hzo.cpp")]
    subprocess.check_call(cmd)
    return out


def main():
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 32
    path = build_counting_oracle()
    from oracle import binding as ob
    from oracle import build as obuild
    obuild.build = lambda force=False: path   # load the counting build instead of libhzo.so
    ob._lib = None
    import workloads as wl
    w = wl.kerr_sweep(n)
    o = ob.Oracle(w.n, w.h, w.bc, ob.OracleParams.default(**w.params))
    o.set_metric(w.alpha, w.beta3, w.gamma6)
    o.set_primitives(w.prim8)
    L = ob.lib()
    L.hzo_opcount_read.argtypes = [C.POINTER(C.c_longlong), C.c_int]
    buf = (C.c_longlong * 6)()
    L.hzo_opcount_read(buf, 1)
    names = ["add", "mul", "div", "sqrt", "cmp", "abs/min/max"]
    tot = [0.0] * 6
    for stage in range(3):
        o.substeps(w.dt, 1)
        L.hzo_opcount_read(buf, 1)
        per = [buf[i] / w.ncell for i in range(6)]
        tot = [a + b for a, b in zip(tot, per)]
        print(f"stage {stage}: " + ", ".join(f"{k} {v:.1f}" for k, v in zip(names, per)))
    avg = [t / 3 for t in tot]
    print("mean per zone-substep: " + ", ".join(f"{k} {v:.1f}" for k, v in zip(names, avg)))
    flops = avg[0] + avg[1] + avg[2] + avg[3]
    print(f"flops per zone-substep (add + mul + div + sqrt, each 1): {flops:.0f}")
    print(f"with div and sqrt weighted 8: {avg[0] + avg[1] + 8 * (avg[2] + avg[3]):.0f}")


if __name__ == "__main__":
    main()
