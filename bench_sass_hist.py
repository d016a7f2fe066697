"""Hot-loop SASS histogram of the built kernels, per integrand evaluation, beside the algorithmic instruction list the
ALU roofline is built from (bench.py ALG_OPS).

    python bench_sass_hist.py            # needs only the built objects (nvcc/cuobjdump, no GPU)

A measurement tool kept beside bench.py, outside the product package, so that profiles/r0N_sass_hist.txt stays
reproducible from a committed command.

For each BASELINE config the kernel bench.py actually launches (AUTO schedule) is disassembled with `cuobjdump -sass`,
its innermost-longest loop (the sample loop) is located by its backward branch, and the opcodes in it are counted and
divided by the evaluations one trip makes.  Classes: integer = everything dispatched at 2 cycles per warp on the main
port (IMAD*, LOP3, SHF, IADD3, VIADD, ISETP, MOV, ...), fp32 = FFMA/FMUL/FADD, fp64 = DFMA/DADD/DMUL, xu = MUFU/F2F/FRND,
uniform = U* (uniform datapath: not a lane instruction).
"""
from __future__ import annotations

import collections
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
OBJ = os.path.join(HERE, "paper_1910_01965_b200", os.environ.get("ZMC_OBJ", "build"))

# config -> (object, substrings of the demangled kernel name, evaluations per loop trip, ALG_OPS (int, fp32, fp64, xu))
KERNELS = {
    "cfg1 (CTA)": ("zmc_inst_c12.o", ["zmc_scan_kernel", "FamC1<double", ", 3>"], 16, (12.5, 0, 15, 0)),
    "cfg2 (THREAD)": ("zmc_inst_c12.o", ["zmc_scan_kernel", "FamC2<double", ", 1>"], 8, (23, 0, 16, 0)),
    "cfg2 (WARP)": ("zmc_inst_c12.o", ["zmc_scan_kernel", "FamC2<double", ", 2>"], 8, (24, 0, 16, 0)),
    "cfg3 (THREAD)": ("zmc_inst_c3.o", ["zmc_scan_kernel", "FamC3<float, 4, true>", ", 1>"], 2, (38, 8, 2, 3)),
    "cfg4 (THREAD)": ("zmc_inst_c45.o", ["zmc_scan_kernel", "FamC4<float, true>", ", 1>"], 2, (57, 13, 2, 2)),
    "cfg5 (THREAD)": ("zmc_inst_c45.o", ["zmc_scan_kernel", "FamC5<float, true>", ", 1>"], 4, (28.5, 18, 2, 4)),
    "eq4 (THREAD)": ("zmc_inst_p6.o", ["zmc_scan_kernel", "FamP6<double, 6", ", 1>"], 4, (65, 0, 20, 0)),
}


def classify(op: str) -> str:
    if op.startswith(("BRA", "BSSY", "BSYNC", "EXIT", "NOP", "WARPSYNC")):
        return "branch"
    if op.startswith("U") and not op.startswith("UTC"):
        return "uniform"
    if op.startswith(("DFMA", "DADD", "DMUL", "DSETP")):
        return "fp64"
    if op.startswith(("MUFU", "F2F", "FRND", "I2F", "F2I")):
        return "xu"
    if op.startswith(("FFMA", "FMUL", "FADD", "FSEL", "FSETP", "FMNMX")):
        return "fp32"
    return "integer"


def loop_of(obj: str, pats):
    txt = subprocess.run(["cuobjdump", "-sass", obj], capture_output=True, text=True, check=True).stdout
    for m in re.finditer(r"Function : (\S+)\n(.*?)(?=\n\s*Function :|\Z)", txt, re.S):
        dem = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip()
        if not all(p in dem for p in pats):
            continue
        ins = []
        for line in m.group(2).splitlines():
            mm = re.match(r"\s*/\*([0-9a-f]{4,5})\*/\s+(@!?U?P\d\s+)?([A-Z0-9_.]+)\s*(.*?);", line)
            if mm:
                ins.append((int(mm.group(1), 16), mm.group(3), mm.group(4)))
        loops = []
        for addr, op, args in ins:
            t = re.search(r"0x([0-9a-f]+)", args) if op.startswith("BRA") else None
            if t and int(t.group(1), 16) < addr:
                loops.append((int(t.group(1), 16), addr))
        a, b = max(loops, key=lambda ab: ab[1] - ab[0])
        return dem, [op for addr, op, _ in ins if a <= addr <= b]
    raise RuntimeError(f"kernel {pats} not found in {obj}")


def main():
    print("# hot-loop SASS per integrand evaluation (cuobjdump -sass of paper_1910_01965_b200/build/*.o, nvcc 12.9, sm_100a)")
    print("# columns: executed in the loop / algorithmic minimum (bench.py ALG_OPS); cost model: every instruction one dispatch slot, an integer lane instruction a second one (DESIGN.md section 6)")
    for name, (obj, pats, evals, alg) in KERNELS.items():
        dem, seq = loop_of(os.path.join(OBJ, obj), pats)
        ops = collections.Counter(seq)
        cls = collections.Counter()
        for op, n in ops.items():
            cls[classify(op)] += n
        per = {k: cls[k] / evals for k in ("integer", "fp32", "fp64", "xu", "uniform", "branch")}
        lane = per["integer"] + per["fp32"] + per["fp64"] + per["xu"] + per["branch"]
        print(f"\n{name}: {dem[:100]}")
        print(f"  loop: {len(seq)} instructions per trip, {evals} evaluations per trip")
        print("  per evaluation: integer %.2f / %.1f   fp32 %.2f / %.0f   fp64 %.2f / %.0f   xu %.2f / %.0f   uniform-datapath %.2f   branch %.2f"
              % (per["integer"], alg[0], per["fp32"], alg[1], per["fp64"], alg[2], per["xu"], alg[3], per["uniform"], per["branch"]))
        print("  dispatch slots %.2f (lane %.2f + uniform %.2f) -> cost model, lane-cycles per evaluation = slots + integer = %.1f"
              % (lane + per["uniform"], lane, per["uniform"], lane + per["uniform"] + per["integer"]))
        print("  opcodes per trip: " + ", ".join(f"{k} {v}" for k, v in sorted(ops.items(), key=lambda kv: -kv[1])))


if __name__ == "__main__":
    main()
