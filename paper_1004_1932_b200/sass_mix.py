"""Instruction mix of the built library, per kernel variant: counts of the SASS mnemonics that show what the hot
kernels are made of (packed FP32 arithmetic FFMA2 / FMUL2 / FADD2, MUFU.RSQ, TMA bulk copies UBLKCP, LDGSTS,
mbarrier SYNCS, register re-allocation USETMAXREG) and of the operand-reuse flags on packed instructions.

    python -m paper_1004_1932_b200.sass_mix [--all] > profiles/<round>_sass_mix.md

Reads `cuobjdump -sass paper_1004_1932_b200/libds.so`; holds no arithmetic of the method.
"""
import re
import subprocess
import sys

from . import build

OPS = ["FFMA2", "FMUL2", "FADD2", "FFMA", "DFMA", "DMUL", "DADD", "MUFU.RSQ", "MUFU.RSQ64H", "LDS", "UBLKCP", "LDGSTS", "SYNCS",
       "USETMAXREG", "SHFL", "REDG", "BAR", "STAS", "UCGABAR_ARV"]


def demangle(names):
    try:
        out = subprocess.run(["cu++filt"] + names, capture_output=True, text=True, check=True).stdout.split("\n")
        return [o.strip() for o in out[:len(names)]]
    except Exception:
        return names


def main():
    lib = build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    parts = re.split(r"\n\s*Function : ", sass)[1:]
    rows = []
    for p in parts:
        name = p.split("\n", 1)[0].strip()
        if "--all" not in sys.argv and not any(k in name for k in ("run_kernel", "pipe_kernel", "cluster_kernel", "cluster_lat_kernel", "small_kernel", "apply_kernel", "avg_")):
            continue
        ins = re.findall(r"/\*[0-9a-f]{4,5}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)([^;]*);", p)
        cnt = {o: 0 for o in OPS}
        packed = reuse = 0
        for op, args in ins:
            base = op.split(".")[0]
            for o in OPS:
                if op == o or op.startswith(o + ".") or (("." not in o) and base == o):
                    cnt[o] += 1
            if base in ("FFMA2", "FMUL2", "FADD2"):
                packed += 1
                reuse += 1 if ".reuse" in args else 0
        rows.append((name, len(ins), cnt, packed, reuse))
    names = demangle([r[0] for r in rows])
    print("| kernel | instr | " + " | ".join(OPS) + " | packed with .reuse |")
    print("|---|---|" + "---|" * (len(OPS) + 1))
    for (name, n, cnt, packed, reuse), dn in zip(rows, names):
        short = dn.replace("void ds::", "")
        k = short.rfind(">(")
        short = short[:k + 1] if k >= 0 else short.split("(")[0]
        print(f"| `{short}` | {n} | " + " | ".join(str(cnt[o]) for o in OPS) + f" | {reuse} / {packed} |")


if __name__ == "__main__":
    main()
