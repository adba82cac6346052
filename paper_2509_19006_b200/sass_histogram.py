"""Per-kernel SASS opcode histogram of the built library: the evidence for "which pipe does this kernel use".

    python -m paper_2509_19006_b200.sass_histogram [--all] > profiles/<name>.md

Runs `cuobjdump -sass` on paper_2509_19006_b200/libtnmc.so and counts, per kernel, the static instructions of the
opcodes that matter here: DMMA (FP64 tensor pipe, mma.sync.m8n8k4.f64), HMMA (TF32 mma.sync), DFMA/DMUL/DADD (FP64
ALU), MUFU, LDGSTS (cp.async), LDG/STG/LDS/STS, SHFL, REDUX, BAR, POPC, UBLKCP (cp.async.bulk: the TMA engine's bulk copy) and
SYNCS (mbarrier operations), UTMALDG/UTMASTG (tensor-map TMA), UTC*MMA (tcgen05.mma), LDTM/STTM (TMEM).  Static counts: how often an instruction executes is ncu's business."""
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
OPS = ["DMMA", "HMMA", "DFMA", "DMUL", "DADD", "MUFU", "LDGSTS", "LDG", "STG", "LDS", "STS", "SHFL", "REDUX", "BAR", "POPC",
       "UBLKCP", "SYNCS", "UTMALDG", "UTMASTG", "UTCHMMA", "UTCQMMA", "LDTM", "STTM"]


def main(show_all):
    lib = os.path.join(HERE, "libtnmc.so")
    txt = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    rows = []
    for f in re.split(r"\n\s*Function : ", txt)[1:]:
        mangled = f.split("\n", 1)[0].strip()
        name = subprocess.run(["c++filt", mangled], capture_output=True, text=True).stdout.strip()
        name = re.sub(r"\(.*", "", name).replace("void ", "").replace("tnmc::", "")
        instr = re.findall(r"^\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\w+\s+)?([A-Z][A-Z0-9_.]*)", f, flags=re.M)
        c = collections.Counter(i.split(".")[0] for i in instr)
        rows.append((name or mangled, len(instr), [c.get(o, 0) for o in OPS]))
    print(f"`cuobjdump -sass paper_2509_19006_b200/libtnmc.so` (sm_100a), static instruction counts per kernel"
          f"{'' if show_all else ' (kernels of the hot path; --all lists every instantiation)'}:\n")
    print("| kernel | instr | " + " | ".join(OPS) + " |")
    print("|---|---|" + "---|" * len(OPS))
    for name, n, cs in sorted(rows, key=lambda r: -r[1]):
        if not show_all and ("true" in name or ", 1>" in name or n < 150 or not name):
            continue      # real-coupling / F32READ / 64-chain instantiations repeat their siblings' mix
        print(f"| `{name}` | {n} | " + " | ".join(str(x) for x in cs) + " |")


if __name__ == "__main__":
    main("--all" in sys.argv)
