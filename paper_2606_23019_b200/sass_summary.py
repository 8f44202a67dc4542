"""Opcode counts of the built library's kernels (evidence that the hot kernels are Blackwell-native).

    python -m paper_2606_23019_b200.sass_summary [> profiles/rN_sass_summary.md]

Runs `cuobjdump -sass` on the in-tree libscalingattn.so and prints, per kernel, the number of SASS
instructions and of the mnemonics that matter here: UTCHMMA (tcgen05.mma), LDTM / STTM (tcgen05.ld /
st), UTMALDG (TMA load), HMMA (mma.sync), MUFU.EX2, R2UR and ELECT (what an MMA / TMA issue costs
beyond the instruction itself), BAR / SYNCS (barriers), STL / LDL (local-memory spills)."""
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libscalingattn.so")
CUOBJDUMP = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")
OPS = ["UTCHMMA", "LDTM", "STTM", "UTMALDG", "HMMA", "MUFU.EX2", "R2UR", "ELECT", "SYNCS", "BAR", "STL", "LDL"]


def demangle_short(name: str) -> str:
    """`fwd_tcgen05_kernel<false>` from the mangled symbol (c++filt, then the last name component)."""
    try:
        full = subprocess.run(["c++filt", name], capture_output=True, text=True, check=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return name[:60]
    m = re.search(r"(\w+_kernel(?:<[^>]*>)?)\(", full)
    short = m.group(1) if m else full[:60]
    return short.replace("(bool)0", "false").replace("(bool)1", "true")


def main() -> int:
    if not os.path.exists(LIB):
        print(f"{LIB} missing: run `python -m paper_2606_23019_b200.build`", file=sys.stderr)
        return 1
    out = subprocess.run([CUOBJDUMP, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    kernels, cur = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = demangle_short(m.group(1))
            kernels[cur] = {"n": 0, **{op: 0 for op in OPS}}
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if cur and m:
            k = kernels[cur]
            k["n"] += 1
            op = m.group(1)
            for name in OPS:
                if op == name or op.startswith(name + "."):
                    k[name] += 1
    print("# SASS opcode counts per kernel of libscalingattn.so (sm_100a)\n")
    print("Command: `python -m paper_2606_23019_b200.sass_summary` (runs `cuobjdump -sass` on the in-tree "
          "library built by `python -m paper_2606_23019_b200.build`).\n")
    print("| kernel | instr | KB | " + " | ".join(OPS) + " |")
    print("|---|---:|---:|" + "---:|" * len(OPS))
    for name, k in sorted(kernels.items(), key=lambda kv: -kv[1]["n"]):
        print(f"| `{name}` | {k['n']} | {k['n'] * 16 / 1024:.1f} | " + " | ".join(str(k[o]) for o in OPS) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
