"""Instruction-level evidence for the resident kernel, read from the built library (no GPU needed).

    python -m paper_0809_3098_b200.sass_report            # markdown report of k_resident<4,6,16,false,0>, the timed variant

Extracts the cubin of cavity_resident.cu from libcavity.so (cuobjdump -xelf), disassembles it with source-line marks
(nvdisasm -g -c; the library is built with -lineinfo) and reports, for one template instance of k_resident:
the opcode histogram of the whole kernel, the flavours of its global / local memory accesses, the source lines the
local-memory (spill) accesses sit on, and every innermost loop of at least 100 instructions with its opcode mix: the
sweep loops of a1 (one per wall class and colour order).  DESIGN.md's "176 instructions per sweep, 120 of them fp64, no
spill in the sweep loops" is this report; tests/test_sass_evidence.py holds the build to it.
"""
import collections
import os
import re
import subprocess
import sys
import tempfile

TIMED_VARIANT = "k_residentILi4ELi6ELi16ELb0ELi0EEE"      # k_resident<C=4, R=6, MAXW=16, FIX=false, KIND=0>: config 3-5's kernel
_INS = re.compile(r"^\s+/\*[0-9a-f]{4,5}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)")


def _base(op):
    return op.split(".")[0]


def disassemble(lib=None):
    """nvdisasm -g -c text of the cavity_resident cubin inside `lib` (default: the in-tree libcavity.so)."""
    if lib is None:
        from .binding import lib_path
        lib = lib_path()
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    with tempfile.TemporaryDirectory() as d:
        subprocess.run([os.path.join(cuda, "bin", "cuobjdump"), "-xelf", "all", os.path.abspath(lib)], cwd=d, check=True,
                       capture_output=True)
        cubins = [f for f in os.listdir(d) if "cavity_resident" in f and f.endswith(".cubin")]
        if len(cubins) != 1:
            raise RuntimeError("expected one cavity_resident cubin in %s, found %r" % (lib, cubins))
        out = subprocess.run([os.path.join(cuda, "bin", "nvdisasm"), "-g", "-c", cubins[0]], cwd=d, check=True,
                             capture_output=True, text=True)
    return out.stdout


def report(sass, variant=TIMED_VARIANT, min_loop=100):
    src = sass.split("\n")
    start = next(i for i, l in enumerate(src) if l.startswith(".text.") and variant in l)
    end = next((i for i in range(start + 1, len(src)) if src[i].startswith("\t.section")), len(src))
    ins, labels, cur = [], {}, None          # ins: (opcode with suffixes, source line, branch target label)
    for l in src[start:end]:
        m = re.match(r'^\s*//## File ".*cavity_resident\.cu", line (\d+)', l)
        if m:
            if "inlined at" not in l:
                cur = int(m.group(1))
            continue
        m = re.match(r"^(\.L_x_\d+):", l)
        if m:
            labels[m.group(1)] = len(ins)
            continue
        m = _INS.match(l)
        if m:
            t = re.search(r"`\((\.L_x_\d+)\)", l)
            ins.append((m.group(1), cur, t.group(1) if t else None))
    hist = collections.Counter(_base(o) for o, _, _ in ins)
    mem = collections.Counter(o for o, _, _ in ins if _base(o) in ("LDG", "STG", "LDL", "STL", "ATOMG", "RED"))
    local_lines = collections.Counter((_base(o), ln) for o, ln, _ in ins if _base(o) in ("LDL", "STL"))
    back = [(labels[t], i) for i, (o, _, t) in enumerate(ins) if _base(o) == "BRA" and t in labels and labels[t] <= i]
    inner = [lp for lp in back if not any(o2 != lp and lp[0] <= o2[0] and o2[1] <= lp[1] for o2 in back)]
    loops = []
    for a, b in sorted(inner):
        seg = ins[a:b + 1]
        if len(seg) < min_loop:
            continue
        h = collections.Counter(_base(o) for o, _, _ in seg)
        lines = [ln for _, ln, _ in seg if ln]
        loops.append({"at": a, "len": len(seg), "fp64": h["DFMA"] + h["DADD"] + h["DMUL"], "DFMA": h["DFMA"], "DADD": h["DADD"],
                      "DMUL": h["DMUL"], "SHFL": h["SHFL"], "LDS": h["LDS"], "STS": h["STS"], "BAR": h["BAR"], "LDL": h["LDL"],
                      "STL": h["STL"], "LDG": h["LDG"], "STG": h["STG"], "lines": (min(lines), max(lines))})
    return {"variant": variant, "instructions": len(ins), "hist": hist, "mem": mem, "local_lines": local_lines, "loops": loops}


def markdown(r):
    o = ["kernel `%s`: %d SASS instructions" % (r["variant"], r["instructions"]), "",
         "whole kernel, by opcode: " + ", ".join("%s %d" % kv for kv in r["hist"].most_common(30)), "",
         "global / local accesses by flavour: " + ", ".join("%s %d" % kv for kv in sorted(r["mem"].items())), "",
         "local-memory accesses (spills) by source line of cavity_resident.cu: " +
         ", ".join("%s@%d x%d" % (k[0], k[1], n) for k, n in sorted(r["local_lines"].items(), key=lambda kv: kv[0][1])), "",
         "innermost loops of >= 100 instructions:", "",
         "| at | len | fp64 | DFMA | DADD | DMUL | SHFL | LDS | STS | BAR | LDL | STL | LDG | STG | source lines |", "|" + "---|" * 15]
    for l in r["loops"]:
        o.append("| %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d-%d |" % (
            l["at"], l["len"], l["fp64"], l["DFMA"], l["DADD"], l["DMUL"], l["SHFL"], l["LDS"], l["STS"], l["BAR"], l["LDL"], l["STL"],
            l["LDG"], l["STG"], l["lines"][0], l["lines"][1]))
    return "\n".join(o)


if __name__ == "__main__":
    print(markdown(report(disassemble(sys.argv[1] if len(sys.argv) > 1 else None))))
