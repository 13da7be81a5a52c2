"""In-tree build of libahs.so with nvcc for sm_100a (and nothing else).

    python -m paper_1809_00995_b200.build                 # (re)build csrc/libahs.so
    python -m paper_1809_00995_b200.build --sass          # per-kernel SASS instruction histogram + registers / spills (markdown)
"""
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libahs.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",                       # IEEE fma contraction only; never --use_fast_math
    "-Xcompiler", "-fPIC,-O2,-fvisibility=hidden",
    "-Xptxas", "-v",
    "-shared",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "ahs.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force=False, verbose=False):
    """Compile csrc/*.cu into csrc/libahs.so. Returns the path."""
    if not force and not stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [NVCC] + NVCC_FLAGS + ["-o", tmp] + sources()
    r = subprocess.run(cmd, capture_output=True, text=True)
    log = os.path.join(CSRC, "build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout[-4000:] + r.stderr[-8000:])
    os.replace(tmp, LIB)
    if verbose:
        print("built", LIB)
    return LIB


# ---------------------------------------------------------------------------------------------------------------------------
# evidence: which Blackwell instructions each kernel of the built library contains (profiles/r4_sass_histogram.md)
# ---------------------------------------------------------------------------------------------------------------------------
SASS_MNEMONICS = ("UTMALDG", "UTMAPF", "UBLKCP", "SYNCS", "FFMA2", "FMUL2", "FADD2", "FFMA", "FMUL", "FADD", "DFMA", "DMUL", "DADD",
                  "MUFU", "LDG", "STG", "LDS", "STS", "ATOMS", "ATOMG", "SHFL", "BAR", "LDL", "STL")


def sass_histogram(lib=LIB):
    """{kernel: {mnemonic: count}} from `cuobjdump -sass`, plus (registers, stack, spill stores, spill loads) from build.log."""
    import collections
    import re
    cuobjdump = os.path.join(os.path.dirname(NVCC), "cuobjdump")
    out = subprocess.run([cuobjdump, "-sass", lib], capture_output=True, text=True, check=True).stdout
    demangle = lambda names: dict(zip(names, subprocess.run(["c++filt"] + names, capture_output=True, text=True).stdout.split("\n")))
    hist, cur = collections.OrderedDict(), None
    for line in out.split("\n"):
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = hist.setdefault(m.group(1), collections.Counter())
            continue
        m = re.search(r"/\*[0-9a-f]{4,5}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)(\.[A-Z0-9_.]+)?", line)
        if m and cur is not None:
            cur[m.group(1)] += 1
            if m.group(1) in ("LDG", "STG", "LDS") and m.group(2) and "128" in m.group(2):
                cur[m.group(1) + ".128"] += 1
            cur["total"] += 1
    res = {}
    log = open(os.path.join(CSRC, "build.log")).read() if os.path.exists(os.path.join(CSRC, "build.log")) else ""
    for name, v in re.findall(r"Compiling entry function '([^']+)' for 'sm_100a'\nptxas info\s+: Function properties for [^\n]+\n\s+"
                              r"(\d+ bytes stack frame, \d+ bytes spill stores, \d+ bytes spill loads)\nptxas info\s+: Used (?:\d+) registers", log):
        pass
    regs = {n: (int(r), st) for n, st, r in re.findall(
        r"Compiling entry function '([^']+)' for 'sm_100a'\nptxas info\s+: Function properties for [^\n]+\n\s+([^\n]+)\nptxas info\s+: Used (\d+) registers", log)}
    names = demangle(list(hist))
    for k, c in hist.items():
        res[names.get(k, k)] = (c, regs.get(k))
    return res


def print_sass_markdown():
    lib = build_library()
    h = sass_histogram(lib)
    cols = ("UTMALDG", "UTMAPF", "UBLKCP", "SYNCS", "FFMA2", "FMUL2", "FADD2", "FFMA", "DFMA", "MUFU", "LDG.128", "STG.128", "LDS.128", "ATOMS", "SHFL", "BAR", "LDL", "STL", "total")
    print("| kernel | registers | stack / spills | " + " | ".join(cols) + " |")
    print("|---|---|---|" + "---|" * len(cols))
    short = lambda n: n.replace("ahs::(anonymous namespace)::", "").replace("void ", "").split("(")[0]
    for name, (c, rg) in h.items():
        print("| `%s` | %s | %s | " % (short(name), rg[0] if rg else "?", rg[1] if rg else "?") + " | ".join(str(c.get(k, 0)) for k in cols) + " |")


if __name__ == "__main__":
    import sys
    if "--sass" in sys.argv:
        print_sass_markdown()
    else:
        build_library(force="--force" in sys.argv, verbose=True)
