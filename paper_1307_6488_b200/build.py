"""Builds paper_1307_6488_b200/libchemora.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1307_6488_b200.build [--force]
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libchemora.so")
SOURCES = ["chemora.cu", "kernels_basic.cu", "kernels_boundary.cu", "kernels_bssn.cu", "kernels_bssn_tma.cu", "kernels_wave_tma.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _deps():
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    files.append(os.path.join(os.path.dirname(HERE), "include", "chemora.h"))
    return files


def build(force=False, verbose=False):
    newest = max(os.path.getmtime(f) for f in _deps())
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        srcp = os.path.join(CSRC, src)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) >= newest:
            return obj, ""
        r = subprocess.run([nvcc] + NVCC_FLAGS + ["-c", srcp, "-o", obj], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s" % (src, r.stderr))
        return obj, r.stderr

    with ThreadPoolExecutor(len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    log = "".join(r[1] for r in results)
    with open(os.path.join(objdir, "ptxas.log"), "a" if not force else "w") as f:
        f.write(log)
    if verbose:
        sys.stderr.write(log)
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.check_call([nvcc, "-shared", "-o", tmp] + [r[0] for r in results] + ["-gencode",
                          "arch=compute_100a,code=sm_100a"])
    os.replace(tmp, LIB)
    return LIB


def report():
    """Static per-kernel report of the built library (the paper's run-time prints one per kernel at the end of a run,
    PAPER.md:272-276; this is its compile-time part): registers and spill bytes from ptxas, SASS instruction counts from
    cuobjdump.  Markdown table on stdout.  Needs a build made by this process or an earlier one (build/ptxas.log)."""
    import collections
    import re
    cuda_bin = os.path.dirname(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"))
    sass = subprocess.run([os.path.join(cuda_bin, "cuobjdump"), "-sass", LIB], capture_output=True, text=True,
                          check=True).stdout
    log = open(os.path.join(HERE, "build", "ptxas.log")).read()
    regs = {}
    for m in re.finditer(r"Compiling entry function '(\S+)' for 'sm_100a'\nptxas info\s+: Function properties for \S+\n"
                         r"\s+\d+ bytes stack frame, (\d+) bytes spill stores, \d+ bytes spill loads\n"
                         r"ptxas info\s+: Used (\d+) registers", log):
        regs[m.group(1)] = (int(m.group(3)), int(m.group(2)))
    cur, cnt = None, collections.defaultdict(collections.Counter)
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+(@!?U?P[0-9T]+ )?([A-Z0-9_]+)", line)
        if m and cur:
            cnt[cur][m.group(2)] += 1
    names = sorted(cnt)
    dem = subprocess.run(["c++filt"] + names, capture_output=True, text=True).stdout.splitlines()
    rows = []
    for n, d in zip(names, dem):
        c, r = cnt[n], regs.get(n, ("?", "?"))
        d = re.sub(r"\(.*", "", d).replace("void chm::", "").replace("chm::", "")
        rows.append((d, r[0], r[1], sum(c.values()), c["DADD"] + c["DMUL"] + c["DFMA"], c["LDS"], c["STS"],
                     c["UTMALDG"], c["SYNCS"], c["LDG"], c["STG"]))
    print("| kernel | regs | spill B | SASS instr | FP64 | LDS | STS | UTMALDG | SYNCS | LDG | STG |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for r in sorted(rows):
        print("| `%s` | %s |" % (r[0], " | ".join(str(x) for x in r[1:])))


def _sass_groups(path):
    """{demangled kernel name: Counter of SASS mnemonics (up to the first '.')} of an object file or library; the
    key "" of a Counter holds a hash of the kernel's whole instruction text (operands included; instruction addresses
    and encodings left out)"""
    import collections
    import hashlib
    import re
    cuda_bin = os.path.dirname(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"))
    sass = subprocess.run([os.path.join(cuda_bin, "cuobjdump"), "-sass", path], capture_output=True, text=True,
                          check=True).stdout
    cur, cnt, text = None, collections.OrderedDict(), {}
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            cnt[cur], text[cur] = collections.Counter(), hashlib.md5()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+((@!?U?P[0-9T]+ )?([A-Z0-9_]+).*?)\s*/\* 0x[0-9a-f]+ \*/", line)
        if m and cur:
            cnt[cur][m.group(3)] += 1
            text[cur].update(m.group(1).encode() + b"\n")
    for k in cnt:
        cnt[k][""] = int(text[k].hexdigest(), 16)
    dem = subprocess.run(["c++filt"], input="\n".join(cnt), capture_output=True, text=True).stdout.split("\n")
    return {re.sub(r"\(.*", "", d).replace("void chm::", "").replace("chm::", ""): c for d, c in zip(dem, cnt.values())}


def compare(old, new):
    """Static SASS comparison of two builds of the same kernels, e.g. the object of an earlier commit against this
    tree's (how profiles/r02_sass_vs_round1.md was made): per kernel present in both, the count of each instruction
    group, `a -> b` where it changed.  Says what a refactoring did to kernels that have run on hardware: which kinds
    of instruction were added or dropped -- not more than that (no two builds schedule alike)."""
    a, b = _sass_groups(old), _sass_groups(new)
    groups = [("DADD", ("DADD",)), ("DMUL", ("DMUL",)), ("DFMA", ("DFMA",)), ("LDS", ("LDS",)), ("STS", ("STS",)),
              ("LDG", ("LDG",)), ("STG", ("STG",)), ("UTMALDG", ("UTMALDG",)), ("SYNCS", ("SYNCS",)),
              ("BAR", ("BAR",)), ("ATOMG", ("ATOMG",)), ("CS2R", ("CS2R",))]
    print("| kernel | " + " | ".join(g for g, _ in groups) + " | all | instruction text |")
    print("|---|" + "---|" * (len(groups) + 2))
    for k in sorted(a):
        if k not in b:
            continue
        cells = []
        for _, ops in groups + [("all", None)]:
            x = sum(v for o, v in a[k].items() if o) if ops is None else sum(a[k][o] for o in ops)
            y = sum(v for o, v in b[k].items() if o) if ops is None else sum(b[k][o] for o in ops)
            cells.append(str(x) if x == y else "%d -> %d" % (x, y))
        cells.append("same" if a[k][""] == b[k][""] else "differs")
        print("| `%s` | %s |" % (k, " | ".join(cells)))
    print()
    print("only in %s: %s" % (old, ", ".join("`%s`" % k for k in sorted(a) if k not in b) or "-"))
    print("only in %s: %s" % (new, ", ".join("`%s`" % k for k in sorted(b) if k not in a) or "-"))


if __name__ == "__main__":
    if "--compare" in sys.argv:        # python -m paper_1307_6488_b200.build --compare OLD.o NEW.o
        i = sys.argv.index("--compare")
        compare(sys.argv[i + 1], sys.argv[i + 2])
        sys.exit(0)
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--report" in sys.argv:
        report()
