"""Builds libfcp.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_08476_b200.build [--force] [--verbose]
    python -m paper_2606_08476_b200.build --sass-summary     # code-object evidence as markdown
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfcp.so")
SOURCES = ["fcp_plan.cpp", "fcp_sched.cpp", "fcp_device.cu", "fcp_attn_fwd.cu", "fcp_attn_bwd.cu"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + \
           [os.path.join(ROOT, "include", "fcp.h"), os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA/C++ source of the package into libfcp.so.  Returns the path."""
    if not force and not _stale():
        return LIB
    objs = []
    common = ["-O3", "-std=c++17", "-lineinfo", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
              "-Xcompiler", "-fPIC"]
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, os.path.splitext(src)[0] + ".o")
        cmd = [_nvcc()] + ARCH + common + ["-c", os.path.join(CSRC, src), "-o", obj]
        if src.endswith(".cu") and verbose:
            cmd += ["-Xptxas", "-v"]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
        objs.append(obj)
    for src, p in procs:
        out = p.communicate()[0].decode()
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s" % (src, out))
        if verbose and out.strip():
            print(out)
    cmd = [_nvcc()] + ARCH + ["-shared", "-o", LIB] + objs + ["-cudart", "static"]
    out = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
    if out.returncode != 0:
        raise RuntimeError("link failed:\n" + out.stdout.decode())
    return LIB


SASS_MNEMONICS = ["UTCHMMA", "LDTM", "STTM", "UTMALDG", "UTMASTG", "UBLKCP", "UBLKRED", "UTMAREDG",
                  "MUFU.EX2", "HMMA", "STL", "LDL"]


def sass_summary():
    """Markdown table of what the shipped code object contains, per kernel: registers, spills,
    shared memory (ptxas -v, via cuobjdump -res-usage) and counts of the SASS mnemonics that
    prove the Blackwell path (UTCHMMA = tcgen05.mma, LDTM / STTM = tcgen05.ld / st, UTMALDG /
    UTMASTG = TMA tensor load / store, UBLKCP / UBLKRED = bulk copy / reduce)."""
    import re
    lib = build()
    cu = os.path.join(os.path.dirname(_nvcc()), "cuobjdump")
    cu = cu if os.path.exists(cu) else "cuobjdump"
    res = subprocess.run([cu, "-res-usage", lib], stdout=subprocess.PIPE, text=True).stdout
    usage = {}
    for m in re.finditer(r"Function ([^:\n]+):\n\s*(.*)", res):
        usage[m.group(1).strip()] = m.group(2).strip()
    sass = subprocess.run([cu, "-sass", lib], stdout=subprocess.PIPE, text=True).stdout
    counts, cur = {}, None
    for line in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = m.group(1)
            counts[cur] = dict.fromkeys(SASS_MNEMONICS, 0)
            counts[cur]["instructions"] = 0
            continue
        if cur and re.match(r"\s*/\*[0-9a-f]{4,}\*/", line):
            counts[cur]["instructions"] += 1
            for k in SASS_MNEMONICS:
                if re.search(r"\b" + re.escape(k), line):
                    counts[cur][k] += 1
    filt = subprocess.run(["c++filt"] + list(counts), stdout=subprocess.PIPE, text=True).stdout.splitlines()
    names = dict(zip(counts, filt)) if len(filt) == len(counts) else {k: k for k in counts}
    out = ["| kernel | " + " | ".join(["instructions"] + SASS_MNEMONICS) + " | resources (cuobjdump -res-usage) |",
           "|---|" + "---:|" * (len(SASS_MNEMONICS) + 1) + "---|"]
    for k in sorted(counts, key=lambda x: names[x]):
        short = names[k].replace("(anonymous namespace)::", "").replace("<unnamed>::", "")
        short = re.sub(r"^void ", "", short)
        short = re.sub(r"\(.*", "", short)
        c = counts[k]
        out.append("| `%s` | %s | %s |" % (short, " | ".join(str(c[x]) for x in ["instructions"] + SASS_MNEMONICS),
                                            usage.get(k, "")))
    return "\n".join(out)


if __name__ == "__main__":
    if "--sass-summary" in sys.argv:
        print(sass_summary())
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
