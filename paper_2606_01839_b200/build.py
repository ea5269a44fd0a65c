"""Builds paper_2606_01839_b200/libconserve_kv.so from csrc/ with nvcc for sm_100a.

In-tree build (the .so travels to the GPU box with the snapshot).  nvcc cross-compiles
without a GPU.  `python -m paper_2606_01839_b200.build [--force] [--verbose] [--sass-opcodes]`.
--sass-opcodes prints, per kernel of the built library, the `cuobjdump -sass` opcode histogram (the
evidence for tcgen05 / TMEM / bulk-copy use: UTCHMMA, LDTM / STTM, UBLKCP, ...; kept under profiles/).
"""
import collections
import re
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libconserve_kv.so")
OBJDIR = os.path.join(HERE, "build")
SOURCES = ["pool.cpp", "plan.cpp", "api.cu", "handoff.cu", "decode_attn.cu", "append_attn.cu", "append_attn_tc2.cu", "tail_fused.cu", "noalloc.cu"]
HEADERS = ["internal.h", "common.cuh", "tc5.cuh", "decode_worker.cuh", "append_tc2_body.cuh", os.path.join("..", "..", "include", "conserve_kv.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr", "-diag-suppress", "550"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src, verbose):
    obj = os.path.join(OBJDIR, src + ".o")
    deps = [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS]
    if _stale(obj, deps):
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-x", "cu", "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s\n%s" % (src, r.stdout, r.stderr))
        if verbose:
            sys.stderr.write(r.stderr)
    return obj


def build_library(force=False, verbose=False):
    os.makedirs(OBJDIR, exist_ok=True)
    if force:
        for f in os.listdir(OBJDIR):
            os.remove(os.path.join(OBJDIR, f))
    with concurrent.futures.ThreadPoolExecutor(max_workers=6) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose), SOURCES))
    if force or _stale(LIB, objs):
        tmp = LIB + ".%d.tmp" % os.getpid()
        cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
        os.replace(tmp, LIB)
    return LIB


def sass_opcodes(lib=LIB):
    """{kernel: Counter(opcode with modifiers)} from `cuobjdump -sass` of the built library."""
    cuobjdump = os.path.join(os.path.dirname(NVCC), "cuobjdump")
    txt = subprocess.run([cuobjdump, "-sass", lib], capture_output=True, text=True, check=True).stdout
    names = sorted(set(re.findall(r"Function : (\S+)", txt)))
    dem = subprocess.run(["c++filt"] + names, capture_output=True, text=True).stdout.split("\n") if names else []
    pretty = {n: (dem[i] if i < len(dem) and dem[i] else n) for i, n in enumerate(names)}
    out, cur = collections.OrderedDict(), None
    for line in txt.split("\n"):
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = pretty[m.group(1)].replace("(anonymous namespace)::", "").replace("void ", "")
            cur = out.setdefault(re.sub(r"\(.*", "", name), collections.Counter())
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m and cur is not None:
            cur[m.group(1)] += 1
    return out


def print_sass_opcodes():
    """Per kernel: instruction count, then every opcode of the families that show which hardware path is in use."""
    fam = re.compile(r"^(UTC|LDTM|STTM|UBLKCP|UTMA|HMMA|LDSM|MUFU|FFMA2|FADD2|FMNMX3|SYNCS|ACQBULK|ELECT|F2FP|ATOMG|RED|"
                     r"FENCE|MEMBAR|BAR|WARPSYNC|USETMAXREG|LDG|STG|UCGABAR)")
    for kern, cnt in sass_opcodes().items():
        print("%s: %d SASS instructions" % (kern, sum(cnt.values())))
        for op in sorted(cnt):
            if fam.match(op):
                print("    %-34s %d" % (op, cnt[op]))


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    if "--sass-opcodes" in sys.argv:
        print_sass_opcodes()
