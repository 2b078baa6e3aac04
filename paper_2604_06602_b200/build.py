"""Build paper_2604_06602_b200/libumi_b200.so (the C-ABI library of include/umi.h)
with nvcc for sm_100a.  In-tree, no JIT cache: the .so travels with the repo
snapshot.  Run `python -m paper_2604_06602_b200.build` or call build().

Each .cu is compiled to an object of its own (in parallel, under _obj/) and the
objects are linked into the shared library; an object is rebuilt when its source,
any header or this file is newer.  `--define NAME=VALUE` compiles a measured, off-by-default
alternative in (a plain build afterwards restores the default).  `--bakeoff` builds libumi_bakeoff.so instead:
the selection / mapping candidates of csrc/bakeoff/ that were measured against the
product kernels; they are never part of libumi_b200.so.
"""
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "_obj")
SOURCES = [os.path.join(CSRC, n) for n in
           ("umi_api.cu", "umi_median.cu", "umi_reweight.cu", "umi_small.cu", "umi_regrid.cu", "umi_static.cu")]
HEADERS = [os.path.join(CSRC, "umi_internal.h"), os.path.join(CSRC, "umi_device.cuh"), os.path.join(ROOT, "include", "umi.h")]
LIB = os.path.join(HERE, "libumi_b200.so")
BAKEOFF_DIR = os.path.join(CSRC, "bakeoff")
BAKEOFF_LIB = os.path.join(HERE, "libumi_bakeoff.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _bakeoff_sources():
    if not os.path.isdir(BAKEOFF_DIR):
        return []
    return sorted(os.path.join(BAKEOFF_DIR, n) for n in os.listdir(BAKEOFF_DIR) if n.endswith(".cu"))


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(p) > t for p in deps)


def needs_build():
    return _stale(LIB, SOURCES + HEADERS + [os.path.abspath(__file__)])


def _compile(src, obj, verbose, extra):
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra) + ["-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-c", "-o", obj, src]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return src, cmd, res.returncode, res.stdout


def _build_lib(lib, sources, force, verbose, extra=()):
    os.makedirs(OBJDIR, exist_ok=True)
    tag = os.path.splitext(os.path.basename(lib))[0]
    objs, jobs = [], []
    for src in sources:
        obj = os.path.join(OBJDIR, "%s.%s.o" % (tag, os.path.splitext(os.path.basename(src))[0]))
        objs.append(obj)
        if force or verbose or _stale(obj, [src] + HEADERS + [os.path.abspath(__file__)]):
            jobs.append((src, obj))
    log = []
    if jobs:
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            for src, cmd, rc, out in ex.map(lambda j: _compile(j[0], j[1], verbose, extra), jobs):
                if rc != 0:
                    raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), out))
                log.append(out)
    if jobs or not os.path.exists(lib):
        tmp = lib + ".tmp.%d" % os.getpid()
        cmd = [_nvcc()] + LINK_FLAGS + ["-o", tmp] + objs
        res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if res.returncode != 0:
            if os.path.exists(tmp):
                os.remove(tmp)
            raise RuntimeError("link failed:\n%s\n%s" % (" ".join(cmd), res.stdout))
        os.replace(tmp, lib)
    if verbose:
        print("\n".join(log))
    return lib


def build(force=False, verbose=False, defines=()):
    """Compile what is out of date and link libumi_b200.so.  Returns the library path.
    defines: compile-time alternatives that were measured and are off by default (e.g. "UMI_K1_RADIX=1")."""
    if not force and not verbose and not defines and not needs_build():
        return LIB
    return _build_lib(LIB, SOURCES, force or bool(defines), verbose, extra=["-D" + d for d in defines])


def build_bakeoff(force=False, verbose=False):
    """libumi_bakeoff.so: the measured alternatives (selection schemes, pass mappings); not product."""
    srcs = _bakeoff_sources()
    if not srcs:
        raise RuntimeError("no sources under %s" % BAKEOFF_DIR)
    return _build_lib(BAKEOFF_LIB, srcs, force, verbose)


if __name__ == "__main__":
    v = "-v" in sys.argv
    defs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define"]
    if "--bakeoff" in sys.argv:
        print(build_bakeoff(force=True, verbose=v))
    else:
        print(build(force=True, verbose=v, defines=defs))
