"""Build paper_2604_06602_b200/libumi_b200.so (the C-ABI library of include/umi.h)
with nvcc for sm_100a.  In-tree, no JIT cache: the .so travels with the repo
snapshot.  Run `python -m paper_2604_06602_b200.build` or call build().
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "umi_api.cu"), os.path.join(CSRC, "umi_median.cu"), os.path.join(CSRC, "umi_reweight.cu"),
           os.path.join(CSRC, "umi_small.cu"), os.path.join(CSRC, "umi_regrid.cu"),
           os.path.join(CSRC, "umi_reweight_tc.cu")]
HEADERS = [os.path.join(CSRC, "umi_internal.h"), os.path.join(CSRC, "umi_device.cuh"), os.path.join(ROOT, "include", "umi.h")]
LIB = os.path.join(HERE, "libumi_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "shared",
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force=False, verbose=False):
    """Compile if sources are newer than the library.  Returns the library path."""
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + ["-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", tmp] + SOURCES
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), res.stdout))
    if verbose:
        print(res.stdout)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
