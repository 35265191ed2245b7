"""Build paper_1912_04457_b200/libbz.so (hand-written CUDA for sm_100a, C ABI of include/bz.h) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbz.so")
TESTHOOKS_LIB = os.path.join(HERE, "libbz_testhooks.so")     # test-only object (csrc/bz_testhooks.cu), never loaded by bz.py
SOURCES = ["bz_api.cu", "bz_collision.cu", "bz_transport.cu", "bz_vlasov.cu", "bz_paper.cu", "bz_is.cu", "bz_calibrate.cu", "bz_noalloc.cu", "bz_diag.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "-cudart", "shared",
              "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    out = [os.path.join(HERE, "..", "include", "bz.h")]
    for name in os.listdir(CSRC):
        if not name.startswith("bz_testhooks"):
            out.append(os.path.join(CSRC, name))
    return out


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(tmp, LIB)
    return LIB


def build_testhooks(force=False):
    """The test-only host build of the kernels' channel algebra (tests/test_host_logic.py); not part of libbz.so."""
    src = os.path.join(CSRC, "bz_testhooks.cu")
    deps = [src, os.path.join(CSRC, "bz_testhooks.h"), os.path.join(CSRC, "bz_channels.cuh")]
    if not force and os.path.exists(TESTHOOKS_LIB) and all(os.path.getmtime(TESTHOOKS_LIB) >= os.path.getmtime(d) for d in deps):
        return TESTHOOKS_LIB
    tmp = TESTHOOKS_LIB + ".tmp.%d" % os.getpid()
    subprocess.run([_nvcc(), *NVCC_FLAGS, src, "-o", tmp], check=True, cwd=CSRC)
    os.replace(tmp, TESTHOOKS_LIB)
    return TESTHOOKS_LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
