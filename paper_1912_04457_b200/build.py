"""Build paper_1912_04457_b200/libbz.so (hand-written CUDA for sm_100a, C ABI of include/bz.h) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbz.so")
TESTHOOKS_LIB = os.path.join(HERE, "libbz_testhooks.so")     # test-only object (csrc/bz_testhooks.cu), never loaded by bz.py
SOURCES = ["bz_api.cu", "bz_collision.cu", "bz_transport.cu", "bz_vlasov.cu", "bz_paper.cu", "bz_is.cu", "bz_calibrate.cu", "bz_noalloc.cu"]
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
        if not name.startswith("bz_testhooks") and not name.endswith("_probe.cu"):
            out.append(os.path.join(CSRC, name))
    return out


def _extra_defines():
    """Measurement builds only: BZ_NVCC_DEFINES="-DBZ_ABLATE=3" python -m paper_1912_04457_b200.build compiles libbz.so with a
    phase of collide_kernel switched off (profiles/r2_collide_ablation.md).  Unset for the product."""
    return os.environ.get("BZ_NVCC_DEFINES", "").split()


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *_extra_defines(), *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
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


def build_scatter_probe():
    """The scatter-design measurement tool (csrc/bz_scatter_probe.cu -> bz_scatter_probe, a stand-alone executable; not part
    of libbz.so): profiles/r2_scatter_variants.md keeps its output."""
    out = os.path.join(HERE, "bz_scatter_probe")
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                    os.path.join(CSRC, "bz_scatter_probe.cu"), "-o", out], check=True, cwd=CSRC)
    return out


def build_issue_probe():
    """The issue-port measurement tool (csrc/bz_issue_probe.cu -> bz_issue_probe, a stand-alone executable; not part of
    libbz.so): profiles/r2_collide_issue_model.md keeps its output."""
    out = os.path.join(HERE, "bz_issue_probe")
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                    os.path.join(CSRC, "bz_issue_probe.cu"), "-o", out], check=True, cwd=CSRC)
    return out


if __name__ == "__main__":
    if "scatter_probe" in sys.argv:
        print(build_scatter_probe())
        sys.exit(0)
    if "issue_probe" in sys.argv:
        print(build_issue_probe())
        sys.exit(0)
    print(build(force=True, verbose="-v" in sys.argv))
