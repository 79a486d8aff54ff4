"""Builds libkrp.so (the C-ABI CUDA library of include/krp.h) in-tree with nvcc for sm_100a."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC_DIR = os.path.join(HERE, "csrc")
SOURCES = ["krp_api.cu"]
HEADERS = ["krp_device.cuh", "krp_kernels.cuh", "krp_twostep.cuh", "krp_noalloc.cuh", os.path.join(ROOT, "include", "krp.h")]
LIB = os.path.join(HERE, "libkrp.so")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


ID_FILE = os.path.join(HERE, "libkrp.id")


def _deps():
    return [os.path.join(SRC_DIR, s) for s in SOURCES] + \
           [h if os.path.isabs(h) else os.path.join(SRC_DIR, h) for h in HEADERS]


def source_id():
    """Build id: hash of the sources and of the compiler flags (compiled into krp_version())."""
    import hashlib
    h = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for d in _deps():
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:12]


def stale():
    """True when the library is missing or was built from other sources than those beside it (content, not mtime:
    the tree is copied to the GPU box with new timestamps)."""
    if not os.path.exists(LIB) or not os.path.exists(ID_FILE):
        return True
    with open(ID_FILE) as f:
        return f.read().strip() != source_id()


def build(force=False, verbose=False):
    """Compile when the library is missing or older than its sources.  Returns the path."""
    if not force and not stale():
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    sid = source_id()
    cmd = [_nvcc()] + NVCC_FLAGS + ['-DKRP_BUILD_ID="%s"' % sid] + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(SRC_DIR, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    with open(ID_FILE, "w") as f:
        f.write(sid + "\n")
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
