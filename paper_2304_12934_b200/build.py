"""Builds libtc.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.  `python -m paper_2304_12934_b200.build`."""
import os, subprocess, sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("TC_LIBTC", os.path.join(HERE, "libtc.so"))      # TC_LIBTC: build / load another file (kernel variants)
SOURCES = ["tc_api.cu", "kernels_nufft.cu", "kernels_mbir.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = os.environ.get("TC_NVCC_FLAGS", "").split() + ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-rdc=false"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "tc.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not _stale():
        return LIB
    bdir = os.path.join(HERE, "build", os.path.basename(LIB).replace(".so", ""))
    os.makedirs(bdir, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def cc(src):
        obj = os.path.join(bdir, src.replace(".cu", ".o"))
        r = subprocess.run([NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj], capture_output=True, text=True)
        return src, obj, r

    with ThreadPoolExecutor(len(SOURCES)) as ex:
        res = list(ex.map(cc, SOURCES))
    for src, obj, r in res:
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed on " + src)
    r = subprocess.run([NVCC, "-shared", "-o", LIB, *[o for _, o, _ in res], "-lcudart", "-ldl"], capture_output=True, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
