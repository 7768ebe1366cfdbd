"""Build liblr.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot)."""
from __future__ import annotations

import concurrent.futures
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "liblr.so")
SOURCES = ("lr_api.cu", "lr_kernels.cu", "lr_peak.cu", "lr_likelihood.cu", "lr_waveform.cu")
INST_PT = (21, 16, 13, 0, 11, 8, 7, 6, 5, 4, 3, 2, 1)   # lr_inst.cu is compiled once per compile-time pair count (0 = run-time P)
HEADERS = ("lr_inst.cu", "lr_device.cuh", "lr_kernels.cuh", "lr_tdi_fir.cuh", "lr_host.hpp", os.path.join("..", "..", "include", "lr.h"))
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: liblr cannot be built (there is no CPU fallback)")


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile csrc/*.cu into liblr.so; returns the library path."""
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    objdir = os.path.join(_HERE, "build")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(job):
        src, pt = job
        obj = os.path.join(objdir, src.replace(".cu", ".o") if pt is None else f"lr_inst_p{pt}.o")
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        if pt is not None:
            cmd.insert(1, f"-DLR_INST_PT={pt}")
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src} (PT={pt}):\n{r.stdout}\n{r.stderr}")
        return obj, r.stderr

    jobs = [("lr_inst.cu", pt) for pt in INST_PT] + [(src, None) for src in SOURCES]
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        results = list(ex.map(compile_one, jobs))
    objs = [o for o, _ in results]
    tmp = LIB + ".tmp"
    # cuFFT (the likelihood leg's real-to-complex transform) is the one library liblr links dynamically
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")
    r = subprocess.run([nvcc, "-shared", "-o", tmp, *objs, "-cudart", "static", "-L" + cuda_lib, "-lcufft",
                        "-Xlinker", "-rpath=" + cuda_lib], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB)
    if verbose:
        for _, log in results:
            print(log)
    return LIB


def ensure_built(local_rank=0, timeout_s=900.0):
    """Make sure liblr.so exists AND is newer than every source it is built from (the .so is git-ignored but
    travels with the repo snapshot, so a stale one can sit beside edited sources).  Under torchrun only local
    rank 0 compiles; the other ranks wait until the library is no longer stale.  Building the product is not a
    fallback: without nvcc this raises."""
    import time
    if local_rank == 0:
        return build(force=False)
    t0 = time.time()
    while _stale():
        if time.time() - t0 > timeout_s:
            raise RuntimeError("timed out waiting for local rank 0 to build liblr.so")
        time.sleep(1.0)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
