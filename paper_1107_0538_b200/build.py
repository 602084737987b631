"""Build libcg_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

cg_api.cu (ABI, setup kernels, generic path) and seven instances of cg_variant.cu (one per streamed
kernel shape and slot format, one for the short-row kernels) and cg_rcm.cpp (host-side renumbering) are compiled in parallel and linked into one shared library."""
from __future__ import annotations

import os
import shutil
import subprocess
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "cg_api.cu"), os.path.join(CSRC, "cg_variant.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("cg_kernels.cuh", "cg_stream.cuh", "cg_stream_kernels.cuh", "cg_variants.h", "cg_rcm.cpp", "cg_noalloc.cu")] \
    + [os.path.join(ROOT, "include", "cg.h")]
LIB = os.path.join(HERE, "libcg_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def find_nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libcg_b200.so cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or is_stale()):
        return LIB
    nvcc = find_nvcc()
    extra = ["-Xptxas=-v"] if verbose else []
    with tempfile.TemporaryDirectory(prefix="cg_b200_build_") as tmp:
        units = [("api", SOURCES[0], [])]
        units += [(f"shape{s}_cmp{c}", SOURCES[1], [f"-DCG_SHAPE={s}", f"-DCG_CMP={c}"]) for s in range(3) for c in range(2)]
        units += [("short", SOURCES[1], ["-DCG_SHORT"])]
        units += [("rcm", os.path.join(CSRC, "cg_rcm.cpp"), [])]
        units += [("noalloc", os.path.join(CSRC, "cg_noalloc.cu"), [])]
        procs = []
        for name, src, defs in units:
            obj = os.path.join(tmp, name + ".o")
            log = open(os.path.join(tmp, name + ".log"), "w+")
            cmd = [nvcc, *NVCC_FLAGS, *extra, *defs, "-c", "-o", obj, src]
            procs.append((name, obj, log, subprocess.Popen(cmd, stdout=log, stderr=subprocess.STDOUT)))
        failed = []
        for name, obj, log, pr in procs:
            rc = pr.wait()
            log.seek(0)
            out = log.read()
            log.close()
            if verbose and out:
                print(f"---- {name}\n{out}")
            if rc != 0:
                failed.append((name, out))
        if failed:
            raise RuntimeError("nvcc failed:\n" + "\n".join(f"[{n}]\n{o}" for n, o in failed))
        out_tmp = LIB + f".{os.getpid()}.tmp"
        subprocess.check_call([nvcc, *NVCC_FLAGS, "-shared", "-o", out_tmp, *[obj for _, obj, _, _ in procs]])
        os.replace(out_tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
