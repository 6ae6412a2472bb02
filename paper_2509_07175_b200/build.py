"""Build libvd.so (the CUDA path) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvd.so")
# (source, object suffix, extra flags): the clip / phase kernels are compiled twice -- lean (optional query features compiled
# out) and full -- into namespaces of their own (header of csrc/vd_clip.cu)
LEAN = ["-DVD_EXT=0", "-DVD_VARIANT=lean"]
FULL = ["-DVD_EXT=1", "-DVD_VARIANT=full"]
SOURCES = [("vd_clip.cu", "_lean", LEAN), ("vd_phase.cu", "_lean", LEAN), ("vd_clip.cu", "_full", FULL), ("vd_phase.cu", "_full", FULL),
           ("vd_api.cu", "", []), ("vd_domain.cu", "", []), ("vd_index.cu", "", []), ("vd_assemble.cu", "", []), ("vd_peak.cu", "", [])]


def lib_path() -> str:
    return os.environ.get("VD_LIB", LIB)   # experiments: another build of the same library


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [(os.path.join(CSRC, s), sfx, fl) for s, sfx, fl in SOURCES]
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "vd.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    extra = os.environ.get("VD_NVCC_FLAGS", "").split()   # experiments: -DVD_... switches of the kernels

    def compile_one(item):
        s, sfx, flags = item
        o = s[:-3] + sfx + ".o"
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
               "-Xcompiler", "-fPIC"] + flags + extra + ["-c", s, "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        return o

    with ThreadPoolExecutor(max_workers=len(srcs)) as pool:   # one nvcc per translation unit, side by side
        objs = list(pool.map(compile_one, srcs))
    subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs + ["-ldl"])
    for o in objs:
        os.remove(o)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
