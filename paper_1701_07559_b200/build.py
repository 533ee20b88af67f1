"""Build libmdwf_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Incremental: an object is recompiled when the content hash of its source and of the headers it includes (transitively)
changes; hashes, not mtimes, because a snapshot copied to another machine does not keep mtimes.
"""
import hashlib
import json
import os
import re
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmdwf_b200.so")
OBJDIR = os.path.join(HERE, "build")
STAMP = os.path.join(HERE, "libmdwf_b200.stamp.json")
SOURCES = ["mdwf_api.cu", "hop_d.cu", "hop_s.cu", "hop_h.cu", "hop3_s.cu", "hop3_h.cu", "hop3b_s.cu", "hop3b_h.cu", "hop5_s.cu", "hop6_h.cu", "blas_kernels.cu",
           "layout_kernels.cu", "flow_kernels.cu", "s5_kernels.cu", "peak_kernels.cu", "sdense_mma.cu", "noalloc_kernels.cu"]
FLAGS = os.environ.get("MDWF_NVCC_EXTRA", "").split() + ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
                                                           "-std=c++17", "-Xcompiler", "-fPIC"]
_INC = re.compile(r'^\s*#\s*include\s+"([^"]+)"', re.M)


def _closure(path, seen):
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return
    seen.add(path)
    for inc in _INC.findall(open(path).read()):
        _closure(os.path.join(os.path.dirname(path), inc), seen)


def _digest(src):
    seen = set()
    _closure(os.path.join(CSRC, src), seen)
    h = hashlib.sha256(" ".join(FLAGS).encode())
    for f in sorted(seen):
        h.update(open(f, "rb").read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    want = {s: _digest(s) for s in SOURCES}
    have = {}
    if os.path.exists(STAMP) and not force:
        try:
            have = json.load(open(STAMP))
        except ValueError:
            have = {}
    if os.path.exists(LIB) and have.get("lib") == want:
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    objs_have = have.get("objs", {})

    def compile_one(src):
        obj = os.path.join(OBJDIR, src.replace(".cu", ".o"))
        if os.path.exists(obj) and objs_have.get(src) == want[src]:
            return obj
        cmd = ["nvcc"] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s" % (src, r.stderr))
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.run(["nvcc", "-shared", "-o", LIB] + objs + ["-lcudart"], check=True)
    json.dump({"lib": want, "objs": want}, open(STAMP, "w"))
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="-f" in sys.argv, verbose="-v" in sys.argv))
