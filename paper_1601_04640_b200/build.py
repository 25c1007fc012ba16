"""Build libdbec.so (the C-ABI library of include/dbec.h) in-tree with nvcc for sm_100a.

    python -m paper_1601_04640_b200.build [--force]

nvcc cross-compiles without a GPU.  The object files land in paper_1601_04640_b200/build/, the
library beside this file so that it travels with the source tree.  The library carries a hash of its
sources (dbec_build_id); build() is a no-op when that hash matches the tree, whatever the file times say.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdbec.so")
SOURCES = ["kernels_fft.cu", "kernels_cn.cu", "kernels_tma.cu", "kernels_xline.cu", "kernels_xwarp.cu", "kernels_gen.cu", "kernels_small.cu", "kernels_small_p2.cu", "kernels_noalloc.cu", "dbec_api.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _deps():
    out = [os.path.join(HERE, "..", "include", "dbec.h")]
    for f in sorted(os.listdir(CSRC)):
        out.append(os.path.join(CSRC, f))
    return out


_MARK = b"DBEC_BUILD_ID="


def source_id() -> str:
    """Hash of every source file the library is built from (and of the compiler flags)."""
    h = hashlib.sha256(" ".join(FLAGS).encode())
    for d in _deps():
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:32]


def built_id(lib=LIB):
    """The source hash compiled into an existing libdbec.so (dbec_build_id), read from the file's bytes so
    that a stale library never has to be loaded; None if the file is missing or carries no id."""
    if not os.path.exists(lib):
        return None
    with open(lib, "rb") as f:
        blob = f.read()
    i = blob.find(_MARK)
    return blob[i + len(_MARK): i + len(_MARK) + 32].decode("ascii", "replace") if i >= 0 else None


def _compile(src, sid):
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    log = obj + ".log"
    cmd = [NVCC, *FLAGS, f'-DDBEC_BUILD_ID_STR="{sid}"', "-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stderr[-4000:]}")
    return obj


def build(force: bool = False) -> str:
    sid = source_id()
    if not force and built_id() == sid:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, sid), SOURCES))
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stderr[-4000:])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
