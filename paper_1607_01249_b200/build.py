"""Build ``libttc.so`` (the C-ABI library of include/ttc.h) in-tree with nvcc for sm_100a.

``python -m paper_1607_01249_b200.build [--force]``.  nvcc cross-compiles without a GPU.  The
built library sits beside this file (git-ignored, but it travels to the GPU box).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB_PATH = os.path.join(HERE, "libttc.so")
SOURCES = ["kernels.cu", "api.cpp", "plan.cpp", "canon.cpp", "specialize.cpp", "static_scratch.cu"]
HEADERS = [os.path.join(CSRC, "ttc_internal.h"), os.path.join(CSRC, "ttc_params.h"), os.path.join(CSRC, "ttc_device.cuh"),
           os.path.join(CSRC, "ttc_tmap.h"), os.path.join(CSRC, "ttc_tmap.cuh"),
           os.path.join(CSRC, "ttc_skew.h"), os.path.join(CSRC, "ttc_skew.cuh"),
           os.path.join(INCLUDE, "ttc.h")]
# Never -use_fast_math: it would flush denormals and contract roundings (reading A10).
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-I" + INCLUDE, "-I" + CSRC]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _embed_device_source(objdir: str) -> str:
    """The device code as a string constant of the library (specialize.cpp hands it to NVRTC): ttc_params.h, a
    marker line, ttc_device.cuh -- without the #pragma once / #include lines that tie them together as files."""
    def text(name):
        with open(os.path.join(CSRC, name)) as fh:
            return "".join(ln for ln in fh if not ln.startswith("#pragma once") and not ln.startswith('#include "ttc_params.h"'))
    body = text("ttc_params.h") + "//@@TTC_DEVICE_CODE@@\n" + text("ttc_device.cuh")
    assert ')TTCSRC"' not in body
    out = os.path.join(objdir, "device_source.cpp")
    chunks = [body[i:i + 8000] for i in range(0, len(body), 8000)]       # string literals of moderate length
    code = "namespace ttc {\nextern const char* const kDeviceSource;\nconst char* const kDeviceSource =\n" + \
        "\n".join('R"TTCSRC(' + c + ')TTCSRC"' for c in chunks) + ";\n}\n"
    old = open(out).read() if os.path.exists(out) else None
    if old != code:
        with open(out, "w") as fh:
            fh.write(code)
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    newest = max(os.path.getmtime(p) for p in srcs + HEADERS + [os.path.abspath(__file__)])
    if not force and os.path.exists(LIB_PATH) and os.path.getmtime(LIB_PATH) >= newest:
        return LIB_PATH
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    srcs = srcs + [_embed_device_source(objdir)]
    objs = []
    procs = []
    hdr_time = max(os.path.getmtime(p) for p in HEADERS + [os.path.abspath(__file__)])
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s) + ".o")
        objs.append(o)
        if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), hdr_time):
            continue                      # object is newer than its source and every header
        cmd = [_nvcc(), *NVCC_FLAGS, "-c", s, "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = LIB_PATH + ".tmp.%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs,
                           "-cudart", "static", "-ldl"])
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
