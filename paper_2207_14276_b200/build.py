"""Compile the CUDA sources under csrc/ into paper_2207_14276_b200/libdhp.so for sm_100a.

`python -m paper_2207_14276_b200.build` or `build()`; nvcc cross-compiles without a GPU.
The library is built IN-TREE so that it travels with the repository snapshot to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdhp.so")
SOURCES = ["api.cu", "nlist.cu", "aev.cu", "mlp_simt.cu", "mlp_tc.cu", "md.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "--fmad=true"]
EXTRA = os.environ.get("DHP_NVCC_EXTRA", "").split()        # e.g. -DMID_TRACE=1 for a timing experiment (never the default)
FLAGS += EXTRA
# An experiment build must not pass for the default library: the extra flags are compiled into dhp_version() (through the
# generated header below) and kept in a stamp beside the library; a build with other flags than the stamp's is stale, and
# binding.load_library() refuses a library that carries extra flags unless DHP_ALLOW_EXPERIMENT=1 is set.
STAMP = LIB + ".flags"
FLAGS_HEADER = os.path.join(HERE, "build", "dhp_build_flags.h")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    if (open(STAMP).read() if os.path.exists(STAMP) else "") != " ".join(EXTRA):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "dhp.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    with open(FLAGS_HEADER, "w") as f:
        f.write('#define DHP_EXTRA_FLAGS "%s"\n' % " ".join(EXTRA).replace("\\", "").replace('"', "'"))
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        cmd = [NVCC, *FLAGS, "-I", os.path.join(HERE, "build"), "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if out.strip() and (verbose or p.returncode != 0):
            print(f"--- {src}\n{out}", file=sys.stderr)
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, "-shared", "--cudart", "static", "-o", tmp, *objs])
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(" ".join(EXTRA))
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
