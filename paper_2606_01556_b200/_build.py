"""In-tree build of libtwq.so (the C-ABI CUDA library) with nvcc for sm_100a.

`python -m paper_2606_01556_b200._build` or `build()`; the .so lands next to this file so
that it travels with the repo snapshot to the GPU box (no JIT cache involved).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtwq.so")
TRACE_LIB = os.path.join(HERE, "libtwq_trace.so")      # --trace: the same library with the in-kernel timeline (csrc/trace.cuh)
SOURCES = ["twq_api.cu", "quantize_act.cu", "pack_weights.cu", "fused_kernel.cu", "decode_kernel.cu", "peak_i8.cu", "cold_fill.cu", "static_ws.cu", "fused_inst_tn16.cu",
           "fused_inst_tn32.cu", "fused_inst_tn64.cu", "fused_inst_tn128.cu", "fused_inst_tn128p.cu"]
HEADERS = ["sm100_ptx.cuh", "trace.cuh", "fused_kernel.h", "fused_kernel.cuh", "packed_layout.h", os.path.join("..", "..", "include", "twq.h"),
           os.path.join("..", "..", "include", "twq_testing.h")]
# No --use_fast_math: the quantizer's FP32 op order is part of the specification.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--fmad=true"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), out: str | None = None) -> str:
    """Build the library.  The default call builds the product (libtwq.so, objects next to the sources).  `defines`
    / `out` build a variant into its own object directory, e.g. the timeline build of csrc/trace.cuh:
    build(defines=["TWQ_TRACE"], out=TRACE_LIB)  ==  python -m paper_2606_01556_b200._build --trace."""
    variant = bool(defines) or out is not None
    lib = out or LIB
    if not variant and not force and not needs_build():
        return LIB
    objdir = CSRC
    if variant:
        objdir = os.path.join(CSRC, "build_" + ("_".join(d.replace("=", "-") for d in defines) or "variant"))
        os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(objdir, s.replace(".cu", ".o"))
        objs.append(o)
        cmd = [_nvcc(), *NVCC_FLAGS, *[f"-D{d}" for d in defines], "-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for cmd, pr in procs:
        out_text, _ = pr.communicate()
        log.append(out_text)
        if pr.returncode != 0:
            sys.stderr.write(out_text)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call([_nvcc(), "-shared", "-o", tmp, *objs, "-cudart", "static"])
    os.replace(tmp, lib)
    with open(os.path.join(objdir, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return lib


if __name__ == "__main__":
    if "--trace" in sys.argv:
        print(build(verbose="-v" in sys.argv, defines=["TWQ_TRACE"], out=TRACE_LIB))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
