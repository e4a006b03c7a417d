"""Build libfarm_map.so (the C-ABI product library) in-tree with nvcc for sm_100a.

    python -m paper_2606_15476_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfarm_map.so")
SOURCES = ["farm_api.cu", "farm_lift.cu", "farm_sim_fma.cu", "farm_sim_tc.cu", "farm_assoc.cu", "farm_query.cu", "farm_edges.cu", "farm_noalloc.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr"]


def _stale(obj, deps):
    return not os.path.exists(obj) or any(os.path.getmtime(d) > os.path.getmtime(obj) for d in deps)


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """trace=True: the development build with -DFARM_TRACE (device-timer stamps, see trace_schedule.py) as libfarm_trace.so;
    the product library is never built with it."""
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdrs.append(os.path.join(HERE, "..", "include", "farm.h"))
    bdir = os.path.join(HERE, "build", "trace") if trace else os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    LIB = os.path.join(HERE, "libfarm_trace.so") if trace else globals()["LIB"]
    FLAGS_ = FLAGS + (["-DFARM_TRACE"] if trace else [])
    objs, procs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(bdir, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + hdrs):
            cmd = [NVCC] + FLAGS_ + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- {src}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if force or procs or _stale(LIB, objs):
        subprocess.check_call([NVCC, "-shared", "-Wno-deprecated-gpu-targets", "-o", LIB + ".tmp"] + objs + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"])
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
