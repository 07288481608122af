"""Builds libgnn.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2312_06838_b200.build [--force]

The shipped library reads no environment variable at run time.  Developer builds: extra nvcc flags come from the build-time
variable GNN_NVCC_DEFS, e.g. GNN_NVCC_DEFS="-DGNN_DEV_KNOBS" compiles in the A/B switches GNN_NO_POOL_FUSE, GNN_NO_GRAPHS,
GNN_NO_PDL and GNN_EDGE_CHUNK (csrc/api.cu, csrc/edgeconv_bf16.cu), "-DEDGE_CWE_256=64" changes an epilogue tile shape.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgnn.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC",
         "-Xcompiler", "-pthread", "--use_fast_math=false"]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cpp")))


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    deps.append(os.path.join(HERE, "..", "include", "gnn.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    flags = [f for f in FLAGS if not f.startswith("--use_fast_math")] + os.environ.get("GNN_NVCC_DEFS", "").split()
    objs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    procs = []
    for src in sources():
        obj = os.path.join(HERE, "build", os.path.basename(src) + ".o")
        objs.append(obj)
        cmd = [NVCC] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-x", "cu", "-c", src, "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.check_call([NVCC] + flags + ["-shared", "-o", tmp] + objs + ["-lcudart", "-lcuda"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
