"""Build libgammanav.so (the CUDA C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_1209_5235_b200.build [--force]

Flags: -gencode arch=compute_100a,code=sm_100a -lineinfo -O3; --fmad=false and host -ffp-contract=off keep
the canonical arithmetic of the navigator (no contraction, explicit fma only); division
and square root stay IEEE (no -use_fast_math)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("GN_LIB_OUT") or os.path.join(HERE, "libgammanav.so")      # GN_LIB_OUT: build a variant beside the product (diagnostics)
SOURCES = ["transport_f32_box.cu", "transport_f32_gen.cu", "transport_f64_box.cu", "transport_f64_gen.cu", "nav_f32.cu", "nav_f64.cu", "noalloc.cu", "api.cu", "geometry.cu"]
HEADERS = ["store.h", "geometry.h", "hostmath.h", "impl.h", "common.cuh", "nav.cuh", "physics.cuh", "nav_kernels.cuh", "transport.cuh", "voxel_pass.cuh", "coherent.cuh",
           os.path.join("..", "..", "include", "gammanav.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "--fmad=false",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-Xptxas", "-v"]


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("GN_NVCC_EXTRA", "").split() + ["-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError(f"nvcc failed on {src}")
    subprocess.run([nvcc, "-shared", "-o", LIB] + objs + ["-lcudart"], check=True)
    with open(os.path.join(CSRC, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
