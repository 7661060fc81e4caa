"""Builds the in-tree shared libraries with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_00866_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

TARGETS = {
    "libmori.so": (["mori.cu"], sorted(f for f in os.listdir(CSRC) if f.endswith(".cuh"))
                   + [os.path.join(ROOT, "include", "mori.h")]),
    "libmori_workload.so": (["workload_fill.cu"], []),
}


def lib_path(name="libmori.so"):
    return os.path.join(HERE, name)


def build(force=False, verbose=False):
    for name, (srcs, deps) in TARGETS.items():
        out = lib_path(name)
        srcs_abs = [os.path.join(CSRC, s) for s in srcs]
        deps_abs = srcs_abs + [d if os.path.isabs(d) else os.path.join(CSRC, d) for d in deps]
        if (not force and os.path.exists(out)
                and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps_abs)):
            continue
        tmp = out + f".tmp{os.getpid()}"
        cmd = [NVCC] + FLAGS + srcs_abs + ["-o", tmp]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}")
        os.replace(tmp, out)
    return lib_path()


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
