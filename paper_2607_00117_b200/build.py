"""Build libschwarmax.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libschwarmax.so")
SOURCES = ["schwarmax.cu", "ferrers_table.cpp"]
DEPS = SOURCES + ["api_build.inc", "api_entry.inc", "api_weights.inc", "weights.cuh", "kernels.cuh", "rowbuild.cuh", "force.cuh", "ferrers.cuh", "dehnen.cuh", "rk32.cuh", "api_rk32.inc",
                  "ferrers_table.h", os.path.join("..", "..", "include", "schwarmax.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc_path():
    for c in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    raise RuntimeError("nvcc not found")


def build_library(force=False, verbose=False):
    deps = [os.path.join(CSRC, d) for d in DEPS]
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in deps):
        return SO
    cmd = [nvcc_path()] + NVCC_FLAGS + os.environ.get("SMX_EXTRA_NVCC_FLAGS", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    env = dict(os.environ)
    if os.path.exists("/usr/bin/g++"):
        cmd[1:1] = ["-ccbin", "/usr/bin/g++"]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout[-2000:] + r.stderr[-4000:])
    if verbose:
        print(r.stderr)
    return SO


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
