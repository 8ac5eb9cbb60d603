"""Build the CPU oracle shared library (test infrastructure; building it is not using it).

Run as a script or call build_oracle().  Tries $CXX, /usr/bin/g++, g++ in turn, first with
OpenMP, then without (some compiler wrappers in this image lack libgomp.spec).
"""
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libsm_oracle.so")
SRC = [os.path.join(HERE, "sm_oracle.cpp"), os.path.join(HERE, "sm_oracle.h"), os.path.join(HERE, "sm_oracle_forces.inc")]
FLAGS = ["-O2", "-ffp-contract=off", "-fPIC", "-std=gnu++17", "-fext-numeric-literals", "-Wall", "-Wextra", "-shared"]


def build_oracle(force=False):
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(s) for s in SRC):
        return SO
    cands = [c for c in (os.environ.get("SMO_CXX"), "/usr/bin/g++", os.environ.get("CXX"), shutil.which("g++")) if c]
    errs = []
    for omp in (["-fopenmp"], []):
        for cxx in cands:
            cmd = [cxx] + FLAGS + omp + ["-o", SO, SRC[0], "-lquadmath"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode == 0:
                return SO
            errs.append(" ".join(cmd) + "\n" + r.stderr[-400:])
    raise RuntimeError("could not build the oracle:\n" + "\n".join(errs))


if __name__ == "__main__":
    print(build_oracle(force=True))
