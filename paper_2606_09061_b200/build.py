"""Build libcp.so in-tree for sm_100a (nvcc cross-compiles without a GPU).

  nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo   csrc/cp_api.cu   (kernels + C ABI)
  nvcc (same flags)                                        csrc/cp_static.cu (the no-allocation entry point)
  g++  -ffp-contract=off                                   csrc/cp_sched.cpp (bit-exact fp64)
The result, paper_2606_09061_b200/libcp.so, travels to the GPU box with the snapshot.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INC = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libcp.so")
OBJ = os.path.join(_HERE, "build")

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-I", INC, "-I", CSRC]
CXX_FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-Wall", "-I", INC, "-I", CSRC]


def _sources():
    out = [os.path.join(INC, "cp.h")]
    for f in sorted(os.listdir(CSRC)):
        out.append(os.path.join(CSRC, f))
    return out


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _sources() + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nv = list(NVCC_FLAGS)
    if verbose:
        nv += ["-Xptxas", "-v"]
    nv += os.environ.get("CP_EXTRA_NVCC", "").split()
    objs = []
    cmds = [
        ["nvcc", *nv, "-c", os.path.join(CSRC, "cp_api.cu"), "-o", os.path.join(OBJ, "cp_api.o")],
        ["nvcc", *nv, "-c", os.path.join(CSRC, "cp_static.cu"), "-o", os.path.join(OBJ, "cp_static.o")],
        ["g++", *CXX_FLAGS, "-c", os.path.join(CSRC, "cp_sched.cpp"), "-o", os.path.join(OBJ, "cp_sched.o")],
        ["g++", *CXX_FLAGS, "-c", os.path.join(CSRC, "cp_error.cpp"), "-o", os.path.join(OBJ, "cp_error.o")],
    ]
    for cmd in cmds:
        subprocess.run(cmd, check=True)
        objs.append(cmd[-1])
    subprocess.run(["nvcc", "-shared", "-o", LIB, *objs, "-cudart", "static"], check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
