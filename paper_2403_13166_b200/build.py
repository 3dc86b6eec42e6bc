"""Build the C-ABI shared library (liblst_b200.so) for sm_100a with nvcc, in-tree."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "liblst_b200.so")
SOURCES = [os.path.join(CSRC, "lst_api.cu"), os.path.join(CSRC, "lst_static.cu")]
HEADERS = [os.path.join(CSRC, "lst_kernels.cuh"), os.path.join(CSRC, "lst_math.cuh"), os.path.join(CSRC, "lst_pairs.cuh"), os.path.join(CSRC, "lst_tuples.cuh"),
           os.path.join(_HERE, "..", "include", "lst.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if p and os.path.exists(p):
            return p
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [nvcc_path(), *NVCC_FLAGS, "-o", LIB, *SOURCES]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            print(res.stdout)
            print(res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        with open(LIB + ".ptxas.log", "w") as f:              # ptxas -v output next to the library (git-ignored)
            f.write(" ".join(cmd) + "\n" + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
