"""Build libssm.so (the C-ABI library of include/ssm.h) in-tree with nvcc for sm_100a.

    python -m paper_1106_2899_b200.build [--force] [--check]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with gpurun.
"""
import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libssm.so")
LIB_CHECK = os.path.join(_HERE, "libssm_check.so")       # the same sources with -DSSM_CHECK: device-side assertions on
SOURCES = ["ssm_step.cu", "ssm_aux.cu", "ssm_api.cu", "ssm_rheo.cu", "ssm_noalloc.cu"]
STEP_G = [1, 2, 4, 8, 16]       # ssm_step.cu is also compiled once per G (-DSSM_G): the kernels of 8G bead places
OBJ = os.path.join(_HERE, "build")
HEADERS = ["ssm_common.h", "ssm_rng.cuh", os.path.join("..", "..", "include", "ssm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-cudart", "shared"]


def nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libssm.so cannot be built (there is no CPU fallback)")
    return exe


def stale(lib=None):
    lib = lib or LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, check=False):
    """Compile csrc/*.cu into libssm.so (check=True: into libssm_check.so with the device-side assertions of
    ssm_common.h compiled in); returns its path."""
    lib = LIB_CHECK if check else LIB
    if not force and not stale(lib):
        return lib
    from concurrent.futures import ThreadPoolExecutor
    obj = OBJ + ("_check" if check else "")
    os.makedirs(obj, exist_ok=True)
    exe = nvcc()
    extra = ["-DSSM_CHECK"] if check else []
    units = [(f, extra, os.path.join(obj, f[:-3] + ".o")) for f in SOURCES]
    units += [("ssm_step.cu", extra + ["-DSSM_G=%d" % g], os.path.join(obj, "ssm_step_g%d.o" % g)) for g in STEP_G]

    def compile_one(u):
        src, defs, obj = u
        cmd = [exe] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 1)) as ex:
        logs = list(ex.map(compile_one, units))
    cmd = [exe] + NVCC_FLAGS + ["-shared", "-o", lib] + [u[2] for u in units]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc link failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        sys.stderr.write("".join(logs))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, check="--check" in sys.argv))
