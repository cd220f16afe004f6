"""In-tree build of the CUDA C-ABI library (libwm_b200.so) for sm_100a with nvcc.

nvcc cross-compiles without a GPU; the built .so sits beside this file so that it travels
to the GPU box with the repository snapshot.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libwm_b200.so")
SOURCES = ["wm_api.cu", "wm_dynamics.cu", "wm_overlap.cu", "wm_offroad.cu", "wm_grid.cu", "wm_rollout_fused.cu", "wm_observe.cu", "wm_variants.cu"]
HEADERS = [os.path.join(CSRC, "wm_internal.cuh"), os.path.join(CSRC, "wm_grid.cuh"), os.path.join(CSRC, "wm_device.cuh"), os.path.join(_HERE, "..", "include", "wm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


# The same sources with the HOST code under AddressSanitizer + UndefinedBehaviorSanitizer (device code is unchanged):
# tests/test_zy_host_sanitizer.py runs the C-ABI's host logic (argument checks, graph cache key, scratch carving,
# host staging) under it on the GPU box.  Never loaded by default.
LIB_SAN = os.path.join(_HERE, "libwm_b200_san.so")
SAN_FLAGS = ["-Xcompiler", "-fsanitize=address", "-Xcompiler", "-fsanitize=undefined", "-Xcompiler", "-fno-omit-frame-pointer", "-g"]   # (nvcc splits -Xcompiler arguments at commas)


def _stale(lib=LIB):
    if not os.path.exists(lib):
        return True
    m = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > m for d in deps)


def build(force=False, verbose=False, sanitize=False):
    """Compile every kernel for sm_100a into one shared library. Returns its path."""
    lib = LIB_SAN if sanitize else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (SAN_FLAGS if sanitize else []) + ["-o", lib] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building %s" % os.path.basename(lib))
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True))
