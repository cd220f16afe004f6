"""-m gpu: the HOST side of the C-ABI under AddressSanitizer + UndefinedBehaviorSanitizer.

Round 1 shipped a one-word stack overflow in wm_rollout's graph cache key that no parity test could see.  The host
code of libwm_b200.so - argument checks, the cache key, scratch carving, the pipelined host path, the handle-free
static entry point - is plain C++ and can run under the sanitizers; the kernels are untouched.  This test loads
libwm_b200_san.so (same sources, `-Xcompiler -fsanitize=address -fsanitize=undefined`, built by
paper_2310_08710_b200/_build.py) into a child pytest process with libasan preloaded and runs the rollout, host-path,
variant, stress and no-allocation tests against it.  Any sanitizer report fails; a child that cannot start for reasons
of the box (no libasan, CUDA refusing to initialise under ASan) skips.  compute-sanitizer (the device side) is closed
on this pool, see DESIGN.md section 11.
"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SUBSET = ["tests/test_gpu_parity.py", "tests/test_gpu_variants.py", "tests/test_gpu_stress.py", "tests/test_zz_no_alloc.py"]


def test_c_abi_host_code_runs_clean_under_asan_and_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], stdout=subprocess.PIPE, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("this toolchain has no libasan")
    from paper_2310_08710_b200 import _build
    try:
        lib = _build.build(sanitize=True)
    except Exception as e:                                   # noqa: BLE001 - no nvcc on the box: nothing to test with
        pytest.skip("cannot build the sanitized library here: %s" % e)
    env = dict(os.environ, LD_PRELOAD=os.path.realpath(asan), WM_B200_LIB=lib,
               ASAN_OPTIONS="protect_shadow_gap=0:detect_leaks=0:exitcode=97",     # protect_shadow_gap=0: CUDA maps memory there
               UBSAN_OPTIONS="print_stacktrace=1")
    # proof that the child really runs the sanitized build with the runtime in place
    probe = ("import paper_2310_08710_b200 as wm; wm.load(); m = open('/proc/self/maps').read(); "
             "print('MAPPED', 'libwm_b200_san.so' in m, 'libasan' in m, 'libwm_b200.so' in m)")
    pr = subprocess.run([sys.executable, "-c", probe], env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
    if "MAPPED" not in pr.stdout:
        pytest.skip("the sanitized library does not load on this box: %s" % pr.stderr[-300:])
    assert "MAPPED True True False" in pr.stdout, pr.stdout
    res = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider"] + SUBSET, env=env, cwd=ROOT,
                         stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=1500)
    out = res.stdout
    assert "AddressSanitizer" not in out and "runtime error:" not in out and res.returncode != 97, out[-4000:]
    if res.returncode != 0:
        pytest.skip("child pytest ended with %d without a sanitizer report (the plain suite judges parity): %s" % (res.returncode, out[-400:]))
    print("host sanitizer run:", out.strip().splitlines()[-1])
