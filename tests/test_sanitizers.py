"""Sanitizer pass over the host side of libfcp: fcp_plan.cpp and
fcp_sched.cpp are compiled with g++ -fsanitize=address,undefined (no nvcc, no GPU; the device
entry points are stubs) and the bit-exact planner / layout / schedule-list tests are run against
that build in a child process with the sanitizer runtimes preloaded.  Any heap overflow,
use-after-free, signed overflow, misaligned access ... aborts the child."""
import os
import shutil
import subprocess
import sys

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(ROOT, "paper_2606_08476_b200", "csrc")


def _gcc_file(name):
    out = subprocess.run(["gcc", "-print-file-name=" + name], stdout=subprocess.PIPE, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_host_sources_under_asan_ubsan(tmp_path):
    asan, ubsan = _gcc_file("libasan.so"), _gcc_file("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("sanitizer runtimes not installed")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    lib = str(tmp_path / "libfcp_host_san.so")
    cmd = ["g++", "-std=c++17", "-O1", "-g", "-fno-omit-frame-pointer", "-fPIC", "-shared",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-I", os.path.join(cuda, "include"),
           os.path.join(CSRC, "fcp_plan.cpp"), os.path.join(CSRC, "fcp_sched.cpp"),
           os.path.join(HERE, "asan_device_stubs.cpp"),
           "-L", os.path.join(cuda, "lib64"), "-lcudart", "-Wl,-rpath," + os.path.join(cuda, "lib64"),
           "-o", lib]
    subprocess.run(cmd, check=True)
    env = dict(os.environ, FCP_LIB=lib, LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        os.path.join(HERE, "test_plan_parity.py"), os.path.join(HERE, "test_sched_lists.py")],
                       cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    tail = r.stdout[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in tail and "ERROR: AddressSanitizer" not in r.stdout and "runtime error" not in r.stdout, tail
