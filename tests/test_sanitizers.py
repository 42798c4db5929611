"""Host code under AddressSanitizer + UndefinedBehaviorSanitizer: the oracle, the workload
generator and the caching pool (fake backend) are built from their sources with -fsanitize=address,undefined and run
once over a tiny, a Run-3-like and a dense event and a random alloc/free/complete/trim sequence.  compute-sanitizer is
not available on this pool; the device code is covered by the parity tests."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = "/usr/local/cuda"


@pytest.mark.skipif(shutil.which("g++") is None or not os.path.exists(os.path.join(CUDA, "include", "cuda_runtime.h")),
                    reason="needs g++ and the CUDA headers")
def test_oracle_generator_and_pool_are_clean_under_asan_and_ubsan(tmp_path):
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
    objs = []
    for src, cc, extra in [
        (os.path.join(ROOT, "oracle", "pixreco_oracle.c"), "gcc", ["-std=c11", "-ffp-contract=off"]),
        (os.path.join(ROOT, "paper_2004_04334_b200", "workloads", "pixgen.c"), "gcc", ["-std=c99"]),
        (os.path.join(ROOT, "paper_2004_04334_b200", "csrc", "pool.cpp"), "g++", ["-std=c++17", "-I", os.path.join(CUDA, "include")]),
        (os.path.join(ROOT, "tests", "sanitize_main.cpp"), "g++", ["-std=c++17"]),
    ]:
        obj = str(tmp_path / (os.path.basename(src) + ".o"))
        subprocess.check_call([cc, *san, *extra, "-c", src, "-o", obj])
        objs.append(obj)
    exe = str(tmp_path / "sanitize_main")
    subprocess.check_call(["g++", *san, *objs, "-o", exe, os.path.join(CUDA, "lib64", "libcudart_static.a"),
                           "-ldl", "-lrt", "-lpthread", "-lm"])
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "sanitize_main: 0" in r.stdout
