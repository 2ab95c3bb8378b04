"""the host logic of the library that needs no device (murmur_chunk_plan, murmur_batch_plan) and
the plain-C oracle twin, built with AddressSanitizer + UndefinedBehaviorSanitizer (gcc) and run on seeded inputs with
exact-capacity buffers.  (compute-sanitizer for the kernels is closed on this pool - DESIGN.md - so the device half is
not run here.)  No GPU needed."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_host_logic_and_c_oracle_under_asan_ubsan(tmp_path):
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("gcc not found")
    exe = str(tmp_path / "host_sanitize")
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
    objs = []
    for src, lang, extra in ((os.path.join(ROOT, "paper_2606_01483_b200", "csrc", "chunk_plan.cu"), "c++", []),
                             (os.path.join(ROOT, "oracle", "c", "murmur_oracle.c"), "c", ["-std=c99", "-fopenmp"]),
                             (os.path.join(ROOT, "tests", "sanitize", "host_sanitize_main.c"), "c", ["-std=c99"])):
        obj = str(tmp_path / (os.path.basename(src) + ".o"))
        cmd = [gcc, "-x", lang, *san, *extra, "-fvisibility=default", "-I", os.path.join(ROOT, "include"), "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        assert r.returncode == 0, r.stderr
        objs.append(obj)
    r = subprocess.run([gcc, *san, "-fopenmp", "-o", exe, *objs, "-lstdc++", "-lm"], capture_output=True, text=True)
    if r.returncode != 0 and ("asan" in r.stderr or "ubsan" in r.stderr):
        pytest.skip("sanitizer runtimes not installed: " + r.stderr.strip().splitlines()[-1])
    assert r.returncode == 0, r.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == "OK", (r.returncode, r.stdout[-500:], r.stderr[-3000:])
