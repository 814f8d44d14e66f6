"""the host-side code under AddressSanitizer + UndefinedBehaviorSanitizer (no GPU).

The mask scheduler (csrc/schedule.cpp: lowering, tiling, worker assignment -- index arithmetic over caller-supplied arrays) and
the fp64 oracle are rebuilt as host-only libraries with `-fsanitize=address,undefined -fno-sanitize-recover`, and the
scheduler's rasterisation tests and the oracle's pins are run against those builds in a child interpreter (the sanitizer
runtimes have to be loaded before Python).  A heap overflow, a use after free, a signed overflow or a misaligned access
anywhere in them aborts the child and fails this test.
"""
import os
import subprocess
import sys

import pytest

from paper_2606_25473_b200 import binding as aj

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2606_25473_b200", "csrc")
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g", "-O1"]


def _runtime(name):
    path = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


CHILD = r"""
import sys
sys.path.insert(0, {root!r}); sys.path.insert(0, {tests!r})
from paper_2606_25473_b200 import binding, build
binding.LIB_PATH = {lib!r}                    # the sanitized host-only build
build.build_library = lambda *a, **k: {lib!r}
import oracle
oracle.build = lambda force=False: {ora!r}
import pytest
# tests of the CUDA part of the ABI (plans, the export list of the real library) do not apply to the host-only build
sys.exit(pytest.main(["-q", "-x", "-p", "no:cacheprovider", "-m", "not gpu", "-k", "not plan and not export and not static"] + {targets!r}))
"""


def test_scheduler_and_oracle_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc's sanitizer runtimes are not installed")
    # every ABI symbol that lives in the CUDA part of the library becomes a stub that refuses, so that the binding loads
    in_schedule = subprocess.run(["grep", "-ohE", r"^(aj_status|const char \*)\s*attn_\w+|^\w[\w \*]*\battn_jvp_(last_error|version)\b",
                                  os.path.join(CSRC, "schedule.cpp")], capture_output=True, text=True).stdout
    have = {tok for line in in_schedule.splitlines() for tok in line.replace("*", " ").split() if tok.startswith("attn_")}
    stubs = "\n".join(f'extern "C" int {s}() {{ return -2; }}' for s in aj.SYMBOLS if s not in have)
    (tmp_path / "stubs.cpp").write_text(stubs + "\n")
    lib = str(tmp_path / "libattn_jvp_host_san.so")
    subprocess.run(["g++", "-std=c++17", "-fPIC", "-shared", *SAN, "-I", os.path.join(ROOT, "include"), "-I", CSRC,
                    os.path.join(CSRC, "schedule.cpp"), str(tmp_path / "stubs.cpp"), "-o", lib], check=True)
    ora = str(tmp_path / "libattn_jvp_oracle_san.so")
    subprocess.run(["gcc", "-std=c11", "-fopenmp", "-fPIC", "-shared", *SAN, os.path.join(ROOT, "oracle", "attn_jvp_oracle.c"),
                    "-o", ora, "-lm"], check=True)
    targets = [os.path.join(ROOT, "tests", "test_schedule_host.py"),
               os.path.join(ROOT, "tests", "test_oracle_pins.py"),
               os.path.join(ROOT, "tests", "test_oracle_bwd_pins.py")]
    env = dict(os.environ, LD_PRELOAD=f"{asan}:{ubsan}", ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", OMP_NUM_THREADS="4",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    code = CHILD.format(root=ROOT, tests=os.path.join(ROOT, "tests"), lib=lib, ora=ora, targets=targets)
    r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, cwd=ROOT, timeout=900)
    tail = (r.stdout[-3000:] + "\n" + r.stderr[-3000:])
    assert r.returncode == 0, f"the sanitized run failed (exit {r.returncode}):\n{tail}"
    assert "passed" in r.stdout and "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, tail
