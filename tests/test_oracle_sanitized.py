"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: its C sources
are built a second time with -fsanitize=address,undefined into a temporary directory and every pin of
the oracle (closed forms, invariants, Jacobian derivatives, the approximate-ANN layer) runs against that
build in a child process with libasan preloaded.  An out-of-bounds index, a use of uninitialised stack
through a wrong length, a signed overflow or a misaligned access in the checker would otherwise be able
to hide behind values that happen to come out right."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PIN_FILES = ["tests/test_oracle_closed_forms.py", "tests/test_oracle_invariants.py",
             "tests/test_oracle_jacobian.py", "tests/test_oracle_ann.py"]


def test_oracle_pins_pass_under_address_and_ub_sanitizers(tmp_path):
    from oracle import build as obuild
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("this gcc ships no libasan")
    lib = obuild.build_sanitized(str(tmp_path))
    env = dict(os.environ, CK_ORACLE_LIB=lib, LD_PRELOAD=os.path.realpath(asan),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=99",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1:exitcode=98")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"]
                       + PIN_FILES, cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout[-3000:] + "\n" + r.stderr[-3000:])
    assert r.returncode == 0, tail
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, tail
    assert " passed" in r.stdout and "failed" not in r.stdout, tail
    # the child really ran on the sanitizer build
    probe = subprocess.run([sys.executable, "-c",
                            "import oracle; oracle._load(); "
                            "print(open('/proc/self/maps').read().count('libck_oracle_san.so') > 0)"],
                           cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert probe.returncode == 0 and probe.stdout.strip().endswith("True"), probe.stdout + probe.stderr
