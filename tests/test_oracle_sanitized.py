"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (`-fsanitize=address,undefined` for
the oracle).  oracle/rk4ip_oracle.cpp is compiled once more with the sanitizers on and the pin tests are run against
that build in a child process (the sanitizer runtime has to be loaded before python: LD_PRELOAD).  Any heap overflow,
use after free, misaligned access, signed overflow or out-of-range shift in the oracle aborts the child."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_pins_pass_under_asan_and_ubsan(tmp_path):
    lib = str(tmp_path / "liboracle_san.so")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-fPIC", "-shared", "-pthread", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-o", lib,
                    os.path.join(ROOT, "oracle", "rk4ip_oracle.cpp")], check=True)
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True, check=True).stdout.strip()
    ubsan = subprocess.run(["gcc", "-print-file-name=libubsan.so"], capture_output=True, text=True, check=True).stdout.strip()
    env = dict(os.environ, MMF_ORACLE_LIB=lib, LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    # the pins of every oracle function; the two long ones (step-size table, 2^22 transform) add nothing for this purpose
    out = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                          "tests/test_oracle_pins.py", "tests/test_oracle_ssfm_pins.py", "tests/test_oracle_general_pins.py", "tests/test_oracle_noise_pins.py",
                          "-k", "not stepsize_table_claim and not full_length"],
                         cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    tail = out.stdout[-3000:] + out.stderr[-3000:]
    assert out.returncode == 0, tail
    assert "passed" in out.stdout and "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail, tail
