"""The three oracles and the two seeded input generators under AddressSanitizer + UndefinedBehaviorSanitizer
("-fsanitize=address,undefined on the oracle/generator").  The C sources are compiled a second time with
the sanitizers into a temporary directory; a child Python process loads THOSE libraries (LD_PRELOAD of the sanitizer
runtimes) and runs every entry point on small inputs; the same script run on the regular libraries must print the same
counts and checksums.  No GPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
WORKER = os.path.join(ROOT, "tests", "sanitize_worker.py")
SOURCES = {"libtpc_gen.so": ("datagen/tpc_gen.c", ["-fopenmp"]), "libtpc_fe_gen.so": ("datagen/tpc_fe_gen.c", ["-fopenmp"]),
           "libtpc_cf_oracle.so": ("oracle/tpc_cf_oracle.c", []), "libtpc_ec_oracle.so": ("oracle/tpc_ec_oracle.c", []),
           "libtpc_fe_oracle.so": ("oracle/tpc_fe_oracle.c", [])}


def _runtime(name):
    p = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracles_and_generators_under_asan_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("sanitizer runtimes not installed")
    for so, (src, extra) in SOURCES.items():
        subprocess.check_call(["gcc", "-std=c99", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
                               "-fno-sanitize-recover=undefined", "-fPIC", "-shared", "-Wall"] + extra +
                              ["-o", str(tmp_path / so), os.path.join(ROOT, src), "-lm"])
    plain = subprocess.run([sys.executable, WORKER, "-"], capture_output=True, text=True, timeout=600)
    assert plain.returncode == 0, plain.stderr[-2000:]
    env = dict(os.environ, LD_PRELOAD=asan + ":" + ubsan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="2")
    san = subprocess.run([sys.executable, WORKER, str(tmp_path)], capture_output=True, text=True, timeout=900, env=env)
    assert san.returncode == 0, "sanitizer report or crash:\n" + san.stderr[-4000:]
    assert "runtime error" not in san.stderr and "AddressSanitizer" not in san.stderr, san.stderr[-4000:]
    assert json.loads(san.stdout.strip().splitlines()[-1]) == json.loads(plain.stdout.strip().splitlines()[-1])
