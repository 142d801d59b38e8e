"""The host oracle under AddressSanitizer and UBSan ("host oracle under -fsanitize=address,undefined").

oracle/oracle.cpp and the small driver oracle/sanitize_main.cpp are compiled with -fsanitize=address,undefined
-fno-sanitize-recover=all into a temporary directory and run on a few seeded events of every process the oracle knows; any
out-of-bounds access, use of uninitialised stack through a pointer past a buffer, signed overflow or misaligned access ends the run with a
non-zero exit code.  The numbers that come back must be those of the regular build (liboracle.so), so the instrumented run
exercised the same code.  CPU only; the oracle is test infrastructure and so is this."""
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import events as ev

ORACLE_DIR = os.path.dirname(os.path.abspath(orc.__file__))
# (config index or photon count, events): the heavy processes get fewer events (an instrumented gg -> tt ggg evaluation takes seconds)
CASES = [(1, 6), (2, 6), (3, 4), (4, 2), (5, 1), (7, 6), (8, 4), ("epem_aa", 4), ("epem_aaaaa", 2)]


@pytest.fixture(scope="module")
def sanitized_binary(tmp_path_factory):
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    exe = str(tmp_path_factory.mktemp("oracle_san") / "oracle_san")
    cmd = ["g++", "-O1", "-g", "-std=c++17", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-o", exe,
           os.path.join(ORACLE_DIR, "oracle.cpp"), os.path.join(ORACLE_DIR, "sanitize_main.cpp")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and ("asan" in r.stderr.lower() or "ubsan" in r.stderr.lower()):
        pytest.skip("sanitizer runtime not installed: " + r.stderr[-200:])
    assert r.returncode == 0, r.stderr[-2000:]
    return exe


def config_of(case):
    if isinstance(case, str):
        return ev.photon_config(len(case) - len("epem_"), 64)
    return ev.config(case)


@pytest.mark.parametrize("case,n", CASES)
def test_oracle_event_loop_is_clean_under_asan_and_ubsan(sanitized_binary, tmp_path, case, n):
    c = config_of(case)
    m, w = ev.generate(c, n)
    fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(fin, "wb") as f:
        for a in (c.params_old, c.params_new, np.ascontiguousarray(m), w):
            f.write(np.asarray(a, dtype="<f8").tobytes())
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", OMP_NUM_THREADS="2")
    r = subprocess.run([sanitized_binary, c.process, str(c.n_ext), str(n), fin, fout], capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0, (c.process, r.returncode, r.stderr[-3000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
    got = np.fromfile(fout, dtype="<f8").reshape(3, n)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    for g, ref in zip(got, (a, b, wn)):
        assert np.all(np.isfinite(g)) and np.abs(g / ref - 1).max() < 1e-12          # -O1 vs -O2: contraction may differ in the last bits
