"""the oracle built under AddressSanitizer + UndefinedBehaviorSanitizer and walked through every entry
point of oracle/mfo.h (oracle/sanitize_main.cpp) on all processes, edge sizes included.  CPU only.  The GPU side has no
compute-sanitizer on this pool, so this is the memory-safety evidence that can be produced here; it
covers the checker the parity claims rest on."""
import os
import shutil
import struct
import subprocess

import numpy as np
import pytest

from paper_2106_10279_b200 import workloads as W

ORACLE = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "oracle")


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "sanitize_main")
    cmd = ["g++", "-std=gnu++17", "-O1", "-g1", "-fno-omit-frame-pointer", "-ffp-contract=off",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-o", exe,
           os.path.join(ORACLE, "sanitize_main.cpp"), os.path.join(ORACLE, "mfo.cpp"), "-lquadmath"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout[-4000:]
    lnx, lnq2, xf = W.pdf_table_flavours()
    table = str(tmp_path / "table.bin")
    with open(table, "wb") as f:
        f.write(struct.pack("<3i", xf.shape[0], len(lnx), len(lnq2)))
        for a in (lnx, lnq2, xf):
            f.write(np.ascontiguousarray(a, dtype="<f8").tobytes())
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe, table], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-6000:])
    assert "sanitize_main: ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr and "LeakSanitizer" not in r.stderr
