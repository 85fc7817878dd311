"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer ("oracle built with
-fsanitize=address,undefined in tests").  The sanitized library is built next to the normal one and exercised in a subprocess
(libasan has to be the first library of the process): full S0..S9 on a C1-shaped input at 10 % plus a continuous-mode frame, the
pick-up / link hooks, and the empty input.  Any report makes the subprocess exit non-zero."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_PROG = r'''
import sys
sys.path.insert(0, %r)
import numpy as np
from gen import workloads as W
from oracle import oracle
from tests import parity as P
so = oracle.build_sanitized()
w = W.config(1, scale=0.1)
for k, ww in enumerate((w, W.config(3, scale=0.1).sector_slice([19]), W.config(4, scale=0.03))):
    o = oracle.Oracle(lib=so, **P.abi_geometry(ww)); o.load(ww.unit_off, ww.y, ww.t); o.run("s9")
    n = len(o.tracks()["sector"])
    if k == 0:
        b = oracle.Oracle(lib=so, **P.abi_geometry(ww)); b.load(ww.unit_off, ww.y, ww.t); b.run("s6", brute_links=True, brute_pickup=True)
        assert np.array_equal(o.get("clean_up"), b.get("clean_up")) and n == len(b.tracks()["sector"])
    print(ww.name, ww.n_clusters, n)
e = oracle.Oracle(lib=so, **P.abi_geometry(w)); e.load(np.zeros_like(w.unit_off), w.y[:0], w.t[:0]); e.run("s9")
assert len(e.tracks()["sector"]) == 0
o = oracle.Oracle(lib=so, bridge_rows=4, bridge_min=3, bridge_rescue=1, **P.abi_geometry(w)); o.load(w.unit_off, w.y, w.t); o.run("s6")
print("ok")
'''


def test_oracle_is_clean_under_asan_and_ubsan():
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-c", _PROG % ROOT], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip().endswith("ok"), (r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
