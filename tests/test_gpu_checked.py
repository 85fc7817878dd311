"""The bounds-checked build of the library (libtpc_b200_checked.so, -DTPC_CHECKED) on small, degenerate and looper inputs.

compute-sanitizer is closed on the GPU pool ("runs under it have left GPUs needing a reset"), so the library carries its own
checks: every data-dependent gather / scatter index in K2, K3, K5 and K6 is tested against the size of its array, and a failed test
makes tpc_find_tracks* return TPC_E_CUDA.  The checked build runs in a subprocess (TPC_B200_LIB selects it) over C1, a looper event,
a continuous frame, both NEXT-2 variants and the degenerate grid cases, and must give the same tracks as the product build.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu

_PROG = r'''
import sys, json
sys.path.insert(0, %r)
import numpy as np
import paper_1905_05515_b200 as T
from gen import workloads as W
from tests import parity as P
lib = T.load_library()
out = {"checked": int(lib.tpc_checked_build())}
rng = np.random.default_rng(5)
cases = [("C1", W.config(1), {}), ("C4@0.3", W.config(4, scale=0.3), {}), ("C3@0.05", W.config(3, scale=0.1), {}),
         ("C1 skip", W.config(1), dict(link_skip=1)), ("C2@0.3 rescue", W.config(2, scale=0.3), dict(bridge_rows=4, bridge_min=3, bridge_rescue=1))]
for name, w, kw in cases:
    with T.Tracker(**P.abi_geometry(w), **kw) as trk:
        trk.load_workload(w)
        r = trk.find_tracks()
        n = int(r.n_tracks)
        trk.refit_tracks(); trk.mark_clusters(1.5); trk.merge_tracks(); trk.find_loopers()
        trk.find_tracks()              # S7..S10 kernels ran with the flag word live: a second call reports what they left
    out[name] = n
print("RESULT " + json.dumps(out))
'''


def _run(lib_path):
    env = dict(os.environ)
    if lib_path:
        env["TPC_B200_LIB"] = lib_path
    r = subprocess.run([sys.executable, "-c", _PROG % ROOT], env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-3000:])
    import json
    return json.loads([l for l in r.stdout.splitlines() if l.startswith("RESULT ")][-1][7:])


def test_checked_build_passes_its_bounds_checks_and_agrees_with_the_product_build():
    checked = os.path.join(ROOT, "paper_1905_05515_b200", "libtpc_b200_checked.so")
    assert os.path.exists(checked), "run `python -m paper_1905_05515_b200.build`"
    a, b = _run(checked), _run(None)
    assert a.pop("checked") == 1 and b.pop("checked") == 0
    assert a == b and all(v > 0 for v in a.values()), (a, b)
