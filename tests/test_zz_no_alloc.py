"""GPU test of tpc_find_loopers_noalloc (include/tpc.h): S10 for callers that cannot call cudaMalloc.  Its scratch is a file-scope
static __device__ array of csrc/k10_loopers.cu, shared by every call on the device and never cleared, so the test makes TWO calls in a
row -- first the larger track list (C4, 6 k tracks), then a smaller one (C4 at scale 0.3, 1.7 k tracks) that leaves the first call's
words behind it in the array -- and compares each with the existing, allocating path tpc_find_loopers on the same tracks.  The outputs are int32 indices and
turn counts: the bar is equality, as in test_gpu_parity.py::test_looper_turns_parity_c4_and_c3_scaled.

The file name sorts after every other test file on purpose: the suite runs with pytest -x, and a failure here must not hide the
parity tests.  It holds no state of its own and passes alone in a fresh process as well as after the other files.
"""
import numpy as np
import pytest

from gen import workloads as W
from tests import parity as P

pytestmark = pytest.mark.gpu


def _tracks_and_existing_result(T, w):
    """S0-S6 on w, then the existing S10 path; owning device copies of (sector, x, par) and of its (prev, root, turn)."""
    trk = T.Tracker(**P.abi_geometry(w))
    trk.load_workload(w)
    t = trk.find_tracks_device()
    n = t.n_tracks
    sector, x, par = t.sector.clone(), t.x.clone(), t.par.clone().contiguous()
    ref = trk.find_loopers(device_result=True)
    assert ref["n_tracks"] == n
    ref = {k: ref[k].clone() for k in ("prev", "root", "turn")}
    return trk, n, sector, x, par, ref


def test_noalloc_loopers_equal_the_allocating_path_on_two_calls_in_a_row():
    import torch
    import paper_1905_05515_b200 as T
    from paper_1905_05515_b200 import binding as B

    cases = [_tracks_and_existing_result(T, W.config(4)), _tracks_and_existing_result(T, W.config(4, scale=0.3))]
    try:
        assert cases[0][1] > cases[1][1] > 1000 and cases[0][1] <= B.NOALLOC_MAX_TRACKS
        assert int((cases[0][5]["prev"] >= 0).sum()) > 1000 and int((cases[1][5]["prev"] >= 0).sum()) > 100   # there is something to find
        # outputs are pre-filled with a value S10 never writes, so a word the kernels skip shows up
        outs = [{k: torch.full((n,), -7, dtype=torch.int32, device="cuda") for k in ("prev", "root", "turn")} for _, n, *_ in cases]
        for rep in range(2):                                   # the pair of calls, twice: large, small, large, small
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            for (trk, n, sector, x, par, _), o in zip(cases, outs):
                trk.find_loopers_noalloc(n, sector, x, par, o["prev"], o["root"], o["turn"])    # queued on the same stream, no sync between
            torch.cuda.synchronize()
            # no device memory was taken from the driver between the two synchronisations (only the library ran there: torch's own
            # kernels load their modules lazily on first use, which is why the comparison below is outside the bracket)
            assert torch.cuda.mem_get_info()[0] == free_before
            for (_, n, _, _, _, ref), o in zip(cases, outs):
                for k in ("prev", "root", "turn"):
                    assert torch.equal(o[k], ref[k]), (rep, n, k, int((o[k] != ref[k]).sum()))
                    if rep == 0:
                        o[k].fill_(-7)
            torch.cuda.synchronize()

        # a context that never ran tpc_find_tracks* gives the same answer (the entry point needs only geometry, field and tunables)
        trk0, n0, sector0, x0, par0, ref0 = cases[0]
        with T.Tracker(**P.abi_geometry(W.config(4))) as fresh:
            o = {k: torch.full((n0,), -7, dtype=torch.int32, device="cuda") for k in ("prev", "root", "turn")}
            fresh.find_loopers_noalloc(n0, sector0, x0, par0, o["prev"], o["root"], o["turn"])
            torch.cuda.synchronize()
            assert all(torch.equal(o[k], ref0[k]) for k in o)

        # sizes beyond the static array are rejected with a clear error and nothing is launched
        o = outs[0]
        for k in o:
            o[k].fill_(-7)
        with pytest.raises(T.TpcError) as e:
            trk0.find_loopers_noalloc(B.NOALLOC_MAX_TRACKS + 1, sector0, x0, par0, o["prev"], o["root"], o["turn"])
        assert e.value.code == -5 and "TPC_NOALLOC_MAX_TRACKS" in str(e.value) and str(B.NOALLOC_MAX_TRACKS) in str(e.value)
        torch.cuda.synchronize()
        assert all(bool((o[k] == -7).all()) for k in o)
        # arrays that break the contract (sectors shuffled, some out of range) give a meaningless grouping but no fault, and the next
        # correct call is right again (the scratch keeps nothing that matters from the bad call)
        g = torch.Generator(device="cuda"); g.manual_seed(5)
        bad = sector0[torch.randperm(n0, device="cuda", generator=g)].clone()
        bad[::7] = 1000
        bad[1::11] = -3
        trk0.find_loopers_noalloc(n0, bad, x0, par0, o["prev"], o["root"], o["turn"])
        torch.cuda.synchronize()
        assert bool(((o["prev"] >= -1) & (o["prev"] < n0)).all())
        trk0.find_loopers_noalloc(n0, sector0, x0, par0, o["prev"], o["root"], o["turn"])
        torch.cuda.synchronize()
        assert all(torch.equal(o[k], ref0[k]) for k in o)
        # host memory is not accepted; n_tracks = 0 is a no-op; negative n_tracks is an argument error
        host = np.zeros(n0, np.int32)
        with pytest.raises(T.TpcError) as e:
            trk0.find_loopers_noalloc(n0, sector0, x0, par0, host.ctypes.data, o["root"], o["turn"])
        assert e.value.code == -1
        trk0.find_loopers_noalloc(0, None, None, None, None, None, None)
        with pytest.raises(T.TpcError) as e:
            trk0.find_loopers_noalloc(-1, sector0, x0, par0, o["prev"], o["root"], o["turn"])
        assert e.value.code == -1
    finally:
        for c in cases:
            c[0].close()
