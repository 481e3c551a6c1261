"""heget_xsec_reduce_noalloc: the cross-section reduction for callers that cannot allocate (CUDA graph capture,
serving loops).  Its block partials live in a file-scope `static __device__` array of libheget.so (96 KB per GPU,
N <= HEGET_NOALLOC_MAX_EVENTS = 2^24), whose device address the library resolves with cudaGetSymbolAddress.

Collected last on purpose (file name): the suite runs with `pytest -x`, so a failure here hides nothing.
The test stands alone (its own context, its own inputs) and must pass in a fresh process and after the others."""
import numpy as np
import pytest
import torch

from paper_0908_4403_b200 import Heget, HegetError, workloads

pytestmark = pytest.mark.gpu

TOL = 1e-13          # the tolerance of test_xsec_reduce_matches_oracle_and_is_deterministic
MAX_EVENTS = 1 << 24


def inputs(N, seed, scale):
    rng = np.random.default_rng(seed)
    a = rng.uniform(0.5, 2.0, size=N) * scale
    w = rng.uniform(0.0, 1.0, size=N)
    w[::3] = 0.0                                   # events that failed the cuts
    a[::21] = np.nan                               # ... whose amp2 must not matter (R26)
    return torch.from_numpy(a).cuda(), torch.from_numpy(w).cuda()


def test_noalloc_reduce_matches_the_existing_path_on_two_calls_in_a_row():
    hg = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    try:
        out3 = torch.empty(3, dtype=torch.float64, device="cuda")
        # the second batch is smaller than the first: stale partials of call 1 stay in the shared array and
        # must not leak into call 2; a ragged size, an exact multiple of the 4,096-event chunk, one event, none
        for N, seed, scale in ((1_000_003, 1, 1e-7), (4096 * 3, 2, 1e-3), (1, 3, 1.0), (0, 4, 1.0)):
            a, w = inputs(N, seed, scale)
            ref = hg.xsec_reduce(a, w, 5).cpu().numpy()
            before = torch.cuda.memory_allocated()
            got = hg.xsec_reduce_noalloc(a, w, 5, out3)
            assert torch.cuda.memory_allocated() == before          # nothing allocated through torch either
            got = got.cpu().numpy()
            assert np.all(np.isfinite(got)) and got[2] == ref[2]
            for k in (0, 1):
                assert abs(got[k] - ref[k]) <= TOL * abs(ref[k]), (N, k, got[k], ref[k])
            again = hg.xsec_reduce_noalloc(a, w, 5, out3).cpu().numpy()   # fixed reduction tree: bit-reproducible
            assert np.array_equal(again, got)
        # on a side stream, ordered after the work above
        a, w = inputs(300_001, 5, 1e-5)
        ref = hg.xsec_reduce(a, w, 4).cpu().numpy()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            got = hg.xsec_reduce_noalloc(a, w, 4, out3)
        s.synchronize()
        got = got.cpu().numpy()
        assert got[2] == ref[2] and abs(got[0] - ref[0]) <= TOL * abs(ref[0]) and abs(got[1] - ref[1]) <= TOL * abs(ref[1])
    finally:
        hg.close()


def test_noalloc_reduce_rejects_batches_beyond_its_scratch():
    hg = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    try:
        out3 = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")
        big = torch.ones(MAX_EVENTS + 1, dtype=torch.float64, device="cuda")
        launches = hg.launch_count()
        with pytest.raises(HegetError, match="HEGET_NOALLOC_MAX_EVENTS"):
            hg.xsec_reduce_noalloc(big, big, 2, out3)
        assert hg.launch_count() == launches and torch.all(out3 == -7.0)     # rejected before anything ran
        assert hg._lib.heget_xsec_reduce_noalloc(hg._ctx, big.data_ptr(), big.data_ptr(), 2, MAX_EVENTS + 1,
                                                 out3.data_ptr(), None) == -4
        # the maximum itself is accepted: N = 2^24 ones with weight 1 -> count = N, sum = N / (4 * 9 * 2!)
        got = hg.xsec_reduce_noalloc(big[:MAX_EVENTS], big[:MAX_EVENTS], 2, out3).cpu().numpy()
        assert got[2] == MAX_EVENTS and abs(got[0] / (MAX_EVENTS / 72.0) - 1.0) < 1e-13
    finally:
        hg.close()
