"""GPU parity on the event subsets BASELINE.json `configs` state: EVERY one of the first 4,096 events of
the 7-photon config, the first 512 of the 8-photon config and the first 2,048 of the 6-photon config,
element by element against stored oracle values (tests/golden/amp2_<config>.npz, written by
tests/golden/make_amp2_golden.py from oracle/ alone; tests/test_golden_sets.py checks them).

Cut-passing events (weight != 0; reading R14) are compared with oracle<long double> at the
north-star tolerances 1e-12 (fp64) / 1e-4 (fp32); events that fail the cuts with oracle<double> at
100x those (R14: without the cuts t_S is arbitrarily ill-conditioned, and the double
oracle's own rounding reaches 1e-12 there)."""
import os

import numpy as np
import pytest
import torch

from paper_0908_4403_b200 import ALGO_SUBSET, ALGO_TREE, ALGO_TREE2, FP32, FP64, Heget, workloads

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
TOL = {FP64: 1e-12, FP32: 1e-4}
ALGO_NAME = {ALGO_TREE: "tree", ALGO_SUBSET: "subset", ALGO_TREE2: "two-sided"}


@pytest.fixture(scope="module")
def hg():
    h = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    yield h
    h.close()


@pytest.mark.parametrize("name", ["6gamma", "7gamma", "8gamma"])
@pytest.mark.parametrize("precision", [FP64, FP32])
@pytest.mark.parametrize("algo", [ALGO_TREE, ALGO_SUBSET, ALGO_TREE2])
def test_amp2_matches_the_oracle_on_every_event_of_the_stated_subset(hg, name, precision, algo):
    path = os.path.join(GOLDEN, "amp2_%s.npz" % name)
    if not os.path.exists(path):
        pytest.skip("missing %s: run tests/golden/make_amp2_golden.py --config %s" % (path, name))
    g = np.load(path)
    mom, w, ld = g["momenta"], g["weight"], g["has_ld"]
    got = hg.amp2(torch.from_numpy(mom).cuda(), precision, algo=algo)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    assert np.all(np.isfinite(got)) and np.all(got > 0)
    rel_pass = np.abs(got[ld] / g["amp2_ld"][ld] - 1.0)
    rel_fail = np.abs(got[~ld] / g["amp2_d"][~ld] - 1.0)
    print("\n[golden] %s %s %-9s passing %4d: max %.3e median %.3e  >1e-13: %d   failing %4d: max %.3e median %.3e"
          % (name, "fp64" if precision == FP64 else "fp32", ALGO_NAME[algo], rel_pass.size, rel_pass.max(),
             np.median(rel_pass), int((rel_pass > 1e-13).sum()), rel_fail.size, rel_fail.max(), np.median(rel_fail)))
    assert rel_pass.size >= 100
    assert np.all(rel_pass <= TOL[precision])
    assert np.all(rel_fail <= 100 * TOL[precision])
