"""The stored oracle values of tests/golden/amp2_<config>.npz (written by tests/golden/make_amp2_golden.py,
which calls only oracle/) are what they claim to be: the momenta are the first events of the config from
the oracle's generator, bit for bit, and the stored values are the oracle's on those momenta.  No GPU."""
import hashlib
import os

import numpy as np
import pytest

import oracle
from paper_0908_4403_b200 import workloads

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
# the subsets BASELINE.json `configs` state for 7 and 8 gamma; 2,048 events at 6 gamma
SUBSET = {"6gamma": 2048, "7gamma": 4096, "8gamma": 512}


def load(name):
    path = os.path.join(GOLDEN, "amp2_%s.npz" % name)
    if not os.path.exists(path):
        pytest.skip("missing %s: run tests/golden/make_amp2_golden.py --config %s" % (path, name))
    return np.load(path)


@pytest.mark.parametrize("name", sorted(SUBSET))
def test_golden_momenta_are_the_configs_first_events(name):
    g = load(name)
    c = workloads.CONFIGS[name]
    N = SUBSET[name]
    assert g["momenta"].shape == (N, c["n"] + 2, 4) and g["amp2_d"].shape == (N,)
    mom, w = oracle.gen_events(c["seed"], c["n"], N, mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                               apply_cuts=c["apply_cuts"], pt_cut=workloads.PT_CUT, eta_cut=workloads.ETA_CUT,
                               dr_cut=workloads.DR_CUT)
    assert np.array_equal(mom, g["momenta"]) and np.array_equal(w, g["weight"])
    assert hashlib.sha256(mom.tobytes()).hexdigest() == str(g["momenta_sha256"])
    # long double values exactly on the cut-passing events (where the 1e-12 gate binds, R14)
    assert np.array_equal(g["has_ld"], w != 0)
    assert np.all(np.isfinite(g["amp2_ld"][g["has_ld"]])) and np.all(np.isnan(g["amp2_ld"][~g["has_ld"]]))
    assert np.all(g["amp2_d"] > 0)


@pytest.mark.parametrize("name,count", [("6gamma", 6), ("7gamma", 1)])
def test_golden_values_are_the_oracles(name, count):
    """Spot check (the full sets are tens of core-hours): recompute a few stored values."""
    g = load(name)
    idx = np.flatnonzero(g["has_ld"])[:count]
    assert np.array_equal(oracle.amp2(g["momenta"][idx]), g["amp2_d"][idx])
    if name == "6gamma":
        assert np.array_equal(oracle.amp2(g["momenta"][idx[:2]], extended=True), g["amp2_ld"][idx[:2]])


@pytest.mark.parametrize("name", sorted(SUBSET))
def test_precision_ladder_on_the_golden_sets(name):
    """Pin P8 at the stated sizes: oracle<double> against oracle<long double> bounds the oracle's own
    rounding on every cut-passing event; it is why the GPU comparison uses the long double values."""
    g = load(name)
    ld = g["has_ld"]
    ladder = np.abs(g["amp2_d"][ld] / g["amp2_ld"][ld] - 1.0)
    print("\n[ladder] %s: %d cut-passing events, oracle<double> vs <long double>: max %.3e median %.3e"
          % (name, int(ld.sum()), ladder.max(), np.median(ladder)))
    assert ladder.max() < 5e-12 and np.median(ladder) < 1e-13
