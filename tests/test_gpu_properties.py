"""Properties of the summed squared amplitude that hold at any size, checked on the CUDA path
itself (all three organisations of the permutation sum, both precisions) at BASELINE.json's
event counts for 4 and 6 photons -- no oracle involved, so every event of the launch is covered:

  * Bose symmetry: relabelling the photons leaves sum |M|^2 unchanged (pin P5 on the oracle);
  * scaling: sum |M|^2 (lambda p) = lambda^(2(2-n)) sum |M|^2 (p)           (pin P6);
  * rotation about the beam axis and the reflection y -> -y leave it unchanged (pin P6).

The transformed inputs are different floating-point numbers, so the comparison is to rounding:
1e-11 in fp64 on cut-passing events (the transformation itself perturbs the inputs by an ulp, which
the conditioning of the forward region amplifies), 1e-4 in fp32 (north_star's bar)."""
import numpy as np
import pytest
import torch

from paper_0908_4403_b200 import ALGO_SUBSET, ALGO_TREE, ALGO_TREE2, FP32, FP64, Heget, workloads

pytestmark = pytest.mark.gpu

TOL = {FP64: 1e-11, FP32: 1e-4}
SIZES = {"4gamma": 1 << 20, "6gamma": 1 << 17}


@pytest.fixture(scope="module")
def hg():
    h = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    yield h
    h.close()


def device_events(hg, name):
    c = workloads.CONFIGS[name]
    return hg.gen_events(c["seed"], c["n"], SIZES[name], mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                         apply_cuts=c["apply_cuts"])


def worst(a, b, passing):
    return (torch.abs(a / b - 1.0)[passing]).max().item()


@pytest.mark.parametrize("name", ["4gamma", "6gamma"])
@pytest.mark.parametrize("precision", [FP64, FP32])
@pytest.mark.parametrize("algo", [ALGO_TREE, ALGO_SUBSET, ALGO_TREE2])
def test_symmetries_of_the_summed_amplitude(hg, name, precision, algo):
    mom, w = device_events(hg, name)
    n = mom.shape[1] - 2
    passing = w != 0
    base = hg.amp2(mom, precision, algo=algo)
    assert torch.all(torch.isfinite(base)) and torch.all(base > 0)
    tol = TOL[precision]

    # Bose symmetry: reverse the photon order and swap two photons
    perm = list(range(n))[::-1]
    perm[0], perm[1] = perm[1], perm[0]
    idx = torch.tensor([0, 1] + [2 + p for p in perm], device=mom.device)
    relabelled = mom.index_select(1, idx).contiguous()
    assert worst(hg.amp2(relabelled, precision, algo=algo), base, passing) <= tol

    # scaling by an exact power of two (the momenta scale exactly; fp32 works in units of sqrt(s_hat))
    lam = 4.0
    scaled = hg.amp2((mom * lam).contiguous(), precision, algo=algo) * lam ** (2 * (n - 2))
    assert worst(scaled, base, passing) <= tol

    # rotation about z by 0.7 rad and reflection y -> -y
    c, s = np.cos(0.7), np.sin(0.7)
    rot = mom.clone()
    rot[:, :, 1] = c * mom[:, :, 1] - s * mom[:, :, 2]
    rot[:, :, 2] = s * mom[:, :, 1] + c * mom[:, :, 2]
    assert worst(hg.amp2(rot, precision, algo=algo), base, passing) <= tol
    ref = mom.clone()
    ref[:, :, 2] = -mom[:, :, 2]
    assert worst(hg.amp2(ref, precision, algo=algo), base, passing) <= tol


def test_algorithms_agree_on_every_event_of_the_headline_launch(hg):
    mom, w = device_events(hg, "4gamma")
    passing = w != 0
    t = hg.amp2(mom, FP64, algo=ALGO_TREE)
    # the thread-per-event kernel (plain light-cone components, t_S from double-double invariants) against
    # the kernels that build the double-double subset table: two independent evaluations of eq. (8)
    for algo in (ALGO_SUBSET, ALGO_TREE2):
        d = torch.abs(hg.amp2(mom, FP64, algo=algo) / t - 1.0)[passing]
        print("\n[cross-check] 4gamma fp64, %d cut-passing events of 2^20: tree vs algo %d: max %.3e, > 1e-13: %d"
              % (int(passing.sum()), algo, d.max().item(), int((d > 1e-13).sum())))
        assert worst(hg.amp2(mom, FP64, algo=algo), t, passing) <= 2e-12
        assert worst(hg.amp2(mom, FP32, algo=algo), t, passing) <= 1e-4
    assert worst(hg.amp2(mom, FP32, algo=ALGO_TREE), t, passing) <= 1e-4


@pytest.mark.parametrize("n,N", [(2, (1 << 18) + 37), (3, (1 << 19) + 37), (4, (1 << 18) + 61), (5, (1 << 18) + 5),
                                 (6, (1 << 16) + 13), (7, (1 << 13) + 1)])
def test_three_organisations_of_the_sum_agree_on_large_ragged_batches(hg, n, N):
    """The one-sided tree (thread per event for n <= 4, lane per helicity assignment above), two-sided chaining
    and the subset recursion are three different evaluation orders of the same n! diagrams: on every event of
    a large batch whose size is not a multiple of the events per CTA they must agree to rounding."""
    for seed in (2, 3):
        mom, w = hg.gen_events(seed, n, N, mode=workloads.LOGUNIFORM, a=100.0 * n, b=1500.0 * n, y_max=1.5,
                               apply_cuts=True)
        ok = w != 0
        ref = hg.amp2(mom, FP64, algo=ALGO_SUBSET)
        for algo in (ALGO_TREE, ALGO_TREE2):
            for precision, tol in ((FP64, 2e-12), (FP32, 1e-4)):
                got = hg.amp2(mom, precision, algo=algo)
                assert torch.all(torch.isfinite(got)) and got.shape == (N,)
                assert worst(got, ref, ok) <= tol
