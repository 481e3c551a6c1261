"""GPU parity of the NEXT-1 entry points (heget_amp2_sampled, heget_histogram) against the CPU
oracle, through the C ABI, on the oracle's own events.

Tolerances.  heget_amp2_sampled returns 4*2^n*|M(h)|^2 for ONE helicity assignment.  Some
assignments are zeros of the amplitude (all photon helicities equal, pin P3) or strongly
suppressed, so a per-entry relative error is undefined there; the error is therefore measured
relative to the event's helicity SUM (the quantity the estimator estimates): 1e-12 in fp64 and
1e-4 in fp32 (north_star), binding on cut-passing events, 10^3 looser on the others (R14).  The
helicity bits are integer work and must be bit-exact.  Histogram bins are sums of at most N
positive fp64 terms in an order that differs from the oracle's: relative 1e-11."""
import numpy as np
import pytest
import torch

import oracle
from paper_0908_4403_b200 import FP32, FP64, OBS_DR_ALL, OBS_DR_MIN, OBS_PT_MAX, Heget, workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hg():
    h = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    yield h
    h.close()


def events(n, N, seed=3):
    lo = {2: 200.0, 3: 200.0, 4: 200.0, 5: 300.0, 6: 400.0, 7: 500.0, 8: 600.0}[n]
    return oracle.gen_events(seed, n, N, mode=oracle.MODE_LOGUNIFORM, a=lo, b=10 * lo, y_max=1.5, apply_cuts=True)


# events per n: several CTAs (8 warps = 8 events per CTA, 4 for n = 8) plus a ragged tail
SIZES = {2: 8 * 40 + 3, 3: 8 * 30 + 5, 4: 8 * 20 + 1, 5: 8 * 12 + 7, 6: 8 * 6 + 3, 7: 8 * 3 + 2, 8: 4 * 3 + 1}


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("precision", [FP64, FP32])
def test_amp2_sampled_matches_oracle(hg, n, precision):
    N = SIZES[n]
    mom, w = events(n, N)
    seed, first = 77, 12345
    ref, ref_bits = oracle.amp2_sampled(seed, mom, first_event=first, extended=(n <= 7))
    # the scale the error is measured against: the helicity sum; for n >= 7 the full sum is too
    # slow for the oracle on every event, so the median non-zero estimator stands in for it
    if n <= 6:
        scale = oracle.amp2(mom)
    else:
        scale = np.maximum(ref, np.median(ref[ref > 0]))
    got, bits = hg.amp2_sampled(seed, torch.from_numpy(mom).cuda(), precision, first_event=first)
    torch.cuda.synchronize()
    got, bits = got.cpu().numpy(), bits.cpu().numpy()
    assert np.array_equal(bits, ref_bits)
    quark_equal = ((bits & 1) == ((bits >> 1) & 1))
    assert np.all(got[quark_equal] == 0.0) and np.all(ref[quark_equal] == 0.0)
    err = np.abs(got - ref) / scale
    tol = 1e-12 if precision == FP64 else 1e-4
    passing = w != 0
    print("\n[sampled parity] n=%d %s events=%d non-zero=%d: passing max %.3e, all max %.3e"
          % (n, "fp64" if precision == FP64 else "fp32", N, int((~quark_equal).sum()),
             err[passing].max(), err.max()))
    assert (~quark_equal).sum() >= 2
    assert np.all(err[passing] <= tol) and np.all(err <= tol * 1e3)
    # where the estimator is not suppressed the plain relative error obeys the same bound
    big = passing & (ref > 1e-2 * scale)
    assert np.all(np.abs(got[big] / ref[big] - 1.0) <= tol * 1e2)


def test_amp2_sampled_is_an_unbiased_estimator_of_heget_amp2(hg):
    n, N = 5, 1 << 15
    mom, _ = events(n, 1)
    rep = torch.from_numpy(np.repeat(mom, N, axis=0)).cuda()
    val, _ = hg.amp2_sampled(5, rep, FP64)
    total = hg.amp2(rep[:1].contiguous(), FP64).item()
    v = val.cpu().numpy()
    assert abs(v.mean() - total) < 5 * v.std() / np.sqrt(N)
    assert abs(total / oracle.amp2(mom, extended=True)[0] - 1.0) < 1e-12


def test_amp2_sampled_shards_and_edges(hg):
    n = 4
    mom, _ = events(n, 300)
    d = torch.from_numpy(mom).cuda()
    whole, hb = hg.amp2_sampled(9, d, FP64, first_event=50)
    a, ha = hg.amp2_sampled(9, d[:113].contiguous(), FP64, first_event=50)
    b, hb2 = hg.amp2_sampled(9, d[113:].contiguous(), FP64, first_event=50 + 113)
    assert torch.equal(torch.cat([a, b]), whole) and torch.equal(torch.cat([ha, hb2]), hb)
    empty = torch.empty((0, n + 2, 4), dtype=torch.float64, device="cuda")
    v, h = hg.amp2_sampled(9, empty)
    assert v.shape == (0,) and h.shape == (0,)
    lib, ctx = hg._lib, hg._ctx
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    assert lib.heget_amp2_sampled(ctx, 1, 0, d.data_ptr(), 9, FP64, out.data_ptr(), None, 4, None) == -1
    assert lib.heget_amp2_sampled(ctx, 1, 0, d.data_ptr(), 4, 5, out.data_ptr(), None, 4, None) == -1
    assert lib.heget_amp2_sampled(ctx, 1, 0, d.data_ptr(), 4, FP64, out.data_ptr(), None, 4, None) == 0   # hel optional


def observables(mom):
    """numpy evaluation used ONLY to drop events whose observable sits on a bin edge, where the
    device's asinh / atan2 and libm's may round to different sides."""
    k = mom[:, 2:, :]
    pt = np.hypot(k[..., 1], k[..., 2])
    eta = np.arcsinh(k[..., 3] / pt)
    phi = np.arctan2(k[..., 2], k[..., 1])
    ii, jj = np.triu_indices(k.shape[1], 1)
    dphi = np.abs(phi[:, ii] - phi[:, jj])
    dphi = np.where(dphi > np.pi, 2 * np.pi - dphi, dphi)
    dr = np.sqrt((eta[:, ii] - eta[:, jj]) ** 2 + dphi ** 2)
    return pt.max(axis=1), dr


@pytest.mark.parametrize("n,N", [(2, 5000), (5, 20011), (8, 3000)])
def test_histograms_match_oracle(hg, n, N):
    mom, w = events(n, N, seed=8)
    rng = np.random.default_rng(1)
    val = w * rng.uniform(0.5, 2.0, size=N) * 1e9           # zero for events that fail the cuts
    ptmax, dr = observables(mom)
    cases = [(OBS_PT_MAX, ptmax[:, None], 0.0, 1500.0, 60), (OBS_PT_MAX, ptmax[:, None], 100.0, 300.0, 7),
             (OBS_DR_MIN, dr.min(axis=1)[:, None], 0.0, 4.0, 40), (OBS_DR_ALL, dr, 0.0, 6.0, 48),
             (OBS_DR_ALL, dr, 0.4, 3.0, 4094)]
    dm = torch.from_numpy(mom).cuda()
    for obs, x, lo, hi, nb in cases:
        edges = lo + (hi - lo) * np.arange(nb + 1) / nb
        near = (np.abs(x[:, :, None] - edges[None, None, :]).min(axis=2) < 1e-9).any(axis=1)
        v = np.where(near, 0.0, val)
        want = oracle.histogram(mom, v, obs, lo, hi, nb)
        got = hg.histogram(dm, torch.from_numpy(v).cuda(), obs, lo, hi, nb).cpu().numpy()
        assert got.shape == (nb + 2,)
        assert np.array_equal(got != 0, want != 0)
        assert np.allclose(got, want, rtol=1e-11, atol=0.0)
        assert want.sum() > 0


def test_histogram_edges_and_errors(hg):
    mom, w = events(3, 100, seed=2)
    dm = torch.from_numpy(mom).cuda()
    zero = torch.zeros(100, dtype=torch.float64, device="cuda")
    h = hg.histogram(dm, zero, OBS_PT_MAX, 0.0, 100.0, 10)
    assert torch.count_nonzero(h).item() == 0                 # zero-valued events are skipped
    empty = torch.empty((0, 5, 4), dtype=torch.float64, device="cuda")
    h = hg.histogram(empty, zero[:0], OBS_DR_MIN, 0.0, 1.0, 3)
    assert h.shape == (5,) and torch.count_nonzero(h).item() == 0
    lib, ctx = hg._lib, hg._ctx
    out = torch.zeros(4100, dtype=torch.float64, device="cuda")
    args = (dm.data_ptr(), zero.data_ptr(), 3, 100)
    assert lib.heget_histogram(ctx, *args, 3, 0.0, 1.0, 10, out.data_ptr(), None) == -1     # bad observable
    assert lib.heget_histogram(ctx, *args, 0, 1.0, 1.0, 10, out.data_ptr(), None) == -1     # hi <= lo
    assert lib.heget_histogram(ctx, *args, 0, 0.0, 1.0, 0, out.data_ptr(), None) == -1      # no bins
    assert lib.heget_histogram(ctx, *args, 0, 0.0, 1.0, 4095, out.data_ptr(), None) == -1   # too many bins
    assert lib.heget_histogram(ctx, *args, 0, 0.0, 1.0, 10, None, None) == -1
    assert lib.heget_histogram(ctx, *args, 0, 0.0, 1.0, 4094, out.data_ptr(), None) == 0


def test_device_philox_matches_the_kat_pinned_oracle_bits(hg):
    # the helicity bits are the device Philox's first output word: bit-exact against the oracle's
    # (KAT-pinned) implementation for large event indices and 64-bit seeds
    n = 8
    mom, _ = events(n, 64)
    d = torch.from_numpy(mom).cuda()
    for seed, first in [(1, 0), (2 ** 40 + 3, 2 ** 33 + 17), (2 ** 63 + 5, 2 ** 62)]:
        _, bits = hg.amp2_sampled(seed, d, FP32, first_event=first)
        want = np.array([oracle.helicity_bits(seed, first + e, n) for e in range(64)], dtype=np.int32)
        assert np.array_equal(bits.cpu().numpy(), want)


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("precision", [FP64, FP32])
def test_paper_list2_program_matches_oracle_and_the_sampled_kernel(hg, n, precision):
    """heget_list2 is the paper's List 2 run as the paper runs it: it must give
    the oracle's estimator for the same drawn helicities, and so must agree with heget_amp2_sampled.

    Tolerance.  The paper's program evaluates every propagator denominator pf^2 in plain working
    precision inside fvoxx0 (no table, no compensated arithmetic), and pf^2 = (p2 - K)^2 cancels for
    forward photons: SURVEY 7 (hard part 2) measured 3e-13 .. 3e-11 in fp64 and up to 2e-4 in fp32
    for exactly this evaluation.  The bars here are therefore 1e-10 (fp64) and 2e-3 (fp32) on
    cut-passing events -- a property of the paper's design that the library's own kernels
    (1e-12 / 1e-4) do not share."""
    N = {2: 600, 3: 500, 4: 400, 5: 300, 6: 200, 7: 64, 8: 13}[n]
    mom, w = events(n, N)
    seed, first = 31, 999
    ref, ref_bits = oracle.amp2_sampled(seed, mom, first_event=first, extended=(n <= 7))
    scale = oracle.amp2(mom) if n <= 5 else np.maximum(ref, np.median(ref[ref > 0]))
    d = torch.from_numpy(mom).cuda()
    got, bits = hg.list2(seed, d, precision, first_event=first)
    ours, _ = hg.amp2_sampled(seed, d, precision, first_event=first)
    got, bits, ours = got.cpu().numpy(), bits.cpu().numpy(), ours.cpu().numpy()
    assert np.array_equal(bits, ref_bits)
    tol = 1e-10 if precision == FP64 else 2e-3
    passing = w != 0
    err = np.abs(got - ref) / scale
    print("\n[list2 parity] n=%d %s events=%d: passing max %.3e median %.3e, all max %.3e"
          % (n, "fp64" if precision == FP64 else "fp32", N, err[passing].max(), np.median(err[passing]), err.max()))
    assert np.all(err[passing] <= tol) and np.all(err <= tol * 1e3)
    assert np.all(np.abs(got - ours)[passing] <= 2 * tol * scale[passing])


@pytest.mark.parametrize("n", [2, 3, 4, 5])
@pytest.mark.parametrize("precision", [FP64, FP32])
def test_paper_list2_summed_over_helicities_matches_oracle_and_heget_amp2(hg, n, precision):
    """heget_list2_sum: the paper's program called for all 4*2^n helicity assignments (the paper's
    arithmetic for the north-star quantity).  Same accuracy class as heget_list2 (plain p_f^2)."""
    N = {2: 700, 3: 400, 4: 300, 5: 100}[n]
    mom, w = events(n, N)
    ref = oracle.amp2(mom, extended=True)
    d = torch.from_numpy(mom).cuda()
    got = hg.list2_sum(d, precision).cpu().numpy()
    ours = hg.amp2(d, precision).cpu().numpy()
    tol = 1e-10 if precision == FP64 else 2e-3
    passing = w != 0
    err = np.abs(got / ref - 1.0)
    print("\n[list2 sum parity] n=%d %s events=%d: passing max %.3e median %.3e, all max %.3e"
          % (n, "fp64" if precision == FP64 else "fp32", N, err[passing].max(), np.median(err[passing]), err.max()))
    assert np.all(err[passing] <= tol) and np.all(err <= tol * 1e3)
    assert np.all(np.abs(got / ours - 1.0)[passing] <= 2 * tol)
