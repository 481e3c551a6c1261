"""Pins for the oracle's event generation (oracle/heget_oracle_gen.c): Philox4x32-10
known-answer vectors, RAMBO invariants and phase-space volume, cuts, weights and the
closed-form partonic cross section for n = 2 (pins P9, P10, P11 of DESIGN.md)."""
import math
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def mdot(a, b):
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


def test_P10_philox_known_answer_vectors():
    # tests/golden/philox4x32_10_kat.txt: the three Philox4x32-10 vectors of the Random123
    # known-answer file (Salmon et al., SC'11)
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_uniform_layout_and_range():
    # counter = (event_lo, event_hi, slot, 0), key = (seed_lo, seed_hi); u = (x+0.5)/2^32
    seed, ev, slot = (5 << 32) | 9, (3 << 32) | 77, 4
    x = oracle.philox4x32_10([77, 3, 4, 0], [9, 5])
    u = oracle.uniforms(seed, ev, slot)
    assert np.array_equal(u, (x.astype(np.float64) + 0.5) / 4294967296.0)
    us = np.array([oracle.uniforms(1, e, 1) for e in range(4000)])
    assert us.min() > 0.0 and us.max() < 1.0
    assert abs(us.mean() - 0.5) < 0.01 and abs(us.var() - 1.0 / 12.0) < 0.005


@pytest.mark.parametrize("n", [2, 3, 5, 8])
def test_P9_rambo_invariants(n):
    rs = 1000.0
    mom, w = oracle.gen_events(1, n, 2000, mode=oracle.MODE_FIXED, a=rs)
    k = mom[:, 2:]
    assert np.max(np.abs(k.sum(axis=1) - [rs, 0, 0, 0])) < 1e-10 * rs
    assert np.max(np.abs(mdot(k, k))) < 1e-9 * rs * rs          # massless (boost amplifies eps)
    assert np.median(np.abs(mdot(k, k))) < 1e-13 * rs * rs
    assert np.all(k[..., 0] > 0)
    assert np.array_equal(mom[:, 0], np.tile([rs / 2, 0, 0, rs / 2], (2000, 1)))
    assert np.array_equal(mom[:, 1], np.tile([rs / 2, 0, 0, -rs / 2], (2000, 1)))
    # constant weight Phi_n(s)/(2s)
    vol = (2 * math.pi) ** (4 - 3 * n) * (math.pi / 2) ** (n - 1) * (rs * rs) ** (n - 2) / (
        math.factorial(n - 1) * math.factorial(n - 2))
    assert np.allclose(w, vol / (2 * rs * rs), rtol=1e-13, atol=0)
    # isotropy and democratic energy sharing: <E> = rs/n, <cos theta> = 0
    assert abs(k[..., 0].mean() * n / rs - 1.0) < 1e-12
    cos = k[..., 3] / k[..., 0]
    assert abs(cos.mean()) < 4.0 / math.sqrt(3 * cos.size)
    assert abs((cos ** 2).mean() - 1.0 / 3.0) < 0.03


def test_P9_two_body_volume_is_one_over_eight_pi():
    assert abs(oracle.phase_space_volume(2, 123.0) - 1.0 / (8.0 * math.pi)) < 1e-17
    # Phi_3(s) = s / (256 pi^3)
    assert abs(oracle.phase_space_volume(3, 50.0) / (50.0 / (256.0 * math.pi ** 3)) - 1.0) < 1e-14


def test_events_do_not_depend_on_batching():
    a, wa = oracle.gen_events(3, 4, 100, mode=oracle.MODE_LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5,
                              apply_cuts=True)
    b, wb = oracle.gen_events(3, 4, 40, mode=oracle.MODE_LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5,
                              apply_cuts=True, first_event=60)
    assert np.array_equal(a[60:], b) and np.array_equal(wa[60:], wb)


def test_loguniform_mode_ranges_boost_and_cuts():
    n, N = 4, 20000
    mom, w = oracle.gen_events(1, n, N, mode=oracle.MODE_LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5,
                               apply_cuts=True)
    p1, p2, k = mom[:, 0], mom[:, 1], mom[:, 2:]
    shat = mdot(p1 + p2, p1 + p2)
    rs = np.sqrt(shat)
    assert rs.min() >= 200.0 and rs.max() <= 3000.0
    lg = np.log(rs / 200.0) / math.log(15.0)
    assert abs(lg.mean() - 0.5) < 0.01                       # log-uniform
    y = 0.5 * np.log(p1[:, 0] / p2[:, 0])
    assert np.abs(y).max() <= 1.5 and abs(y.mean()) < 0.03 and abs(y.var() - 0.75) < 0.03
    assert np.max(np.abs(k.sum(axis=1) - (p1 + p2))) < 1e-9 * rs.max()
    # cuts recomputed here with plain numpy (eq. 9)
    pt = np.hypot(k[..., 1], k[..., 2])
    eta = np.arcsinh(k[..., 3] / pt)
    phi = np.arctan2(k[..., 2], k[..., 1])
    ok = np.all(pt > 20.0, axis=1) & np.all(np.abs(eta) < 2.5, axis=1)
    for i in range(n):
        for j in range(i + 1, n):
            dphi = np.abs(phi[:, i] - phi[:, j])
            dphi = np.where(dphi > math.pi, 2 * math.pi - dphi, dphi)
            ok &= np.hypot(eta[:, i] - eta[:, j], dphi) > 0.4
    assert np.array_equal(ok, w != 0.0)
    assert 0.55 < ok.mean() < 0.75                            # SURVEY measured 0.647
    vol = np.array([oracle.phase_space_volume(n, s) for s in shat[:50]])
    assert np.allclose(w[:50][ok[:50]], (vol / (2 * shat[:50]))[ok[:50]], rtol=1e-13)


def test_toypdf_mode_weights():
    n, N, rs_coll = 3, 5000, 14000.0
    mom, w = oracle.gen_events(1, n, N, mode=oracle.MODE_TOYPDF, a=rs_coll, apply_cuts=False)
    p1, p2 = mom[:, 0], mom[:, 1]
    x1, x2 = 2.0 * p1[:, 0] / rs_coll, 2.0 * p2[:, 0] / rs_coll
    tau = x1 * x2
    tau_min = (n * 20.0) ** 2 / rs_coll ** 2
    assert tau.min() >= tau_min * (1 - 1e-12) and tau.max() <= 1.0 and x1.max() <= 1 and x2.max() <= 1
    f = lambda x: x ** -0.5 * (1 - x) ** 3
    shat = tau * rs_coll ** 2
    vol = np.array([oracle.phase_space_volume(n, s) for s in shat])
    expect = vol / (2 * shat) * tau * math.log(1 / tau_min) * np.log(1 / tau) * 2 * f(x1) * f(x2)
    assert np.allclose(w, expect, rtol=1e-11, atol=0)
    # the (tau, y) map has unit total measure: MC integral of 1 over dx1 dx2 above tau_min
    jac = tau * math.log(1 / tau_min) * np.log(1 / tau)
    exact = 1.0 - tau_min + tau_min * math.log(tau_min)      # area of {x1 x2 > tau_min} in the unit square
    assert abs(jac.mean() / exact - 1.0) < 5 * jac.std() / math.sqrt(N) / exact


def test_xsec_reduce_sums():
    rng = np.random.default_rng(0)
    a = rng.uniform(0.5, 2.0, size=1000)
    w = rng.uniform(0.0, 1.0, size=1000)
    w[::3] = 0.0
    out = oracle.xsec_reduce(a, w, 4)
    cf = 0.25 / 9.0 / 24.0
    x = a * w * cf
    assert abs(out[0] / math.fsum(x) - 1.0) < 1e-14
    assert abs(out[1] / math.fsum(x * x) - 1.0) < 1e-14
    assert out[2] == np.count_nonzero(w)


def test_xsec_reduce_ignores_amp2_of_events_that_failed_the_cuts():
    """DESIGN.md R26: weight 0 means the event is outside the cuts of eq. (9); whatever amp2 holds
    there (NaN, Inf from a forward photon or an fp32 range excursion) contributes exactly 0."""
    rng = np.random.default_rng(1)
    a = rng.uniform(0.5, 2.0, size=64)
    w = rng.uniform(0.1, 1.0, size=64)
    w[[3, 17, 40]] = 0.0
    ref = oracle.xsec_reduce(a, w, 3)
    b = a.copy()
    b[3], b[17], b[40] = np.nan, np.inf, -np.inf
    out = oracle.xsec_reduce(b, w, 3)
    assert np.array_equal(out, ref) and out[2] == 61


@pytest.mark.parametrize("n", [3, 4, 5, 6, 7])
def test_P9_phase_space_volume_obeys_the_two_body_recursion(n):
    """Phi_{n+1}(s) = int_0^s dM^2/(2 pi) Phi_n(M^2) Phi_2(s; M, 0): n+1 massless particles = one massless
    particle recoiling against a cluster of n of mass M, with the two-body volume of masses (M, 0),
    Phi_2 = (1/8 pi)(1 - M^2/s).  Integrated numerically on the oracle's own Phi_n -- the closed form
    with its (n-1)!(n-2)! is not restated here."""
    from scipy.integrate import quad
    s = 3.7e5
    integrand = lambda m2: oracle.phase_space_volume(n, m2) * (1.0 - m2 / s) / (8.0 * math.pi) / (2.0 * math.pi)
    val, err = quad(integrand, 0.0, s, epsabs=0.0, epsrel=1e-12)
    assert abs(val / oracle.phase_space_volume(n + 1, s) - 1.0) < 1e-10


def test_P11_two_photon_partonic_cross_section_closed_form():
    """u ubar -> gamma gamma at sqrt(s_hat) = 1 TeV with |eta| < 2.5 only:
    sigma = 1/(2s) * (1/4)(1/9)(1/2!) * (1/16 pi) * 8 e^4 Q^4 * 4 [ln((1+c)/(1-c)) - c], c = tanh(2.5)
    (integral of u/t + t/u over |cos theta| < c).  Monte Carlo through the whole oracle chain:
    gen_events -> amp2 -> xsec_reduce."""
    rs, N = 1000.0, 400000
    c = math.tanh(2.5)
    e4q4 = (4 * math.pi * oracle.ALPHA) ** 2 * oracle.Q_U ** 4
    sigma = (1 / (2 * rs * rs)) * (1 / 36.0) * 0.5 * (1 / (16 * math.pi)) * 8 * e4q4 * 4 * (
        math.log((1 + c) / (1 - c)) - c)
    assert abs(sigma - 3.3780282913638616e-11) < 1e-24       # value quoted in SURVEY/DESIGN (GeV^-2)
    mom, w = oracle.gen_events(1, 2, N, mode=oracle.MODE_FIXED, a=rs, apply_cuts=True,
                               pt_cut=0.0, eta_cut=2.5, dr_cut=0.0)
    s1, s2, cnt = oracle.xsec_reduce(oracle.amp2(mom), w, 2)
    mean = s1 / N
    err = math.sqrt((s2 / N - mean * mean) / N)
    assert abs(cnt / N - c) < 4 * math.sqrt(c * (1 - c) / N)  # acceptance = tanh(eta_cut)
    assert abs(mean - sigma) < 4 * err and err < 3e-3 * sigma
