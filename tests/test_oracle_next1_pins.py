"""Pins of the oracle's NEXT-1 functions (helicity sampling, Fig. 2 histograms) against what
the paper and the mathematics fix -- no GPU, no CUDA code involved.

  * the sampled estimator 4*2^n*|M(h)|^2 averaged over ALL assignments h is the helicity sum of
    eq. (2), and averaged over Philox draws converges to it;
  * helicity-conservation zeros (sigma_1 = sigma_2) are exact zeros of the estimator;
  * the helicity bits are the documented bits of the KAT-pinned Philox word (R21);
  * pT and Delta R (eqs. 9, 10) of photons BUILT from chosen (pT, eta, phi)
    must come back as those parameters, bin by bin (the oracle goes through asinh / atan2, the
    construction through sinh / cos / sin);
  * histogram bookkeeping: conservation of the summed weight, under/overflow, edges.
"""
import itertools

import numpy as np

import oracle


def photons_from(pt, eta, phi):
    """[n][4] four-momenta (E,px,py,pz) of massless photons with the given pT, eta, phi."""
    pt, eta, phi = map(np.asarray, (pt, eta, phi))
    return np.stack([pt * np.cosh(eta), pt * np.cos(phi), pt * np.sin(phi), pt * np.sinh(eta)], axis=-1)


def event_from(pt, eta, phi):
    k = photons_from(pt, eta, phi)
    tot = k.sum(axis=0)
    # incoming partons along z that balance E and pz (transverse balance is irrelevant here)
    e1, e2 = 0.5 * (tot[0] + tot[3]), 0.5 * (tot[0] - tot[3])
    return np.concatenate([[[e1, 0, 0, e1], [e2, 0, 0, -e2]], k])


def test_helicity_bits_are_the_low_bits_of_the_philox_word():
    for seed, event, n in [(1, 0, 2), (1, 5, 4), (7, 123456789012, 8), (2 ** 40 + 3, 17, 6)]:
        word = oracle.philox4x32_10([event & 0xFFFFFFFF, event >> 32, 15, 0], [seed & 0xFFFFFFFF, seed >> 32])[0]
        assert oracle.helicity_bits(seed, event, n) == int(word) & ((1 << (n + 2)) - 1)


def test_helicity_bits_are_unbiased_and_independent_of_the_generator_slots():
    n, N = 6, 40000
    bits = np.array([oracle.helicity_bits(3, e, n) for e in range(N)])
    for b in range(n + 2):
        frac = ((bits >> b) & 1).mean()
        assert abs(frac - 0.5) < 5 * 0.5 / np.sqrt(N)
    counts = np.bincount(bits, minlength=1 << (n + 2))
    chi2 = ((counts - N / 256.0) ** 2 / (N / 256.0)).sum()
    assert chi2 < 255 + 6 * np.sqrt(2 * 255)
    # slot 15 is not one of the generator's slots 0..n: the momenta do not move
    assert not np.array_equal(oracle.uniforms(3, 0, 15), oracle.uniforms(3, 0, 0))


def test_exhaustive_average_of_the_estimator_is_the_helicity_sum():
    for n in (2, 3, 4):
        mom, _ = oracle.gen_events(11, n, 1, mode=oracle.MODE_LOGUNIFORM, a=300.0, b=2000.0, y_max=1.0)
        total = oracle.amp2(mom)[0]
        acc = 0.0
        for h in itertools.product([-1, 1], repeat=n + 2):
            acc += 4 * 2 ** n * abs(oracle.amp(mom[0], list(h))) ** 2
        assert abs(acc / (4 * 2 ** n) / total - 1.0) < 1e-13


def test_sampled_value_is_the_estimator_of_the_drawn_assignment_and_zero_for_equal_quark_helicities():
    n, N = 4, 200
    mom, _ = oracle.gen_events(5, n, N, mode=oracle.MODE_LOGUNIFORM, a=300.0, b=2000.0, y_max=1.0)
    val, bits = oracle.amp2_sampled(9, mom, first_event=1000)
    n_zero = 0
    for e in range(N):
        assert bits[e] == oracle.helicity_bits(9, 1000 + e, n)
        h = [1 if (bits[e] >> b) & 1 else -1 for b in range(n + 2)]
        want = 4 * 2 ** n * abs(oracle.amp(mom[e], h)) ** 2
        if h[0] == h[1]:
            assert val[e] == 0.0          # helicity conservation on a massless line: exact zero
            n_zero += 1
        else:
            assert abs(val[e] / want - 1.0) < 1e-14
    assert 60 < n_zero < 140
    vx, bx = oracle.amp2_sampled(9, mom, first_event=1000, extended=True)
    assert np.array_equal(bx, bits)
    # all-equal photon helicities are zeros of the amplitude too (pin P3): there both results are
    # rounding noise, so the comparison is relative to the event's helicity sum
    assert np.all(np.abs(vx - val) < 1e-10 * oracle.amp2(mom))


def test_monte_carlo_over_helicities_converges_to_the_helicity_sum():
    n, N = 3, 20000
    mom, _ = oracle.gen_events(2, n, 1, mode=oracle.MODE_FIXED, a=500.0)
    rep = np.repeat(mom, N, axis=0)
    val, _ = oracle.amp2_sampled(4, rep)
    total = oracle.amp2(mom)[0]
    err = val.std() / np.sqrt(N)
    assert abs(val.mean() - total) < 5 * err
    assert err < 0.05 * total


def test_histogram_recovers_the_generating_pt_eta_phi():
    rng = np.random.default_rng(0)
    n, N = 5, 400
    pt = rng.uniform(20.0, 400.0, size=(N, n))
    eta = rng.uniform(-2.5, 2.5, size=(N, n))
    phi = rng.uniform(-np.pi, np.pi, size=(N, n))
    mom = np.stack([event_from(pt[e], eta[e], phi[e]) for e in range(N)])
    val = rng.uniform(0.5, 2.0, size=N)
    # expected observables from the generating parameters, not from the momenta
    ptmax = pt.max(axis=1)
    ii, jj = np.triu_indices(n, 1)
    dphi = np.abs(phi[:, ii] - phi[:, jj])
    dphi = np.where(dphi > np.pi, 2 * np.pi - dphi, dphi)
    dr = np.sqrt((eta[:, ii] - eta[:, jj]) ** 2 + dphi ** 2)
    for obs, x, wts, lo, hi, nb in [
            (oracle.OBS_PT_MAX, ptmax, val, 0.0, 400.0, 40),
            (oracle.OBS_PT_MAX, ptmax, val, 100.0, 300.0, 7),       # under- and overflow populated
            (oracle.OBS_DR_MIN, dr.min(axis=1), val, 0.0, 3.0, 30),
            (oracle.OBS_DR_ALL, dr.ravel(), np.repeat(val, len(ii)), 0.0, 6.0, 24)]:
        got = oracle.histogram(mom, val, obs, lo, hi, nb)
        want = np.zeros(nb + 2)
        want[1:-1] = np.histogram(x, bins=nb, range=(lo, hi), weights=wts)[0]
        # np.histogram puts x == hi into the last bin; the oracle's bins are [lo, hi)
        want[0] = wts[x < lo].sum()
        want[-1] = wts[x >= hi].sum()
        # values within 1e-9 of an edge may land on either side (asinh(sinh(eta)) rounding)
        edges = lo + (hi - lo) * np.arange(nb + 1) / nb
        near = np.min(np.abs(x[:, None] - edges[None, :]), axis=1) < 1e-9
        assert not near.any()
        assert np.allclose(got, want, rtol=1e-12, atol=1e-12)
        assert abs(got.sum() - wts.sum()) < 1e-9 * wts.sum()


def test_histogram_edges_and_zero_weight_events():
    # one photon pair, pT_max exactly on edges
    ev = event_from([50.0, 30.0], [0.0, 1.0], [0.0, 2.0])
    mom = np.stack([ev, ev, ev])
    val = np.array([1.0, 0.0, 2.5])
    h = oracle.histogram(mom, val, oracle.OBS_PT_MAX, 0.0, 100.0, 4)       # 50 is the edge of bin 2
    assert np.array_equal(h, [0, 0, 0, 3.5, 0, 0])
    h = oracle.histogram(mom, val, oracle.OBS_PT_MAX, 0.0, 50.0, 5)        # x == hi -> overflow
    assert np.array_equal(h, [0, 0, 0, 0, 0, 0, 3.5])
    h = oracle.histogram(mom, val, oracle.OBS_PT_MAX, 50.0, 60.0, 2)       # x == lo -> first bin
    assert np.array_equal(h, [0, 3.5, 0, 0])
    # Delta phi wraps: phi = 3.0 and -3.0 are 2*pi - 6 apart
    ev2 = event_from([40.0, 40.0], [0.5, 0.5], [3.0, -3.0])
    want = 2 * np.pi - 6.0
    h = oracle.histogram(ev2[None], np.ones(1), oracle.OBS_DR_MIN, 0.0, 1.0, 100)
    assert h[1 + int(want * 100)] == 1.0 and h.sum() == 1.0
