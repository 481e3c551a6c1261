"""Pins of the oracle's HEGET function set (oracle/heget_oracle_helas.c) --
no GPU, no CUDA code involved.

  * Lists 9/10 of the paper (golden fixture) fix vxxxx1 / vxxxx2 including the
    momentum slots; the "1"/"2" forms are the beam-axis limits of the generic "0" forms;
  * Dirac equation, chirality and the normalisation ubar gamma^mu u = 2 p^mu fix the spinors
    and the relative phase of <fo| and |fi>;
  * fvoxx0 (List 2's chain from the ubar end) and fvixx0 (eq. 7's chain from the
    u end) must give the same diagram, and the two orderings must add up to the two-photon
    amplitude whose square is pinned by the closed form P1;
  * jioxx0: current conservation, and q qbar -> q' qbar' through the off-shell photon has the
    textbook sum over helicities 8 g^2 g'^2 (t^2 + u^2) / s^2.
"""
import itertools
import os

import numpy as np

import oracle
from oracle import (FN_IXXXX0, FN_IXXXX1, FN_IXXXX2, FN_OXXXX0, FN_OXXXX1, FN_OXXXX2, FN_VXXXX0, FN_VXXXX1,
                    FN_VXXXX2, VTX_FVIXX0, VTX_FVOXX0, VTX_IOVXXX, VTX_JIOXX0)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
METRIC = np.array([1.0, -1.0, -1.0, -1.0])


def massless(rng, e_lo=20.0, e_hi=500.0):
    e = rng.uniform(e_lo, e_hi)
    c = rng.uniform(-0.95, 0.95)
    phi = rng.uniform(-np.pi, np.pi)
    s = np.sqrt(1 - c * c)
    return np.array([e, e * s * np.cos(phi), e * s * np.sin(phi), e * c])


def slash(a):
    return sum(METRIC[mu] * a[mu] * oracle.gamma(mu) for mu in range(4))


def test_lists_9_and_10_and_momentum_slots():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "vxxxx_lists_9_10.txt")) if l.strip() and l[0] != "#"]
    r2 = 1 / np.sqrt(2.0)
    for direction, nhel, re1, im2 in rows:
        fn = FN_VXXXX1 if direction == "+z" else FN_VXXXX2
        e = 123.0
        w = oracle.helas_wavefunction(fn, [e, 0, 0, 0], int(nhel), -1)
        assert w[0] == 0 and w[3] == 0
        assert abs(w[1] - float(re1) * r2) < 1e-15 and abs(w[2] - 1j * float(im2) * r2) < 1e-15
        pz = e if direction == "+z" else -e
        assert w[4] == complex(-e, -pz) and w[5] == 0          # vc[4] = (-p0,-p3), vc[5] = (-p1,-p2)


def test_special_direction_forms_are_limits_of_the_generic_forms():
    e, eps = 250.0, 1e-7
    for sign, i_fn, o_fn, v_fn in ((+1, FN_IXXXX1, FN_OXXXX1, FN_VXXXX1), (-1, FN_IXXXX2, FN_OXXXX2, FN_VXXXX2)):
        axis = np.array([e, 0.0, 0.0, sign * e])
        # +z: approached at azimuth 0; -z: Lists 9/10 fix the azimuth-pi approach for the vector
        near = np.array([e, sign * e * eps, 0.0, sign * e * np.sqrt(1 - eps * eps)])
        for nhel, ns in itertools.product((-1, 1), (-1, 1)):
            for special, generic in ((i_fn, FN_IXXXX0), (o_fn, FN_OXXXX0), (v_fn, FN_VXXXX0)):
                a = oracle.helas_wavefunction(special, [e, 9.0, 9.0, 9.0], nhel, ns)    # only |p| is used
                b = oracle.helas_wavefunction(generic, axis, nhel, ns)
                assert np.array_equal(a, b)
                if generic == FN_VXXXX0 or sign == +1:
                    # continuous limit (the -z spinors sit on the branch point of the HELAS
                    # phase convention: their limit depends on the azimuth and is not taken)
                    c = oracle.helas_wavefunction(generic, near, nhel, ns)
                    assert np.allclose(a[:4], c[:4], atol=2e-5 * np.sqrt(e))


def test_spinors_dirac_equation_chirality_and_current_normalisation():
    rng = np.random.default_rng(5)
    g5 = 1j * oracle.gamma(0) @ oracle.gamma(1) @ oracle.gamma(2) @ oracle.gamma(3)
    for _ in range(20):
        p = massless(rng)
        ps = slash(p)
        for nhel in (-1, 1):
            for ns in (-1, 1):
                fi = oracle.helas_wavefunction(FN_IXXXX0, p, nhel, ns)
                fo = oracle.helas_wavefunction(FN_OXXXX0, p, nhel, ns)
                assert np.abs(ps @ fi[:4]).max() < 1e-11 * p[0] ** 1.5
                assert np.abs(fo[:4] @ ps).max() < 1e-11 * p[0] ** 1.5
                assert np.allclose(g5 @ fi[:4], nhel * ns * fi[:4], atol=1e-12 * np.sqrt(p[0]))
                cur = np.array([fo[:4] @ oracle.gamma(mu) @ fi[:4] for mu in range(4)])
                assert np.allclose(cur, 2 * p, atol=1e-10 * p[0])
                assert fi[4] == ns * complex(p[0], p[3]) and fi[5] == ns * complex(p[1], p[2])
                assert np.array_equal(fo[4:], fi[4:])


def two_photon_event(seed):
    mom, _ = oracle.gen_events(seed, 2, 1, mode=oracle.MODE_LOGUNIFORM, a=300.0, b=2000.0, y_max=1.0)
    return mom[0]


def test_fvoxx0_chain_equals_fvixx0_chain_and_sums_to_the_two_photon_amplitude():
    g = oracle.G_DEFAULT
    for seed in range(1, 6):
        p1, p2, k1, k2 = two_photon_event(seed)
        for h in itertools.product((-1, 1), repeat=4):
            fi = oracle.helas_wavefunction(FN_IXXXX1, p1, h[0], +1)
            fo = oracle.helas_wavefunction(FN_OXXXX2, p2, h[1], -1)
            v1 = oracle.helas_wavefunction(FN_VXXXX0, k1, h[2], +1)
            v2 = oracle.helas_wavefunction(FN_VXXXX0, k2, h[3], +1)
            total = 0.0
            for va, vb in ((v1, v2), (v2, v1)):          # photon va attached next to u, vb next to ubar
                from_u = oracle.helas_vertex(VTX_IOVXXX, fi=oracle.helas_vertex(VTX_FVIXX0, fi=fi, vc=va, g=g),
                                             fo=fo, vc=vb, g=g)
                from_ubar = oracle.helas_vertex(VTX_IOVXXX, fi=fi,
                                                fo=oracle.helas_vertex(VTX_FVOXX0, fo=fo, vc=vb, g=g), vc=va, g=g)
                scale = abs(from_u) + 1e-30
                assert abs(from_u - from_ubar) < 1e-10 * scale + 1e-14   # helicity zeros are rounding noise
                total += from_ubar
            want = oracle.amp(np.array([p1, p2, k1, k2]), list(h), g)
            assert abs(total - want) < 1e-10 * abs(want) + 1e-14
    # and the squared sum is the closed form P1 (checked here once more through the w[6] route)
    p1, p2, k1, k2 = two_photon_event(9)
    acc = 0.0
    for h in itertools.product((-1, 1), repeat=4):
        fi = oracle.helas_wavefunction(FN_IXXXX1, p1, h[0], +1)
        fo = oracle.helas_wavefunction(FN_OXXXX2, p2, h[1], -1)
        v = [oracle.helas_wavefunction(FN_VXXXX0, k, hh, +1) for k, hh in ((k1, h[2]), (k2, h[3]))]
        m = sum(oracle.helas_vertex(VTX_IOVXXX, fi=fi, fo=oracle.helas_vertex(VTX_FVOXX0, fo=fo, vc=v[b], g=g),
                                    vc=v[a], g=g) for a, b in ((0, 1), (1, 0)))
        acc += abs(m) ** 2

    def dot(a, b):
        return a[0] * b[0] - a[1:] @ b[1:]
    t, u = -2 * dot(p1, k1), -2 * dot(p1, k2)
    assert abs(acc / (8 * g ** 4 * (u / t + t / u)) - 1.0) < 1e-12


def test_fvoxx0_momentum_slots_and_definition():
    rng = np.random.default_rng(2)
    p, k = massless(rng), massless(rng)
    fo = oracle.helas_wavefunction(FN_OXXXX0, p, 1, +1)
    vc = oracle.helas_wavefunction(FN_VXXXX0, k, -1, +1)
    fvo = oracle.helas_vertex(VTX_FVOXX0, fo=fo, vc=vc, g=0.3)
    pf = p + k
    assert np.allclose([fvo[4].real, fvo[5].real, fvo[5].imag, fvo[4].imag], pf)
    want = -0.3 * (fo[:4] @ slash(vc[:4]) @ slash(pf)) / (pf[0] ** 2 - pf[1:] @ pf[1:])
    assert np.allclose(fvo[:4], want, rtol=1e-12, atol=1e-14)


def test_jioxx0_current_conservation_and_four_fermion_closed_form():
    g, gp = 0.31, -0.17
    rng = np.random.default_rng(11)
    for _ in range(5):
        # q(p1) qbar(p2) -> q'(p3) qbar'(p4), all massless, CM frame
        e = rng.uniform(50.0, 400.0)
        c, phi = rng.uniform(-0.9, 0.9), rng.uniform(-np.pi, np.pi)
        s_ = np.sqrt(1 - c * c)
        p1, p2 = np.array([e, 0, 0, e]), np.array([e, 0, 0, -e])
        p3 = np.array([e, e * s_ * np.cos(phi), e * s_ * np.sin(phi), e * c])
        p4 = np.array([e, -p3[1], -p3[2], -p3[3]])
        acc = 0.0
        for h in itertools.product((-1, 1), repeat=4):
            fi = oracle.helas_wavefunction(FN_IXXXX1, p1, h[0], +1)      # q in
            fo = oracle.helas_wavefunction(FN_OXXXX2, p2, h[1], -1)      # qbar in (flowing out)
            j = oracle.helas_vertex(VTX_JIOXX0, fi=fi, fo=fo, g=g)
            q = np.array([j[4].real, j[5].real, j[5].imag, j[4].imag])
            assert np.allclose(q, -(p1 + p2))                            # jio[4] = fo[4] - fi[4]
            assert abs(np.sum(METRIC * q * j[:4])) < 1e-10 * e * np.abs(j[:4]).max() + 1e-300
            fo3 = oracle.helas_wavefunction(FN_OXXXX0, p3, h[2], +1)     # q' out
            fi4 = oracle.helas_wavefunction(FN_IXXXX0, p4, h[3], -1)     # qbar' out (flowing in)
            acc += abs(oracle.helas_vertex(VTX_IOVXXX, fi=fi4, fo=fo3, vc=j, g=gp)) ** 2
        s = 4 * e * e
        t = -2 * (p1[0] * p3[0] - p1[1:] @ p3[1:])
        u = -2 * (p1[0] * p4[0] - p1[1:] @ p4[1:])
        assert abs(acc / (8 * g * g * gp * gp * (t * t + u * u) / (s * s)) - 1.0) < 1e-12
