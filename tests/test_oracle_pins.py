"""Pins for the CPU oracle (oracle/): closed forms, invariants and special cases that the
paper and the mathematics fix, none of them computed by the oracle itself.

Pin labels P1..P11 are those of DESIGN.md section "What pins the oracle".  Every expected
value below is either a textbook closed form typed out here in numpy, a property that must
hold exactly, or a value printed in PAPER.md / a published test vector (tests/golden/).
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle

G = oracle.G_DEFAULT
E2Q2 = 4.0 * math.pi * oracle.ALPHA * oracle.Q_U ** 2  # e^2 Q_u^2
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def mdot(a, b):
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


def events(n, N, seed=7, rs=1000.0):
    mom, _ = oracle.gen_events(seed, n, N, mode=oracle.MODE_FIXED, a=rs)
    return mom


def central(mom, min_frac=0.05):
    """Events whose photons all have k^+ and k^- above min_frac*omega (away from the beam) --
    keeps closed-form comparisons away from the ill-conditioned collinear corner."""
    k = mom[:, 2:]
    ok = np.all((k[..., 0] - np.abs(k[..., 3])) > min_frac * k[..., 0], axis=1)
    return mom[ok]


# ---------------------------------------------------------------- Dirac algebra


def test_gamma_matrices_clifford_algebra_and_chirality():
    g = [oracle.gamma(mu) for mu in range(4)]
    metric = np.diag([1.0, -1.0, -1.0, -1.0])
    for mu in range(4):
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.array_equal(anti, 2.0 * metric[mu, nu] * np.eye(4))
    g5 = 1j * g[0] @ g[1] @ g[2] @ g[3]
    # components 0,1 left-handed, 2,3 right-handed (eq. 16)
    assert np.array_equal(g5, np.diag([-1.0, -1.0, 1.0, 1.0]).astype(complex))
    # gamma^0 hermitian, gamma^i anti-hermitian
    assert np.array_equal(g[0], g[0].conj().T)
    for i in (1, 2, 3):
        assert np.array_equal(g[i], -g[i].conj().T)


def slash(a):
    g = [oracle.gamma(mu) for mu in range(4)]
    return a[0] * g[0] - a[1] * g[1] - a[2] * g[2] - a[3] * g[3]


def test_external_spinors_obey_massless_dirac_equation_and_normalisation():
    rng = np.random.default_rng(3)
    for _ in range(20):
        v = rng.normal(size=3) * 100.0
        p = np.array([np.linalg.norm(v), *v])
        for nhel in (-1, 1):
            for nsf in (-1, 1):
                fi = oracle.wavefunction("i", p, nhel, nsf)
                fo = oracle.wavefunction("o", p, nhel, nsf)
                assert np.max(np.abs(slash(p) @ fi)) < 1e-11 * p[0] ** 1.5
                assert np.max(np.abs(fo @ slash(p))) < 1e-11 * p[0] ** 1.5
                # fo = fi^dagger gamma^0 for the same (p, nhel, nsf)
                assert np.allclose(fo, fi.conj() @ oracle.gamma(0), rtol=1e-14, atol=0)
                # u^dagger u = 2 p0
                assert abs(np.vdot(fi, fi).real - 2.0 * p[0]) < 1e-12 * p[0]
                # chirality: nh = nhel*nsf = +1 -> right-handed slots (2,3) for |fi>
                if nhel * nsf == 1:
                    assert fi[0] == 0 and fi[1] == 0
                    assert fo[2] == 0 and fo[3] == 0      # List 8 fragment
                else:
                    assert fi[2] == 0 and fi[3] == 0
                    assert fo[0] == 0 and fo[1] == 0


def test_beam_direction_spinors_have_one_component():
    # ixxxx1: p along +z; oxxxx2: p along -z, nSF=-1
    e = 321.0
    for nhel in (-1, 1):
        fi = oracle.wavefunction("i", [e, 0, 0, e], nhel, +1)
        assert np.count_nonzero(fi) == 1 and abs(abs(fi).max() - math.sqrt(2 * e)) < 1e-13
        fo = oracle.wavefunction("o", [e, 0, 0, -e], nhel, -1)
        assert np.count_nonzero(fo) == 1 and abs(abs(fo).max() - math.sqrt(2 * e)) < 1e-13


def test_polarisation_vectors_light_cone_gauge():
    rng = np.random.default_rng(5)
    for _ in range(20):
        v = rng.normal(size=3) * 50.0
        p = np.array([np.linalg.norm(v), *v])
        nvec = np.array([p[0], -p[1], -p[2], -p[3]])           # eq. (15)
        eps = {}
        for lam in (-1, 1):
            for nsv in (-1, 1):
                e = oracle.wavefunction("v", p, lam, nsv)
                eps[(lam, nsv)] = e
                assert e[0] == 0
                assert abs(mdot(e, p.astype(complex))) < 1e-13 * p[0]      # transversality
                assert abs(mdot(e, nvec.astype(complex))) < 1e-13 * p[0]   # eq. (14)
                assert abs(mdot(e, e.conj()) + 1.0) < 1e-13                # eps.eps^* = -1
                assert abs(mdot(e, e)) < 1e-13                             # eps.eps = 0
        for lam in (-1, 1):
            # eq. (13a/b): nSV=+1 is the complex conjugate of nSV=-1
            assert np.allclose(eps[(lam, 1)], eps[(lam, -1)].conj(), rtol=0, atol=1e-15)
            # eps(-lambda) = -eps(lambda)^*
            assert np.allclose(eps[(-lam, 1)], -eps[(lam, 1)].conj(), rtol=0, atol=1e-15)
        # opposite helicities are orthogonal: eps(+).eps(-)^* = 0
        assert abs(mdot(eps[(1, 1)], eps[(-1, 1)].conj())) < 1e-13


def test_polarisation_slash_chiral_blocks_have_rank_one():
    """eps-slash eps-slash = eps.eps = 0 for a circularly polarised massless photon, so each 2x2
    chiral block of eps-slash (chiral representation, eq. 16 at PAPER.md:248) is singular: it is a
    column times a row.  The factorised tree nodes of the CUDA path (v9) rest on
    this property of vxxxx0 (eqs. 13-15); here it is checked on the oracle's
    own polarisation vectors and gamma matrices."""
    rng = np.random.default_rng(17)
    metric = np.array([1.0, -1.0, -1.0, -1.0])
    for _ in range(20):
        v = rng.normal(size=3) * 80.0
        p = np.array([np.linalg.norm(v), *v])
        for lam in (-1, 1):
            e = oracle.wavefunction("v", p, lam, 1)
            slash = sum(metric[mu] * e[mu] * oracle.gamma(mu) for mu in range(4))
            assert np.abs(slash @ slash).max() < 1e-13
            upper, lower = slash[:2, 2:], slash[2:, :2]
            assert np.abs(slash[:2, :2]).max() == 0 and np.abs(slash[2:, 2:]).max() == 0
            for blk in (upper, lower):
                scale = np.abs(blk).max() ** 2
                assert scale > 1e-3                                   # the block itself is not zero
                assert abs(np.linalg.det(blk)) < 1e-13 * max(scale, 1.0)
                assert np.linalg.matrix_rank(blk, tol=1e-10) == 1


def test_polarisation_vector_matches_paper_lists_9_and_10():
    # tests/golden/vxxxx_lists_9_10.txt: values printed in PAPER.md:553-559 (List 9, +z)
    # and 571-577 (List 10, -z); both lists are the nSV = -1 (initial-state) form.
    rows = [l.split() for l in open(os.path.join(GOLDEN, "vxxxx_lists_9_10.txt"))
            if l.strip() and not l.startswith("#")]
    r2 = 1.0 / math.sqrt(2.0)
    for direction, nhel, c1re, c2im in rows:
        pz = 80.0 if direction == "+z" else -80.0
        e = oracle.wavefunction("v", [80.0, 0.0, 0.0, pz], int(nhel), -1)
        assert e[0] == 0 and e[3] == 0
        assert abs(e[1] - float(c1re) * r2) < 1e-15
        assert abs(e[2] - 1j * float(c2im) * r2) < 1e-15
    # the generic-direction formula tends to the lists continuously: +z approached at
    # azimuth phi = 0, -z approached at phi = pi (the lists fix that phase convention)
    for sgn in (1.0, -1.0):
        th = 1e-7
        p = [80.0, sgn * 80.0 * math.sin(th), 0.0, sgn * 80.0 * math.cos(th)]
        for lam in (-1, 1):
            gen = oracle.wavefunction("v", p, lam, -1)
            lim = oracle.wavefunction("v", [80.0, 0.0, 0.0, sgn * 80.0], lam, -1)
            assert np.allclose(gen, lim, rtol=0, atol=1e-6)


# ---------------------------------------------------------------- amplitudes


def all_helicities(n):
    return itertools.product((-1, 1), repeat=n + 2)


def test_P1_two_photon_closed_form():
    """sum |M|^2 = 8 e^4 Q^4 (u/t + t/u)  (north_star: (1/4) sum = 2 e^4 Q^4 (u/t+t/u))."""
    mom = events(2, 4000)
    p1, k1, k2 = mom[:, 0], mom[:, 2], mom[:, 3]
    t = mdot(p1 - k1, p1 - k1)
    u = mdot(p1 - k2, p1 - k2)
    expect = 8.0 * E2Q2 ** 2 * (u / t + t / u)
    got = oracle.amp2(mom)
    # The closed form holds for exactly massless, momentum-conserving momenta.  RAMBO's
    # output is that only up to rounding (amplified by its boost), so the formula and the
    # amplitude on the stored doubles may differ by (input residue)/min(|t|,|u|).
    p2 = mom[:, 1]
    d = p1 + p2 - k1 - k2
    res = np.maximum.reduce([np.abs(mdot(k1, k1)), np.abs(mdot(k2, k2)), np.abs(d).max(axis=1) * 1000.0])
    bound = res / np.minimum(np.abs(t), np.abs(u))
    err = np.abs(got / expect - 1.0)
    assert np.all(err < 4.0 * bound + 1e-14)
    assert np.median(err) < 3e-15
    assert np.mean(err < 1e-13) > 0.99
    # the constant BASELINE/SURVEY quote for alpha = 1/128, Q = 2/3
    assert abs(8.0 * E2Q2 ** 2 - 0.015230870989335427) < 1e-17


def mhv_expected(mom, j, cube_on_a):
    """(2 e^2 Q^2)^n s12^(n-2) a_j^3 b_j / prod(a_i b_i)  (or a_j b_j^3): the
    Kleiss-Stirling / Brown-Hagiwara-Martin single-flipped-helicity result the paper's
    ref. [5] gives for q qbar -> n gamma."""
    n = mom.shape[0] - 2
    p1, p2, k = mom[0], mom[1], mom[2:]
    a = 2.0 * mdot(p1[None], k)
    b = 2.0 * mdot(p2[None], k)
    s12 = 2.0 * mdot(p1, p2)
    num = a[j] ** 3 * b[j] if cube_on_a else a[j] * b[j] ** 3
    return (2.0 * E2Q2) ** n * s12 ** (n - 2) * num / np.prod(a * b)


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_P2_P3_mhv_amplitudes_and_zeros(n):
    mom_all = central(events(n, 60, seed=11))[:4]
    assert len(mom_all) == 4
    for mom in mom_all:
        scale = mhv_expected(mom, 0, True)
        for nhel in all_helicities(n):
            s1, s2, lam = nhel[0], nhel[1], nhel[2:]
            m2 = abs(oracle.amp(mom, nhel)) ** 2
            if s1 == s2:
                assert m2 == 0.0                                   # P3: helicity conservation
                continue
            npos = sum(1 for x in lam if x == 1)
            if npos == 0 or npos == n:
                assert m2 < 1e-24 * scale                          # all-equal photon helicities
            elif npos == 1 or npos == n - 1:
                lone = +1 if npos == 1 else -1     # n = 2: (+,-) read as lone +; same value
                j = lam.index(lone)
                # a_j^3 b_j when the lone photon's helicity is opposite to the quark's
                cube_on_a = (s1 * lone == -1)
                exp = mhv_expected(mom, j, cube_on_a)
                assert abs(m2 / exp - 1.0) < 5e-12, (nhel, m2, exp)


def test_P2_three_photon_total_closed_form():
    mom = central(events(3, 600, seed=13))
    p1, p2, k = mom[:, 0], mom[:, 1], mom[:, 2:]
    a = 2.0 * mdot(p1[:, None], k)
    b = 2.0 * mdot(p2[:, None], k)
    s12 = 2.0 * mdot(p1, p2)
    expect = 2.0 * (2.0 * E2Q2) ** 3 * s12 * np.sum(a * b * (a ** 2 + b ** 2), axis=1) / np.prod(a * b, axis=1)
    got = oracle.amp2(mom)
    assert len(mom) > 200
    assert np.max(np.abs(got / expect - 1.0)) < 1e-12


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_P4_gauge_invariance(n):
    """eps(k_i) -> k_i kills the full amplitude (sum over all n! diagrams) while single
    diagrams do not vanish: compare with the amplitude's natural size |M| * omega_i."""
    mom_all = central(events(n, 40, seed=17))[:3]
    rng = np.random.default_rng(1)
    for mom in mom_all:
        for _ in range(6):
            nhel = [1, -1] + list(rng.choice([-1, 1], size=n))
            if rng.random() < 0.5:
                nhel[0], nhel[1] = -1, 1
            ref = max(abs(oracle.amp(mom, [nhel[0], nhel[1]] + list(l))) for l in
                      itertools.product((-1, 1), repeat=n))
            for i in range(n):
                m = abs(oracle.amp(mom, nhel, gauge_idx=i))
                assert m < 1e-10 * ref * mom[2 + i, 0], (n, i, m, ref)


def test_P4_gauge_probe_is_not_trivially_zero():
    # with the wrong (non-conserved) current -- one diagram dropped by making photon
    # momenta violate momentum conservation -- the Ward identity fails: the probe has teeth
    mom = central(events(3, 40, seed=17))[0].copy()
    nhel = [1, -1, 1, -1, 1]
    ok = abs(oracle.amp(mom, nhel, gauge_idx=0))
    mom[1] = [mom[1, 0] * 1.3, 0, 0, -mom[1, 0] * 1.3]   # ubar momentum no longer p_gammas - p1
    # (the amplitude never uses p2 except through v-bar's normalisation, so break a photon instead)
    mom2 = central(events(3, 40, seed=17))[0].copy()
    mom2[3, 1:] *= 1.2
    mom2[3, 0] = np.linalg.norm(mom2[3, 1:])
    bad = abs(oracle.amp(mom2, nhel, gauge_idx=0))
    assert bad > 1e6 * ok


@pytest.mark.parametrize("n", [3, 4, 5])
def test_P5_bose_symmetry(n):
    mom = central(events(n, 40, seed=19))[:6]
    base = oracle.amp2(mom)
    rng = np.random.default_rng(2)
    for _ in range(3):
        perm = rng.permutation(n)
        m2 = mom.copy()
        m2[:, 2:] = mom[:, 2 + perm]
        assert np.max(np.abs(oracle.amp2(m2) / base - 1.0)) < 1e-12
    # per helicity: permuting photons together with their helicities leaves M unchanged
    ev = mom[0]
    nhel = [1, -1] + [1, -1, -1, 1, 1][:n]
    perm = np.roll(np.arange(n), 1)
    ev2 = ev.copy()
    ev2[2:] = ev[2 + perm]
    nhel2 = nhel[:2] + [nhel[2 + p] for p in perm]
    a, b = oracle.amp(ev, nhel), oracle.amp(ev2, nhel2)
    assert abs(a - b) < 1e-12 * abs(a)


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_P6_scaling_rotation_boost_reflection(n):
    mom = central(events(n, 40, seed=23))[:6]
    base = oracle.amp2(mom)
    # homogeneity: sum|M|^2 (lambda p) = lambda^(2(2-n)) sum|M|^2 (p)
    lam = 0.37
    assert np.max(np.abs(oracle.amp2(lam * mom) / (lam ** (2 * (2 - n)) * base) - 1.0)) < 1e-12
    # rotation about the beam axis
    c, s = math.cos(0.83), math.sin(0.83)
    rot = mom.copy()
    rot[..., 1] = c * mom[..., 1] - s * mom[..., 2]
    rot[..., 2] = s * mom[..., 1] + c * mom[..., 2]
    assert np.max(np.abs(oracle.amp2(rot) / base - 1.0)) < 1e-12
    # boost along the beam axis (the light-cone gauge vector of eq. 15 is frame dependent,
    # the helicity sum is not)
    y = 0.9
    bst = mom.copy()
    bst[..., 0] = math.cosh(y) * mom[..., 0] + math.sinh(y) * mom[..., 3]
    bst[..., 3] = math.cosh(y) * mom[..., 3] + math.sinh(y) * mom[..., 0]
    assert np.max(np.abs(oracle.amp2(bst) / base - 1.0)) < 1e-11
    # reflection y -> -y (parity times a rotation)
    ref = mom.copy()
    ref[..., 2] = -mom[..., 2]
    assert np.max(np.abs(oracle.amp2(ref) / base - 1.0)) < 1e-12
    # parity relation between single helicity amplitudes: |M(-h)| = |M(h)|
    rng = np.random.default_rng(4)
    for _ in range(4):
        nhel = [1, -1] + list(rng.choice([-1, 1], size=n))
        a = abs(oracle.amp(mom[0], nhel))
        b = abs(oracle.amp(mom[0], [-h for h in nhel]))
        assert abs(a - b) <= 1e-12 * max(a, b)


@pytest.mark.parametrize("n", [3, 4])
def test_P7_soft_photon_limit(n):
    """omega_n -> 0: sum|M_n|^2 -> sum|M_(n-1)|^2 * e^2 Q^2 * 4 s12/(a_n b_n)  (eikonal factor
    -e^2Q^2 (p1/(p1.k) - p2/(p2.k))^2 = 4 e^2 Q^2 p1.p2 /((2p1.k)(2p2.k)) * ... ), error O(omega/E)."""
    hard = central(events(n - 1, 40, seed=29))[:4]
    for ev in hard:
        ratios = []
        for omega in (1e-2, 1e-4):
            d = np.array([0.3, -0.5, 0.4])
            d /= np.linalg.norm(d)
            soft = np.array([omega, *(omega * d)])
            # the hard photons recoil against the soft one: rescale them to invariant mass
            # M' and boost them to total momentum P - k_soft, P = p1 + p2 = (sqrt_s, 0)
            rs = ev[0, 0] + ev[1, 0]
            tot = np.array([rs, 0.0, 0.0, 0.0]) - soft
            m_new = math.sqrt(mdot(tot, tot))
            hard_k = ev[2:] * (m_new / rs)
            bvec = tot[1:] / m_new
            gam = tot[0] / m_new
            bk = hard_k[:, 1:] @ bvec
            rec = np.empty_like(hard_k)
            rec[:, 0] = gam * hard_k[:, 0] + bk
            rec[:, 1:] = hard_k[:, 1:] + np.outer(hard_k[:, 0] + bk / (1.0 + gam), bvec)
            assert np.max(np.abs(rec.sum(axis=0) + soft - [rs, 0, 0, 0])) < 1e-9
            full = np.concatenate([ev[:2], rec, soft[None]], axis=0)
            p1, p2 = ev[0], ev[1]
            a, b = 2.0 * mdot(p1, soft), 2.0 * mdot(p2, soft)
            s12 = 2.0 * mdot(p1, p2)
            eik = E2Q2 * 4.0 * s12 / (a * b)
            got = oracle.amp2(full[None])[0]
            exp = oracle.amp2(ev[None])[0] * eik
            ratios.append(got / exp)
        assert abs(ratios[0] - 1.0) < 2e-3
        assert abs(ratios[1] - 1.0) < 2e-5


@pytest.mark.parametrize("n", [2, 4, 6])
def test_P8_precision_ladder(n):
    N = {2: 500, 4: 60, 6: 4}[n]
    mom = events(n, N, seed=31)
    d = oracle.amp2(mom)
    ld = oracle.amp2(mom, extended=True)
    k = mom[:, 2:]
    cen = np.all((k[..., 0] - np.abs(k[..., 3])) > 0.02 * k[..., 0], axis=1)
    assert np.max(np.abs(d[cen] / ld[cen] - 1.0)) < 1e-12
    assert np.all(np.abs(d / ld - 1.0) < 1e-9)


def test_amp2_equals_sum_over_single_helicity_amplitudes():
    mom = events(3, 3, seed=37)
    tot = oracle.amp2(mom)
    for e in range(3):
        s = sum(abs(oracle.amp(mom[e], h)) ** 2 for h in all_helicities(3))
        assert abs(s / tot[e] - 1.0) < 1e-14


def test_diagram_count_through_coupling_scaling():
    # M is homogeneous of degree n in g (n vertices per diagram, eq. 7): |M|^2 ~ g^(2n)
    for n in (2, 3, 4):
        mom = events(n, 2, seed=41)
        a = oracle.amp2(mom, g=G)
        b = oracle.amp2(mom, g=2.0 * G)
        assert np.max(np.abs(b / a / 4.0 ** n - 1.0)) < 1e-13
