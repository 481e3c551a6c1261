"""GPU parity of the HEGET function set (heget_helas_wavefunction, heget_helas_vertex; SURVEY 8(f)
NEXT-4) against the CPU oracle, element by element, through the C ABI.

Tolerance: every function is a handful of multiplications and additions of O(1)-conditioned
quantities (the off-shell ones divide by pf^2 or q^2, which the inputs here keep away from
zero), so each output w[6] must agree to 1e-13 (fp64) / 2e-5 (fp32) of its own largest component.
fp32 results are compared with the oracle evaluated on the SAME fp64 inputs (the kernel converts
on load)."""
import itertools

import numpy as np
import pytest
import torch

import oracle
from paper_0908_4403_b200 import FP32, FP64, Heget, binding, workloads

pytestmark = pytest.mark.gpu

TOL = {FP64: 1e-13, FP32: 2e-5}


@pytest.fixture(scope="module")
def hg():
    h = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    yield h
    h.close()


def momenta(N, seed):
    rng = np.random.default_rng(seed)
    e = rng.uniform(20.0, 800.0, N)
    c = rng.uniform(-0.98, 0.98, N)
    phi = rng.uniform(-np.pi, np.pi, N)
    s = np.sqrt(1 - c * c)
    return np.stack([e, e * s * np.cos(phi), e * s * np.sin(phi), e * c], axis=1)


def to_c(w):
    """[N][6][2] doubles -> [N][6] complex"""
    return w[..., 0] + 1j * w[..., 1]


def to_r(w):
    return np.ascontiguousarray(np.stack([w.real, w.imag], axis=-1))


def close(got, ref, tol):
    scale = np.abs(ref).max(axis=-1, keepdims=True) if ref.ndim > 1 else np.abs(ref)
    return np.all(np.abs(got - ref) <= tol * np.maximum(scale, 1e-300))


@pytest.mark.parametrize("precision", [FP64, FP32])
def test_wavefunctions_match_oracle(hg, precision):
    N = 256 * 3 + 17                          # several CTAs and a ragged tail
    p = momenta(N, 1)
    dp = torch.from_numpy(p).cuda()
    for fn, nhel, ns in itertools.product(range(9), (-1, 1), (-1, 1)):
        got = to_c(hg.helas_wavefunction(fn, dp, nhel, ns, precision).cpu().numpy())
        ref = np.array([oracle.helas_wavefunction(fn, p[e], nhel, ns) for e in range(0, N, 7)])
        assert close(got[::7], ref, TOL[precision]), (fn, nhel, ns)
        assert np.all(np.isfinite(got.view(np.float64)))


def build_inputs(N, seed):
    """On-shell fi, fo, vc for independent random momenta, all helicity / nS combinations mixed."""
    rng = np.random.default_rng(seed)
    pi_, po_, pv_ = momenta(N, seed + 1), momenta(N, seed + 2), momenta(N, seed + 3)
    hel = rng.choice([-1, 1], size=(N, 5))
    fi = np.array([oracle.helas_wavefunction(oracle.FN_IXXXX0, pi_[e], hel[e, 0], hel[e, 1]) for e in range(N)])
    fo = np.array([oracle.helas_wavefunction(oracle.FN_OXXXX0, po_[e], hel[e, 2], hel[e, 3]) for e in range(N)])
    vc = np.array([oracle.helas_wavefunction(oracle.FN_VXXXX0, pv_[e], hel[e, 4], 1) for e in range(N)])
    return fi, fo, vc


@pytest.mark.parametrize("precision", [FP64, FP32])
def test_vertices_match_oracle(hg, precision):
    N = 256 * 2 + 9
    g = oracle.G_DEFAULT
    fi, fo, vc = build_inputs(N, 20)
    dfi, dfo, dvc = (torch.from_numpy(to_r(w)).cuda() for w in (fi, fo, vc))
    tol = TOL[precision]
    amp = hg.helas_vertex(binding.VTX_IOVXXX, fi=dfi, fo=dfo, vc=dvc, g=g, precision=precision).cpu().numpy()
    amp = amp[:, 0] + 1j * amp[:, 1]
    ref = np.array([oracle.helas_vertex(oracle.VTX_IOVXXX, fi=fi[e], fo=fo[e], vc=vc[e], g=g) for e in range(N)])
    # an amplitude is a sum of products that may cancel (helicity zeros): scale = |fo||vc||fi| g
    scale = np.abs(g) * np.abs(fo[:, :4]).max(1) * np.abs(vc[:, :4]).max(1) * np.abs(fi[:, :4]).max(1)
    assert np.all(np.abs(amp - ref) <= 8 * tol * scale)
    for fn, kw in ((binding.VTX_FVIXX0, dict(fi=dfi, vc=dvc)), (binding.VTX_FVOXX0, dict(fo=dfo, vc=dvc)),
                   (binding.VTX_JIOXX0, dict(fi=dfi, fo=dfo))):
        got = to_c(hg.helas_vertex(fn, g=g, precision=precision, **kw).cpu().numpy())
        okw = {k: {"fi": fi, "fo": fo, "vc": vc}[k] for k in kw}
        ref = np.array([oracle.helas_vertex(fn, g=g, **{k: v[e] for k, v in okw.items()}) for e in range(N)])
        # off-shell denominators: skip the rare element whose pf^2 / q^2 nearly vanishes
        mom = ref[:, 4:]
        p2 = mom[:, 0].real ** 2 - mom[:, 0].imag ** 2 - mom[:, 1].real ** 2 - mom[:, 1].imag ** 2
        well = np.abs(p2) > 1e-3 * (mom[:, 0].real ** 2)
        assert well.sum() > 0.9 * N
        assert close(got[well][:, :4], ref[well][:, :4], 20 * tol), fn
        assert close(got[:, 4:], ref[:, 4:], tol), fn


def test_two_photon_amplitude_through_the_helas_set_on_gpu(hg):
    """List 2 for n = 2 evaluated on the GPU with the HEGET functions themselves (ixxxx1, oxxxx2,
    vxxxx0, fvoxx0, iovxxx) must square to what heget_amp2 returns."""
    N = 300
    mom, _ = oracle.gen_events(6, 2, N, mode=oracle.MODE_LOGUNIFORM, a=300.0, b=3000.0, y_max=1.0)
    d = torch.from_numpy(mom).cuda()
    g = oracle.G_DEFAULT
    p1, p2, k1, k2 = (d[:, i, :].contiguous() for i in range(4))
    total = torch.zeros(N, dtype=torch.float64, device="cuda")
    for h in itertools.product((-1, 1), repeat=4):
        fi = hg.helas_wavefunction(binding.FN_IXXXX1, p1, h[0], +1)
        fo = hg.helas_wavefunction(binding.FN_OXXXX2, p2, h[1], -1)
        v = [hg.helas_wavefunction(binding.FN_VXXXX0, k, hh, +1) for k, hh in ((k1, h[2]), (k2, h[3]))]
        amp = torch.zeros((N, 2), dtype=torch.float64, device="cuda")
        for a, b in ((0, 1), (1, 0)):
            fvo = hg.helas_vertex(binding.VTX_FVOXX0, fo=fo, vc=v[b], g=g)
            amp += hg.helas_vertex(binding.VTX_IOVXXX, fi=fi, fo=fvo, vc=v[a], g=g)
        total += (amp ** 2).sum(dim=1)
    want = hg.amp2(d, FP64)
    assert torch.all(torch.abs(total / want - 1.0) < 1e-11)
    assert np.all(np.abs(total.cpu().numpy() / oracle.amp2(mom, extended=True) - 1.0) < 1e-11)


def test_helas_argument_errors(hg):
    lib, ctx = hg._lib, hg._ctx
    p = torch.zeros((4, 4), dtype=torch.float64, device="cuda")
    w = torch.zeros((4, 6, 2), dtype=torch.float64, device="cuda")
    assert lib.heget_helas_wavefunction(ctx, 9, FP64, p.data_ptr(), 1, 1, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_wavefunction(ctx, 0, FP64, p.data_ptr(), 0, 1, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_wavefunction(ctx, 0, FP64, p.data_ptr(), 1, 2, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_wavefunction(ctx, 0, 3, p.data_ptr(), 1, 1, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_wavefunction(ctx, 0, FP64, None, 1, 1, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_wavefunction(ctx, 0, FP64, p.data_ptr(), 1, 1, w.data_ptr(), 0, None) == 0
    assert lib.heget_helas_vertex(ctx, 4, FP64, w.data_ptr(), w.data_ptr(), w.data_ptr(), 0.1, w.data_ptr(), 4, None) == -1
    assert lib.heget_helas_vertex(ctx, 1, FP64, None, None, w.data_ptr(), 0.1, w.data_ptr(), 4, None) == -1   # fvixx0 needs fi
    assert lib.heget_helas_vertex(ctx, 3, FP64, w.data_ptr(), w.data_ptr(), None, 0.1, w.data_ptr(), 0, None) == 0
