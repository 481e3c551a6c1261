"""GPU parity for the rest of the path: event generation (Philox + RAMBO + cuts + weights),
the cross-section reduction, the host-buffer entry point, and the full-size configurations
of BASELINE.json in the launch configuration bench.py times (sampled outputs)."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_0908_4403_b200 import ALGO_SUBSET, ALGO_TREE2, FP32, FP64, Heget, workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hg():
    h = Heget(0, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    yield h
    h.close()


def both_generators(hg, name, N, first_event=0):
    c = workloads.CONFIGS[name]
    kw = dict(mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"], apply_cuts=c["apply_cuts"],
              first_event=first_event)
    mo, wo = oracle.gen_events(c["seed"], c["n"], N, pt_cut=workloads.PT_CUT, eta_cut=workloads.ETA_CUT,
                               dr_cut=workloads.DR_CUT, **kw)
    mg, wg = hg.gen_events(c["seed"], c["n"], N, **kw)
    torch.cuda.synchronize()
    return mo, wo, mg.cpu().numpy(), wg.cpu().numpy()


@pytest.mark.parametrize("name", workloads.ORDER)
def test_gen_events_matches_oracle(hg, name):
    N = 20000 + 37
    mo, wo, mg, wg = both_generators(hg, name, N)
    rs = mo[:, 0, 0] + mo[:, 1, 0]                      # scale of every component
    err = np.abs(mg - mo).max(axis=(1, 2)) / rs
    print("\n[gen parity] %s: momenta max rel %.3e median %.3e" % (name, err.max(), np.median(err)))
    # DESIGN.md reading R25: device log/sincos/pow differ from libm by ulps; RAMBO's conformal boost
    # amplifies an ulp by gamma^2 = (Q0/M)^2, unbounded for nearly collinear q_i (worst for n = 2,
    # measured max 1.2e-11), so the bound is on quantiles plus a loose cap
    assert np.median(err) < 1e-15 and np.quantile(err, 0.999) < 1e-12 and err.max() < 1e-9
    # cut decisions: identical except where an observable sits within 1e-9 of a threshold
    same = (wo != 0) == (wg != 0)
    assert same.mean() == 1.0 or (~same).sum() <= 1
    both = (wo != 0) & (wg != 0)
    assert both.sum() > 100
    assert np.max(np.abs(wg[both] / wo[both] - 1.0)) < 1e-11


def test_heget_rambo_is_the_fixed_energy_form(hg):
    mo, _ = oracle.gen_events(1, 3, 5000, mode=oracle.MODE_FIXED, a=1000.0)
    mg = hg.rambo(1, 3, 1000.0, 5000)
    torch.cuda.synchronize()
    mg = mg.cpu().numpy()
    assert np.array_equal(mg[:, 0], mo[:, 0]) and np.array_equal(mg[:, 1], mo[:, 1])
    assert np.abs(mg - mo).max() < 1e-8
    k = mg[:, 2:]
    assert np.abs(k.sum(axis=1) - [1000.0, 0, 0, 0]).max() < 1e-9
    m2 = k[..., 0] ** 2 - k[..., 1] ** 2 - k[..., 2] ** 2 - k[..., 3] ** 2
    assert np.median(np.abs(m2)) < 1e-9


def test_gen_events_shards_reproduce_the_whole(hg):
    c = workloads.CONFIGS["4gamma"]
    kw = dict(mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"], apply_cuts=True)
    m, w = hg.gen_events(1, 4, 1001, **kw)
    parts = []
    for rank in range(3):
        first, cnt = workloads.shard_range(1001, rank, 3)
        parts.append(hg.gen_events(1, 4, cnt, first_event=first, **kw))
    torch.cuda.synchronize()
    assert torch.equal(torch.cat([p[0] for p in parts]), m)
    assert torch.equal(torch.cat([p[1] for p in parts]), w)


def test_gen_events_empty(hg):
    m, w = hg.gen_events(1, 4, 0)
    assert m.shape == (0, 6, 4) and w.shape == (0,)


def test_invalid_arguments_are_refused_before_any_launch(hg):
    """include/heget.h, error behaviour: HEGET_EINVAL (-1) for n outside [2,8], N < 0 or above
    HEGET_MAX_EVENTS, a bad precision / algorithm, null or misaligned buffers -- checked before the
    buffers are touched, so the dummy pointers below are never dereferenced and nothing is launched."""
    lib, ctx = hg._lib, hg._ctx
    buf = torch.zeros(64, dtype=torch.float64, device=hg.device)
    ptr = buf.data_ptr()
    before = hg.launch_count()
    bad = [
        (ctx, ptr, 1, FP64, ptr, 1, None), (ctx, ptr, 9, FP64, ptr, 1, None),          # n
        (ctx, ptr, 4, FP64, ptr, -1, None), (ctx, ptr, 4, FP64, ptr, 1 << 31, None),   # N
        (ctx, ptr, 4, 2, ptr, 1, None),                                                # precision
        (ctx, None, 4, FP64, ptr, 1, None), (ctx, ptr, 4, FP64, None, 1, None),        # null buffers
        (ctx, ptr + 8, 4, FP64, ptr, 1, None),                                         # momenta not 16-byte aligned
        (None, ptr, 4, FP64, ptr, 1, None),                                            # no context
    ]
    for args in bad:
        assert lib.heget_amp2(*args) == -1, args
    assert lib.heget_amp2_algo(ctx, ptr, 4, FP64, 3, ptr, 1, None) == -1
    assert lib.heget_amp2_algo(ctx, ptr, 4, FP64, -1, ptr, 1, None) == -1
    assert lib.heget_list2_sum(ctx, ptr, 4, FP64, ptr, 1 << 31, None) == -1
    assert lib.heget_xsec_reduce(ctx, ptr, ptr, 4, 1 << 31, ptr, None) == -1
    assert lib.heget_histogram(ctx, ptr, ptr, 4, 1, 0, 0.0, 1.0, 4095, ptr, None) == -1   # nbins > HEGET_HIST_MAX_BINS
    assert lib.heget_histogram(ctx, ptr, ptr, 4, 1, 0, 1.0, 1.0, 8, ptr, None) == -1      # hi <= lo
    assert hg.launch_count() == before
    assert b"invalid argument" in lib.heget_strerror(-1)
    # the largest accepted N is a property of the header: 2^31 - 1
    hdr = open(__import__("os").path.join(__import__("os").path.dirname(__file__), "..", "include", "heget.h")).read()
    assert "#define HEGET_MAX_EVENTS 2147483647LL" in hdr
    assert lib.heget_amp2(ctx, ptr, 2, FP64, ptr, 0, None) == 0   # N = 0 is valid and launches nothing
    assert hg.launch_count() == before


@pytest.mark.parametrize("N", [0, 1, 255, 100003])
def test_xsec_reduce_matches_oracle_and_is_deterministic(hg, N):
    rng = np.random.default_rng(N)
    a = rng.uniform(0.5, 2.0, size=N) * 1e-7
    w = rng.uniform(0.0, 1.0, size=N)
    w[::3] = 0.0
    ref = oracle.xsec_reduce(a, w, 5)
    da, dw = torch.from_numpy(a).cuda(), torch.from_numpy(w).cuda()
    r1 = hg.xsec_reduce(da, dw, 5).cpu().numpy()
    r2 = hg.xsec_reduce(da, dw, 5).cpu().numpy()
    assert np.array_equal(r1, r2)
    assert r1[2] == ref[2]
    assert abs(r1[0] - ref[0]) <= 1e-13 * abs(ref[0]) and abs(r1[1] - ref[1]) <= 1e-13 * abs(ref[1])


def test_xsec_reduce_on_two_streams_does_not_share_scratch(hg):
    """[dev] calls of one context may run concurrently on different streams (include/heget.h): the
    block partials of heget_xsec_reduce come from a ring of HEGET_REDUCE_SLOTS buffers, so reductions
    issued back to back on two streams must each give the result they give alone."""
    N = 1 << 22
    rng = np.random.default_rng(7)
    sets = []
    for k in range(2):
        a = torch.from_numpy(rng.uniform(0.5, 2.0, size=N) * 10.0 ** (-7 - 3 * k)).cuda()
        w = torch.from_numpy(rng.uniform(0.1, 1.0, size=N)).cuda()
        sets.append((a, w, hg.xsec_reduce(a, w, 4).clone()))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for _ in range(20):
        outs = []
        for k in (0, 1, 0, 1):
            with torch.cuda.stream(streams[k]):
                outs.append((k, hg.xsec_reduce(sets[k][0], sets[k][1], 4)))
        torch.cuda.synchronize()
        for k, o in outs:
            assert torch.equal(o, sets[k][2])
    # heget_xsec_host has partials of its own: it may follow a reduction that is still running
    hm, hw = sets[0][0].cpu().pin_memory(), sets[0][1].cpu().pin_memory()
    mom, _ = oracle.gen_events(2, 2, 64)
    with torch.cuda.stream(streams[0]):
        pending = hg.xsec_reduce(sets[1][0], sets[1][1], 4)
    h3 = hg.xsec_host(torch.from_numpy(mom), torch.ones(64, dtype=torch.float64), FP64)
    torch.cuda.synchronize()
    assert torch.equal(pending, sets[1][2]) and torch.isfinite(h3).all()


def test_xsec_reduce_ignores_amp2_of_events_that_failed_the_cuts(hg):
    """DESIGN.md R26: a NaN / Inf amp2 under weight 0 contributes exactly 0 (oracle pinned the same way)."""
    rng = np.random.default_rng(1)
    a = rng.uniform(0.5, 2.0, size=5000)
    w = rng.uniform(0.1, 1.0, size=5000)
    w[::7] = 0.0
    clean = hg.xsec_reduce(torch.from_numpy(a).cuda(), torch.from_numpy(w).cuda(), 3).cpu().numpy()
    b = a.copy()
    b[::21], b[7::21], b[14::21] = np.nan, np.inf, -np.inf
    dirty = hg.xsec_reduce(torch.from_numpy(b).cuda(), torch.from_numpy(w).cuda(), 3).cpu().numpy()
    assert np.array_equal(clean, dirty) and np.all(np.isfinite(dirty))
    ref = oracle.xsec_reduce(b, w, 3)
    assert ref[2] == dirty[2] and abs(dirty[0] / ref[0] - 1.0) < 1e-13


def test_gen_events_rejects_what_it_cannot_generate():
    """heget_gen_events: TOYPDF needs tau_min = (n pt_cut)^2 / s inside (0, 1); weight must not be NULL;
    heget_init rejects non-finite or negative cuts."""
    import ctypes
    from paper_0908_4403_b200 import binding
    lib = binding.load_library()
    ctx = ctypes.c_void_p()
    for bad in ((float("nan"), 2.5, 0.4), (20.0, float("inf"), 0.4), (20.0, 2.5, -1.0)):
        assert lib.heget_init(0, workloads.ALPHA, workloads.Q_U, *bad, ctypes.byref(ctx)) == -1
    assert lib.heget_init(0, workloads.ALPHA, float("nan"), 20.0, 2.5, 0.4, ctypes.byref(ctx)) == -1
    h0 = Heget(0, workloads.ALPHA, workloads.Q_U, 0.0, 2.5, 0.4)          # pt_cut = 0: tau_min = 0
    try:
        with pytest.raises(Exception):
            h0.gen_events(1, 4, 16, mode=workloads.TOYPDF, a=14000.0, apply_cuts=False)
        m, w = h0.gen_events(1, 4, 16, mode=workloads.LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5)   # fine without tau_min
        assert torch.isfinite(m).all() and torch.isfinite(w).all()
        cfg = binding.GenCfg(workloads.LOGUNIFORM, 0, 200.0, 3000.0, 1.5)
        assert lib.heget_gen_events(h0._ctx, 1, 4, ctypes.byref(cfg), 0, 16, m.data_ptr(), None, None) == -1   # weight NULL
    finally:
        h0.close()
    h1 = Heget(0, workloads.ALPHA, workloads.Q_U, 2000.0, 2.5, 0.4)       # 8 x 2 TeV > 14 TeV: tau_min > 1
    try:
        with pytest.raises(Exception):
            h1.gen_events(1, 8, 16, mode=workloads.TOYPDF, a=14000.0, apply_cuts=True)
    finally:
        h1.close()


@pytest.mark.parametrize("precision", [FP64, FP32])
def test_xsec_host_equals_device_path(hg, precision):
    mo, wo = oracle.gen_events(1, 4, 3000, mode=oracle.MODE_LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5,
                               apply_cuts=True)
    hm, hw = torch.from_numpy(mo), torch.from_numpy(wo)
    out_amp2 = torch.empty(3000, dtype=torch.float64)
    out3 = hg.xsec_host(hm, hw, precision, out_amp2=out_amp2)
    dm, dw = hm.cuda(), hw.cuda()
    a = hg.amp2(dm, precision)
    r = hg.xsec_reduce(a, dw, 4)
    torch.cuda.synchronize()
    assert torch.equal(a.cpu(), out_amp2) and torch.equal(r.cpu(), out3)
    # and the whole chain against the oracle
    ref = oracle.xsec_reduce(oracle.amp2(mo), wo, 4)
    tol = 1e-12 if precision == FP64 else 1e-5
    assert abs(out3[0].item() / ref[0] - 1.0) < tol and out3[2].item() == ref[2]


def test_xsec_host_pipelined_chunks_equal_device_path(hg):
    """N >= 65536 takes the chunked path (H2D of chunk c+1 overlapping chunk c's kernel); a ragged
    N that the 8 chunks do not divide must give bit-identical amp2 and sums."""
    N = 65536 + 4099
    c = workloads.CONFIGS["2gamma"]
    dm, dw = hg.gen_events(3, 2, N, mode=workloads.LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5, apply_cuts=True)
    hm, hw = dm.cpu().pin_memory(), dw.cpu().pin_memory()
    out_amp2 = torch.empty(N, dtype=torch.float64).pin_memory()
    for precision in (FP64, FP32):
        out3 = hg.xsec_host(hm, hw, precision, out_amp2=out_amp2)
        a = hg.amp2(dm, precision)
        r = hg.xsec_reduce(a, dw, c["n"])
        torch.cuda.synchronize()
        assert torch.equal(a.cpu(), out_amp2) and torch.equal(r.cpu(), out3)
        again = hg.xsec_host(hm, hw, precision)           # staging buffers reused
        assert torch.equal(again, out3)


def test_other_quark_flavour_rescales_with_charge(hg):
    """SURVEY 8(f) NEXT-4, flavours: the amplitude is proportional to Q_q^n, so a d-type line
    (Q = -1/3) gives (1/2)^(2n) of the u-type result; the oracle is evaluated with g of that
    charge, the library through heget_init's q_charge."""
    hd = Heget(0, workloads.ALPHA, -1.0 / 3.0, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    try:
        for n in (2, 5):
            mom, w = oracle.gen_events(4, n, 40, mode=oracle.MODE_LOGUNIFORM, a=300.0, b=3000.0, y_max=1.5,
                                       apply_cuts=True)
            g_d = oracle.G_DEFAULT * (-1.0 / 3.0) / workloads.Q_U
            ref = oracle.amp2(mom, g=g_d, extended=True)
            d = torch.from_numpy(mom).cuda()
            got_d = hd.amp2(d, FP64).cpu().numpy()
            got_u = hg.amp2(d, FP64).cpu().numpy()
            assert np.all(np.abs(got_d / ref - 1.0)[w != 0] <= 1e-12)
            assert np.all(np.abs(got_d / got_u * 4.0 ** n - 1.0) <= 1e-13)
    finally:
        hd.close()


def test_fma_peak_patterns_are_ordered(hg):
    """Roofline denominators: constant-operand FMA >= node pattern >= three-register FMA, and the
    constant-operand figure is within the B200's theoretical non-tensor peak."""
    for prec, lanes in ((FP32, 128), (FP64, 64)):
        p0, p1, p2 = (hg.fma_peak(prec, k) for k in (0, 1, 2))
        sm = torch.cuda.get_device_properties(0).multi_processor_count
        assert p0 <= sm * lanes * 2 * 2.2e9 and p0 >= 0.5 * sm * lanes * 2 * 1.0e9
        assert p0 >= p2 * 0.98 and p2 >= p1 * 0.98


def test_two_photon_cross_section_closed_form_on_gpu(hg):
    """Pin P11 through the CUDA path: gen (eta cut only) -> amp2 -> reduce vs the closed form."""
    h = Heget(0, workloads.ALPHA, workloads.Q_U, 0.0, 2.5, 0.0)
    N, rs = 1 << 20, 1000.0
    m, w = h.gen_events(1, 2, N, mode=0, a=rs, apply_cuts=True)
    s1, s2, cnt = h.xsec_reduce(h.amp2(m), w, 2).cpu().numpy()
    h.close()
    c = math.tanh(2.5)
    e4q4 = (4 * math.pi * workloads.ALPHA) ** 2 * workloads.Q_U ** 4
    sigma = (1 / (2 * rs * rs)) / 36.0 * 0.5 / (16 * math.pi) * 8 * e4q4 * 4 * (math.log((1 + c) / (1 - c)) - c)
    mean = s1 / N
    err = math.sqrt((s2 / N - mean * mean) / N)
    assert abs(mean - sigma) < 4 * err and err < 2e-3 * sigma
    assert abs(cnt / N - c) < 4 * math.sqrt(c * (1 - c) / N)


FULL_SAMPLES = {"2gamma": 4096, "3gamma": 4096, "4gamma": 4096, "5gamma": 512}
GOLDEN = __import__("os").path.join(__import__("os").path.dirname(__file__), "golden")


@pytest.mark.parametrize("name", workloads.ORDER)
def test_full_size_config_sampled_against_oracle(hg, name):
    """BASELINE.json's full event counts, the launch configuration bench.py times.  Inputs come
    from the oracle's generator; sampled events are checked one by one, the rest by properties
    that hold at any size (finite, positive, identical to a re-evaluation of a sub-batch)."""
    c = workloads.CONFIGS[name]
    n, N = c["n"], c["N"]
    mom, w = oracle.gen_events(c["seed"], n, N, mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                               apply_cuts=c["apply_cuts"])
    dm = torch.from_numpy(mom).cuda()
    out64 = hg.amp2(dm, FP64)
    out32 = hg.amp2(dm, FP32)
    torch.cuda.synchronize()
    g64, g32 = out64.cpu().numpy(), out32.cpu().numpy()
    assert np.all(np.isfinite(g64)) and np.all(g64 > 0) and np.all(np.isfinite(g32)) and np.all(g32 > 0)
    passing = np.flatnonzero(w != 0)
    if n >= 6:
        # every cut-passing event of the subset BASELINE.json states (first 2,048 / 4,096 / 512 events),
        # against the stored oracle<long double> values (tests/golden/, test_golden_sets.py)
        path = __import__("os").path.join(GOLDEN, "amp2_%s.npz" % name)
        if not __import__("os").path.exists(path):
            pytest.skip("missing %s" % path)
        g = np.load(path)
        assert np.array_equal(mom[: len(g["weight"])], g["momenta"])
        idx = np.flatnonzero(g["has_ld"])
        ref = g["amp2_ld"][idx]
    else:
        rng = np.random.default_rng(123)
        idx = np.sort(rng.choice(passing, size=FULL_SAMPLES[name], replace=False))
        idx = np.union1d(idx, [passing[0], passing[-1]])
        ref = oracle.amp2(mom[idx], extended=True)
    r64 = np.abs(g64[idx] / ref - 1.0)
    r32 = np.abs(g32[idx] / ref - 1.0)
    print("\n[full-size parity] %s N=%d sampled=%d: fp64 max %.3e median %.3e; fp32 max %.3e median %.3e"
          % (name, N, len(idx), r64.max(), np.median(r64), r32.max(), np.median(r32)))
    assert np.all(r64 <= 1e-12) and np.all(r32 <= 1e-4)
    # fp32 against fp64 on every passing event of the run
    rel = np.abs(g32[passing] / g64[passing] - 1.0)
    assert rel.max() <= 1e-4
    # a sub-batch evaluated alone reproduces the full launch bit for bit
    lo = N // 2 + 1
    sub = hg.amp2(dm[lo:lo + 300].contiguous(), FP64).cpu().numpy()
    assert np.array_equal(sub, g64[lo:lo + 300])
    # the other organisations of the permutation sum (heget_amp2_algo: subset recursion,
    # two-sided chaining) at the same full size: sampled events against the oracle, every
    # passing event against the tree mode
    for algo, tag in ((ALGO_SUBSET, "subset"), (ALGO_TREE2, "two-sided")):
        s64 = hg.amp2(dm, FP64, algo=algo).cpu().numpy()
        s32 = hg.amp2(dm, FP32, algo=algo).cpu().numpy()
        q64 = np.abs(s64[idx] / ref - 1.0)
        q32 = np.abs(s32[idx] / ref - 1.0)
        print("[full-size parity] %s %s mode: fp64 max %.3e median %.3e; fp32 max %.3e median %.3e"
              % (name, tag, q64.max(), np.median(q64), q32.max(), np.median(q32)))
        assert np.all(q64 <= 1e-12) and np.all(q32 <= 1e-4)
        assert np.abs(s64[passing] / g64[passing] - 1.0).max() <= 2e-12
        assert np.abs(s32[passing] / g64[passing] - 1.0).max() <= 1e-4
