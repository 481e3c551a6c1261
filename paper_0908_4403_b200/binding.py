"""ctypes binding of libheget.so (include/heget.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; this module passes torch
tensors' device pointers and the current torch stream through the C ABI.  There is no CPU
fallback: a missing library or a CUDA-less host raises."""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libheget.so")

FP32, FP64 = 0, 1
ALGO_TREE, ALGO_SUBSET, ALGO_TREE2 = 0, 1, 2
OBS_PT_MAX, OBS_DR_MIN, OBS_DR_ALL = 0, 1, 2
FN_IXXXX0, FN_IXXXX1, FN_IXXXX2, FN_OXXXX0, FN_OXXXX1, FN_OXXXX2, FN_VXXXX0, FN_VXXXX1, FN_VXXXX2 = range(9)
VTX_IOVXXX, VTX_FVIXX0, VTX_FVOXX0, VTX_JIOXX0 = range(4)
GEN_FIXED, GEN_LOGUNIFORM, GEN_TOYPDF = 0, 1, 2

EXPORTS = ["heget_init", "heget_destroy", "heget_strerror", "heget_last_cuda_error", "heget_rambo",
           "heget_gen_events", "heget_amp2", "heget_amp2_algo", "heget_amp2_sampled", "heget_list2", "heget_list2_sum", "heget_histogram", "heget_helas_wavefunction", "heget_helas_vertex", "heget_xsec_reduce", "heget_xsec_reduce_noalloc", "heget_xsec_host", "heget_fma_peak", "heget_fma_peak_pattern",
           "heget_launch_count"]


class GenCfg(ctypes.Structure):
    _fields_ = [("mode", ctypes.c_int), ("apply_cuts", ctypes.c_int), ("a", ctypes.c_double),
                ("b", ctypes.c_double), ("y_max", ctypes.c_double)]


class HegetError(RuntimeError):
    pass


_lib = None


def load_library():
    """dlopen libheget.so and declare the prototypes of include/heget.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise HegetError("libheget.so is not built: run `python -m paper_0908_4403_b200.build` "
                         "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, dp, i64, u64, ci, cd = (ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64,
                                ctypes.c_int, ctypes.c_double)
    lib.heget_init.argtypes = [ci, cd, cd, cd, cd, cd, ctypes.POINTER(vp)]
    lib.heget_init.restype = ci
    lib.heget_destroy.argtypes = [vp]
    lib.heget_destroy.restype = None
    lib.heget_strerror.argtypes = [ci]
    lib.heget_strerror.restype = ctypes.c_char_p
    lib.heget_last_cuda_error.argtypes = [vp]
    lib.heget_last_cuda_error.restype = ctypes.c_char_p
    lib.heget_rambo.argtypes = [vp, u64, ci, cd, i64, dp, vp]
    lib.heget_rambo.restype = ci
    lib.heget_gen_events.argtypes = [vp, u64, ci, ctypes.POINTER(GenCfg), u64, i64, dp, dp, vp]
    lib.heget_gen_events.restype = ci
    lib.heget_amp2.argtypes = [vp, dp, ci, ci, dp, i64, vp]
    lib.heget_amp2.restype = ci
    lib.heget_amp2_algo.argtypes = [vp, dp, ci, ci, ci, dp, i64, vp]
    lib.heget_amp2_algo.restype = ci
    lib.heget_amp2_sampled.argtypes = [vp, u64, u64, dp, ci, ci, dp, vp, i64, vp]
    lib.heget_amp2_sampled.restype = ci
    lib.heget_list2.argtypes = [vp, u64, u64, dp, ci, ci, dp, vp, i64, vp]
    lib.heget_list2.restype = ci
    lib.heget_list2_sum.argtypes = [vp, dp, ci, ci, dp, i64, vp]
    lib.heget_list2_sum.restype = ci
    lib.heget_histogram.argtypes = [vp, dp, dp, ci, i64, ci, cd, cd, ci, dp, vp]
    lib.heget_histogram.restype = ci
    lib.heget_helas_wavefunction.argtypes = [vp, ci, ci, dp, ci, ci, dp, i64, vp]
    lib.heget_helas_wavefunction.restype = ci
    lib.heget_helas_vertex.argtypes = [vp, ci, ci, dp, dp, dp, cd, dp, i64, vp]
    lib.heget_helas_vertex.restype = ci
    lib.heget_xsec_reduce.argtypes = [vp, dp, dp, ci, i64, dp, vp]
    lib.heget_xsec_reduce.restype = ci
    lib.heget_xsec_reduce_noalloc.argtypes = [vp, dp, dp, ci, i64, dp, vp]
    lib.heget_xsec_reduce_noalloc.restype = ci
    lib.heget_xsec_host.argtypes = [vp, dp, dp, ci, ci, i64, dp, dp]
    lib.heget_xsec_host.restype = ci
    lib.heget_fma_peak.argtypes = [vp, ci, ctypes.POINTER(cd)]
    lib.heget_fma_peak.restype = ci
    lib.heget_fma_peak_pattern.argtypes = [vp, ci, ci, ctypes.POINTER(cd)]
    lib.heget_fma_peak_pattern.restype = ci
    lib.heget_launch_count.argtypes = [vp]
    lib.heget_launch_count.restype = i64
    _lib = lib
    return lib


def _stream_ptr(device):
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _check_dev(t, shape, device):
    if not (t.is_cuda and t.device == device and t.dtype == torch.float64 and t.is_contiguous()):
        raise HegetError("expected a contiguous float64 tensor on %s" % device)
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise HegetError("expected shape %s, got %s" % (tuple(shape), tuple(t.shape)))


class Heget:
    """One library context on one CUDA device (heget_init / heget_destroy)."""

    def __init__(self, device=0, alpha=1.0 / 128.0, q_charge=2.0 / 3.0, pt_cut=20.0, eta_cut=2.5, dr_cut=0.4):
        if not torch.cuda.is_available():
            raise HegetError("no CUDA device: libheget.so has no CPU fallback")
        self._lib = load_library()
        self.device = torch.device("cuda", device)
        self._ctx = ctypes.c_void_p()
        rc = self._lib.heget_init(device, alpha, q_charge, pt_cut, eta_cut, dr_cut, ctypes.byref(self._ctx))
        if rc != 0:
            self._ctx = None
            raise HegetError("heget_init: " + self._lib.heget_strerror(rc).decode())

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.heget_destroy(self._ctx)
            self._ctx = None

    __del__ = close

    def _check(self, rc, what):
        if rc != 0:
            msg = self._lib.heget_strerror(rc).decode()
            if rc == -2:
                msg += ": " + self._lib.heget_last_cuda_error(self._ctx).decode()
            raise HegetError("%s: %s" % (what, msg))

    def rambo(self, seed, n, sqrt_s_hat, N):
        momenta = torch.empty((N, n + 2, 4), dtype=torch.float64, device=self.device)
        self._check(self._lib.heget_rambo(self._ctx, seed, n, sqrt_s_hat, N, momenta.data_ptr(),
                                          _stream_ptr(self.device)), "heget_rambo")
        return momenta

    def gen_events(self, seed, n, N, mode=GEN_FIXED, a=1000.0, b=0.0, y_max=0.0, apply_cuts=False,
                   first_event=0, momenta=None, weight=None):
        if momenta is None:
            momenta = torch.empty((N, n + 2, 4), dtype=torch.float64, device=self.device)
        if weight is None:
            weight = torch.empty((N,), dtype=torch.float64, device=self.device)
        _check_dev(momenta, (N, n + 2, 4), self.device)
        _check_dev(weight, (N,), self.device)
        cfg = GenCfg(mode, int(bool(apply_cuts)), a, b, y_max)
        self._check(self._lib.heget_gen_events(self._ctx, seed, n, ctypes.byref(cfg), first_event, N,
                                               momenta.data_ptr(), weight.data_ptr(),
                                               _stream_ptr(self.device)), "heget_gen_events")
        return momenta, weight

    def amp2(self, momenta, precision=FP64, out=None, algo=ALGO_TREE):
        _check_dev(momenta, None, self.device)
        if momenta.dim() != 3 or momenta.shape[2] != 4:
            raise HegetError("momenta must be [N][n+2][4]")
        N, n = momenta.shape[0], momenta.shape[1] - 2
        if out is None:
            out = torch.empty((N,), dtype=torch.float64, device=self.device)
        _check_dev(out, (N,), self.device)
        self._check(self._lib.heget_amp2_algo(self._ctx, momenta.data_ptr(), n, precision, algo, out.data_ptr(), N,
                                              _stream_ptr(self.device)), "heget_amp2_algo")
        return out

    def amp2_sampled(self, seed, momenta, precision=FP64, first_event=0, out=None, out_hel=None):
        """One Philox-drawn helicity assignment per event: (4 * 2^n * |M(h)|^2 [N], bits [N] int32)."""
        _check_dev(momenta, None, self.device)
        if momenta.dim() != 3 or momenta.shape[2] != 4:
            raise HegetError("momenta must be [N][n+2][4]")
        N, n = momenta.shape[0], momenta.shape[1] - 2
        if out is None:
            out = torch.empty((N,), dtype=torch.float64, device=self.device)
        if out_hel is None:
            out_hel = torch.empty((N,), dtype=torch.int32, device=self.device)
        _check_dev(out, (N,), self.device)
        self._check(self._lib.heget_amp2_sampled(self._ctx, seed, first_event, momenta.data_ptr(), n, precision,
                                                 out.data_ptr(), out_hel.data_ptr(), N,
                                                 _stream_ptr(self.device)), "heget_amp2_sampled")
        return out, out_hel

    def list2(self, seed, momenta, precision=FP64, first_event=0):
        """The paper's List 2 program (thread per event, no reuse): same result as amp2_sampled."""
        _check_dev(momenta, None, self.device)
        if momenta.dim() != 3 or momenta.shape[2] != 4:
            raise HegetError("momenta must be [N][n+2][4]")
        N, n = momenta.shape[0], momenta.shape[1] - 2
        out = torch.empty((N,), dtype=torch.float64, device=self.device)
        out_hel = torch.empty((N,), dtype=torch.int32, device=self.device)
        self._check(self._lib.heget_list2(self._ctx, seed, first_event, momenta.data_ptr(), n, precision,
                                          out.data_ptr(), out_hel.data_ptr(), N, _stream_ptr(self.device)),
                    "heget_list2")
        return out, out_hel

    def list2_sum(self, momenta, precision=FP64):
        """The paper's List 2 program looped over all helicity assignments: same result as amp2."""
        _check_dev(momenta, None, self.device)
        N, n = momenta.shape[0], momenta.shape[1] - 2
        out = torch.empty((N,), dtype=torch.float64, device=self.device)
        self._check(self._lib.heget_list2_sum(self._ctx, momenta.data_ptr(), n, precision, out.data_ptr(), N,
                                              _stream_ptr(self.device)), "heget_list2_sum")
        return out

    def histogram(self, momenta, value, observable, lo, hi, nbins, hist=None):
        """Weighted histogram [underflow, nbins bins, overflow] of max pT / min Delta R / all Delta R."""
        _check_dev(momenta, None, self.device)
        N, n = momenta.shape[0], momenta.shape[1] - 2
        _check_dev(value, (N,), self.device)
        if hist is None:
            hist = torch.empty((nbins + 2,), dtype=torch.float64, device=self.device)
        _check_dev(hist, (nbins + 2,), self.device)
        self._check(self._lib.heget_histogram(self._ctx, momenta.data_ptr(), value.data_ptr(), n, N, observable,
                                              lo, hi, nbins, hist.data_ptr(), _stream_ptr(self.device)),
                    "heget_histogram")
        return hist

    def helas_wavefunction(self, fn, p, nhel, ns, precision=FP64):
        """ixxxxk / oxxxxk / vxxxxk on p[N][4] -> w[N][6][2] (cmplx w[6])."""
        _check_dev(p, None, self.device)
        if p.dim() != 2 or p.shape[1] != 4:
            raise HegetError("p must be [N][4]")
        w = torch.empty((p.shape[0], 6, 2), dtype=torch.float64, device=self.device)
        self._check(self._lib.heget_helas_wavefunction(self._ctx, fn, precision, p.data_ptr(), nhel, ns,
                                                       w.data_ptr(), p.shape[0], _stream_ptr(self.device)),
                    "heget_helas_wavefunction")
        return w

    def helas_vertex(self, fn, fi=None, fo=None, vc=None, g=0.0, precision=FP64):
        """iovxxx -> [N][2]; fvixx0 / fvoxx0 / jioxx0 -> [N][6][2]."""
        given = [t for t in (fi, fo, vc) if t is not None]
        for t in given:
            _check_dev(t, (given[0].shape[0], 6, 2), self.device)
        N = given[0].shape[0]
        out = torch.empty((N, 2) if fn == VTX_IOVXXX else (N, 6, 2), dtype=torch.float64, device=self.device)
        ptr = lambda t: t.data_ptr() if t is not None else None  # noqa: E731
        self._check(self._lib.heget_helas_vertex(self._ctx, fn, precision, ptr(fi), ptr(fo), ptr(vc), g,
                                                 out.data_ptr(), N, _stream_ptr(self.device)), "heget_helas_vertex")
        return out

    def xsec_reduce(self, amp2, weight, n, out3=None):
        _check_dev(amp2, None, self.device)
        _check_dev(weight, amp2.shape, self.device)
        if out3 is None:
            out3 = torch.empty((3,), dtype=torch.float64, device=self.device)
        _check_dev(out3, (3,), self.device)
        self._check(self._lib.heget_xsec_reduce(self._ctx, amp2.data_ptr(), weight.data_ptr(), n,
                                                amp2.shape[0], out3.data_ptr(), _stream_ptr(self.device)),
                    "heget_xsec_reduce")
        return out3

    def xsec_reduce_noalloc(self, amp2, weight, n, out3):
        """heget_xsec_reduce with its scratch in a static device array of the library: allocates nothing (the
        caller passes out3), N <= 2^24 events, calls must not overlap on the GPU."""
        _check_dev(amp2, None, self.device)
        _check_dev(weight, amp2.shape, self.device)
        _check_dev(out3, (3,), self.device)
        rc = self._lib.heget_xsec_reduce_noalloc(self._ctx, amp2.data_ptr(), weight.data_ptr(), n, amp2.shape[0],
                                                 out3.data_ptr(), _stream_ptr(self.device))
        if rc == -4:
            raise HegetError(self._lib.heget_strerror(rc).decode() + ": " + self._lib.heget_last_cuda_error(self._ctx).decode())
        self._check(rc, "heget_xsec_reduce_noalloc")
        return out3

    def xsec_host(self, momenta, weight, precision=FP64, out_amp2=None, out3=None):
        """Host tensors in, host tensors out (H2D, amp2, reduce, D2H inside the call)."""
        for t in (momenta, weight):
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
                raise HegetError("xsec_host expects contiguous float64 host tensors")
        N, n = momenta.shape[0], momenta.shape[1] - 2
        if out3 is None:
            out3 = torch.empty((3,), dtype=torch.float64)
        amp_ptr = out_amp2.data_ptr() if out_amp2 is not None else None
        self._check(self._lib.heget_xsec_host(self._ctx, momenta.data_ptr(), weight.data_ptr(), n, precision,
                                              N, amp_ptr, out3.data_ptr()), "heget_xsec_host")
        return out3

    def fma_peak(self, precision, pattern=0):
        v = ctypes.c_double()
        self._check(self._lib.heget_fma_peak_pattern(self._ctx, precision, pattern, ctypes.byref(v)),
                    "heget_fma_peak_pattern")
        return v.value

    def launch_count(self):
        return int(self._lib.heget_launch_count(self._ctx))
