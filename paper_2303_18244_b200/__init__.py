"""paper_2303_18244_b200 — B200-native tree-level matrix-element engine (arXiv:2303.18244 hot path).

Thin ctypes binding over the C-ABI library declared in include/me.h (same names, argument
marshalling only).  PyTorch supplies device memory and streams; every arithmetic step runs in the
CUDA kernels of libme_b200.so.  There is NO CPU fallback: importing works anywhere (so the build
check can run), but any call raises if the library is missing or no CUDA device is usable.
"""
import ctypes
import os

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libme_b200.so")

ME_OK, ME_EINVAL, ME_EPROCESS, ME_ENOTFILTERED, ME_EALIGN, ME_ENOMEM, ME_ECUDA, ME_ETOOLARGE = range(8)
ME_STATIC_MAX_EVENTS = 8192
ME_EPEM_MUPMUM, ME_GG_TTX, ME_GG_TTXG, ME_GG_TTXGG, ME_GG_TTXGGG = range(5)
ME_FP64, ME_MIXED, ME_FP32 = range(3)
ME_OPT_PARITY_PAIRING, ME_OPT_SHARE_CURRENTS = 0, 1
PRECISIONS = {"fp64": ME_FP64, "mixed": ME_MIXED, "fp32": ME_FP32}

EXPORTS = ("me_create", "me_destroy", "me_get_info", "me_filter_helicities", "me_set_helicities", "me_compute", "me_compute_host", "me_compute_static",
           "me_compute_helicities", "me_compute_jamps", "me_set_option", "me_select_helicity_color", "me_unweight", "me_color_matrix", "me_philox_uniform", "me_rambo",
           "me_fma_peak", "me_strerror")


class me_sm_params(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in ("mz", "wz", "aewm1", "sw2", "mt", "wt", "alpha_s")]


class me_info(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int) for k in ("npar", "ninitial", "ndiagrams", "ncomb", "ncolor", "color_denom", "avg_denom",
                                            "page", "nkernels", "namplitudes")] + \
               [("mass", ctypes.c_double * 8), ("flops_per_helicity", ctypes.c_double * 3),
                ("flops_per_event_fixed", ctypes.c_double * 3), ("flops_executed_per_helicity", ctypes.c_double * 3),
                ("flops_per_event_shared", ctypes.c_double), ("flops_executed_per_event_shared", ctypes.c_double)]


class MEError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("me status %d: %s" % (status, msg))
        self.status = status


_lib = None


def lib():
    """Load libme_b200.so (built by `python -m paper_2303_18244_b200.build`); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not built: run `python -m paper_2303_18244_b200.build` (there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, u64, dbl, cint = ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_int
        L.me_create.argtypes = [cint, ctypes.POINTER(me_sm_params), ctypes.POINTER(vp)]
        L.me_destroy.argtypes = [vp]
        L.me_get_info.argtypes = [vp, ctypes.POINTER(me_info)]
        L.me_filter_helicities.argtypes = [vp, vp, i64, ctypes.POINTER(u64), ctypes.POINTER(cint), vp]
        L.me_set_helicities.argtypes = [vp, ctypes.POINTER(u64)]
        L.me_set_option.argtypes = [vp, cint, cint]
        L.me_select_helicity_color.argtypes = [vp, vp, i64, u64, u64, vp, vp, vp]
        L.me_unweight.argtypes = [vp, vp, i64, dbl, u64, u64, dbl, ctypes.POINTER(dbl), vp, ctypes.POINTER(i64), vp]
        L.me_compute.argtypes = [vp, vp, i64, cint, vp, vp]
        L.me_compute_host.argtypes = [vp, vp, i64, cint, vp, vp]
        L.me_compute_static.argtypes = [vp, vp, i64, cint, vp, vp]
        L.me_compute_helicities.argtypes = [vp, vp, i64, cint, vp, vp, vp]
        L.me_compute_jamps.argtypes = [vp, vp, i64, cint, vp, vp]
        L.me_color_matrix.argtypes = [vp, ctypes.POINTER(dbl)]
        L.me_philox_uniform.argtypes = [u64, u64, i64, cint, vp, vp]
        L.me_rambo.argtypes = [vp, dbl, vp, i64, vp, vp, vp]
        L.me_fma_peak.argtypes = [cint, ctypes.POINTER(dbl)]
        L.me_strerror.argtypes = [cint]
        L.me_strerror.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name != "me_strerror":
                getattr(L, name).restype = cint
        _lib = L
    return _lib


def _check(status):
    if status != ME_OK:
        raise MEError(status, lib().me_strerror(status).decode())


def _stream(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


def _ptr(t, dtype=None):
    if t is None:
        return ctypes.c_void_p(0)
    import torch
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    return ctypes.c_void_p(t.data_ptr())


DEFAULT_SM = dict(mz=91.188, wz=2.441404, aewm1=132.507, sw2=0.2222, mt=173.0, wt=0.0, alpha_s=0.118)


def me_philox_uniform(seed, first_event, n, per_event, device="cuda", stream=None):
    """-> torch.float64 [n][per_event][4] uniforms in (0,1) (include/me.h me_philox_uniform)."""
    import torch
    out = torch.empty((n, per_event, 4), dtype=torch.float64, device=device)
    _check(lib().me_philox_uniform(seed, first_event, n, per_event, _ptr(out), _stream(stream)))
    return out


def me_unweight(weight, me_values, flux, seed, first_event=0, wmax=0.0, want_accept=True, stream=None):
    """-> (sum w, sum w^2, max w, accept uint8 [n] or None, n accepted)  (include/me.h me_unweight)"""
    import torch
    n = me_values.numel()
    sums = (ctypes.c_double * 3)()
    na = ctypes.c_int64(0)
    acc = torch.empty(n, dtype=torch.uint8, device=me_values.device) if want_accept else None
    _check(lib().me_unweight(_ptr(weight, torch.float64), _ptr(me_values, torch.float64), n, float(flux), seed, first_event, float(wmax),
                             sums, _ptr(acc), ctypes.byref(na), _stream(stream)))
    return sums[0], sums[1], sums[2], acc, na.value


def me_fma_peak(fp64):
    v = ctypes.c_double(0)
    _check(lib().me_fma_peak(int(bool(fp64)), ctypes.byref(v)))
    return v.value


def launches_per_pass(info, nhel, n=None, nsm=None, shared=True):
    """kernels one me_compute pass launches for `nhel` helicities: one for the single-kernel processes; for the staged process
    (info.nkernels > 1: diagram kernels + colour sum per helicity chunk of 32; the memset that clears the staging buffer in float mode
    is not a kernel of ours and is not counted).  g g -> t t~ g g with current sharing on and a batch of n events that leaves CTA slots
    of the nsm multiprocessors free: the helicity list is split over several CTAs and a second kernel sums the steps (two launches)."""
    if info.nkernels <= 1:
        if info.npar == 6 and shared and n is not None and nsm is not None:
            ctas = (n + info.page - 1) // info.page * info.page // 128 + (1 if ((n + info.page - 1) // info.page * info.page) % 128 else 0)
            if min((2 * nsm) // max(ctas, 1), nhel // 8) > 1:
                return 2
        return 1
    return info.nkernels * ((nhel + 31) // 32)


class MEContext:
    """Owns one me_ctx (include/me.h).  Methods mirror the C entry points."""

    def __init__(self, process, **sm):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2303_18244_b200 needs a CUDA device (no CPU fallback)")
        p = dict(DEFAULT_SM); p.update(sm)
        self._prm = me_sm_params(**p)
        self._h = ctypes.c_void_p(0)
        _check(lib().me_create(int(process), ctypes.byref(self._prm), ctypes.byref(self._h)))
        self.info = me_info()
        _check(lib().me_get_info(self._h, ctypes.byref(self.info)))
        self.process = int(process)

    def close(self):
        if self._h:
            lib().me_destroy(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- layout helpers (no arithmetic)
    def npages(self, n):
        return (n + self.info.page - 1) // self.info.page

    def momenta_numel(self, n):
        return self.npages(n) * self.info.npar * 4 * self.info.page

    def me_rambo(self, sqrt_s, rnd, n=None, want_weight=True, stream=None):
        """rnd [n][nfinal][4] -> (momenta AoSoA flat tensor, weight [n] or None)"""
        import torch
        n = rnd.shape[0] if n is None else n
        mom = torch.empty(self.momenta_numel(n), dtype=torch.float64, device=rnd.device)
        wt = torch.empty(n, dtype=torch.float64, device=rnd.device) if want_weight else None
        _check(lib().me_rambo(self._h, float(sqrt_s), _ptr(rnd, torch.float64), n, _ptr(mom), _ptr(wt), _stream(stream)))
        return mom, wt

    def me_filter_helicities(self, momenta, n, stream=None):
        import torch
        mask = (ctypes.c_uint64 * 2)()
        ng = ctypes.c_int(0)
        assert momenta.numel() >= self.momenta_numel(n)
        _check(lib().me_filter_helicities(self._h, _ptr(momenta, torch.float64), n, mask, ctypes.byref(ng), _stream(stream)))
        return (int(mask[0]) | (int(mask[1]) << 64)), ng.value

    def me_set_helicities(self, mask):
        m = (ctypes.c_uint64 * 2)(mask & ((1 << 64) - 1), mask >> 64)
        _check(lib().me_set_helicities(self._h, m))

    def me_set_option(self, option, value):
        _check(lib().me_set_option(self._h, int(option), int(value)))

    def me_compute(self, momenta, n, precision=ME_FP64, out=None, stream=None):
        import torch
        assert momenta.numel() >= self.momenta_numel(n)
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=momenta.device)
        _check(lib().me_compute(self._h, _ptr(momenta, torch.float64), n, int(precision), _ptr(out, torch.float64), _stream(stream)))
        return out

    def me_compute_static(self, momenta, n, precision=ME_FP64, out=None, stream=None):
        """me_compute without any allocation inside the library (include/me.h me_compute_static): pass `out` to allocate nothing here either"""
        import torch
        assert momenta.numel() >= self.momenta_numel(n)
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=momenta.device)
        _check(lib().me_compute_static(self._h, _ptr(momenta, torch.float64), n, int(precision), _ptr(out, torch.float64), _stream(stream)))
        return out

    def me_compute_helicities(self, momenta, n, precision=ME_FP64, stream=None):
        import torch
        assert momenta.numel() >= self.momenta_numel(n)
        me = torch.empty(n, dtype=torch.float64, device=momenta.device)
        mh = torch.empty((self.info.ncomb, n), dtype=torch.float64, device=momenta.device)
        _check(lib().me_compute_helicities(self._h, _ptr(momenta, torch.float64), n, int(precision), _ptr(me), _ptr(mh), _stream(stream)))
        return me, mh

    def me_select_helicity_color(self, momenta, n, seed, first_event=0, stream=None):
        """-> (ihel int32 [n], icol int32 [n]) (include/me.h me_select_helicity_color)"""
        import torch
        ihel = torch.empty(n, dtype=torch.int32, device=momenta.device)
        icol = torch.empty(n, dtype=torch.int32, device=momenta.device)
        _check(lib().me_select_helicity_color(self._h, _ptr(momenta, torch.float64), n, seed, first_event, _ptr(ihel), _ptr(icol), _stream(stream)))
        return ihel, icol

    def me_compute_jamps(self, momenta, n, ihel, stream=None):
        import torch
        out = torch.empty((self.info.ncolor, 2, n), dtype=torch.float64, device=momenta.device)
        _check(lib().me_compute_jamps(self._h, _ptr(momenta, torch.float64), n, int(ihel), _ptr(out), _stream(stream)))
        return out

    def me_color_matrix(self):
        import numpy as np
        nc = self.info.ncolor
        out = np.zeros((nc, nc))
        _check(lib().me_color_matrix(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
        return out

    def me_compute_host(self, momenta_host, n, precision=ME_FP64, stream=None, out=None):
        """End-to-end call with HOST buffers (pinned torch tensors) through the C-ABI me_compute_host: sliced H2D copies of the
        momenta overlapped with the computation, D2H copies of the MEs; returns the (pinned) host tensor after synchronising."""
        import torch
        assert not momenta_host.is_cuda and momenta_host.dtype == torch.float64 and momenta_host.is_contiguous()
        assert momenta_host.numel() >= self.momenta_numel(n)
        s = stream if stream is not None else torch.cuda.current_stream()
        if out is None:
            out = torch.empty(n, dtype=torch.float64, pin_memory=True)
        _check(lib().me_compute_host(self._h, ctypes.c_void_p(momenta_host.data_ptr()), n, int(precision), ctypes.c_void_p(out.data_ptr()), _stream(s)))
        s.synchronize()
        return out
