"""Thin Python binding of libmg5b200.so (include/mg5b200.h): argument marshalling only.

PyTorch supplies device memory and streams; every step of the hot path runs in the library's CUDA kernels.
There is no CPU fallback: importing works without a GPU (so the C ABI can be inspected), but every compute call
needs a CUDA device and raises otherwise.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmg5b200.so")

MG_EE_MUMU, MG_GG_TT, MG_GG_TTG, MG_GG_TTGG, MG_GG_TTGGG = 1, 2, 3, 4, 5
MG_UU_EE, MG_UU_EEG, MG_UU_EEGG, MG_UU_EEGGG = 6, 7, 8, 9
MG_FP64, MG_FP32, MG_MIXED, MG_FP32_ALL = 0, 1, 2, 3
MG_LAYOUT_AOS, MG_LAYOUT_AOSOA, MG_LAYOUT_SOA = 0, 1, 2
MG_AOSOA_V = 32
MG_NOALLOC_SCRATCH_BYTES = 16 << 20
MG_OK, MG_EINVAL, MG_ENOTFILTERED, MG_ECUDA, MG_ENOMEM = 0, -1, -2, -3, -4

EXPORTS = ["mg_create", "mg_destroy", "mg_get_info", "mg_sample_rambo", "mg_sample_uniforms", "mg_filter_helicities",
           "mg_set_good_helicities", "mg_compute", "mg_compute_multichannel", "mg_compute_noalloc", "mg_compute_host", "mg_get_last_details", "mg_measure_fma_peak", "mg_measure_fp64_pipes", "mg_launch_count", "mg_enable_kernel_timing",
           "mg_kernel_time_ms", "mg_strerror"]


class mg_sm_params(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("MZ", "WZ", "MT", "WT", "aEWM1", "Gf", "alpha_s")]


class mg_info(C.Structure):
    _fields_ = [("npar", C.c_int), ("ndiag", C.c_int), ("namp", C.c_int), ("ncolor", C.c_int), ("ncomb", C.c_int),
                ("ngood", C.c_int), ("denom", C.c_int), ("mass", C.c_double * 8), ("flops_per_event", C.c_longlong),
                ("flops_per_event_canonical", C.c_longlong), ("nchannel", C.c_int)]


class MGError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("mg5b200 error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load the C-ABI library (fails loudly if it has not been built: run __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libmg5b200.so is missing: build it with `python -m paper_2507_21039_b200.build`")
        L = C.CDLL(LIB_PATH)
        vp, dp, ip, ull = C.c_void_p, C.c_void_p, C.c_void_p, C.c_ulonglong
        L.mg_create.argtypes = [C.POINTER(vp), C.c_int, C.POINTER(mg_sm_params), C.c_int, C.c_int]
        L.mg_destroy.argtypes = [vp]
        L.mg_get_info.argtypes = [vp, C.POINTER(mg_info)]
        L.mg_sample_rambo.argtypes = [vp, ull, ull, C.c_int, C.c_double, C.c_int, dp, dp, vp]
        L.mg_sample_uniforms.argtypes = [vp, ull, ull, C.c_int, dp, dp, vp]
        L.mg_filter_helicities.argtypes = [vp, dp, dp, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int), C.c_char_p, vp]
        L.mg_set_good_helicities.argtypes = [vp, C.c_char_p, vp]
        L.mg_compute.argtypes = [vp, dp, dp, dp, dp, C.c_int, C.c_int, dp, ip, ip, vp]
        L.mg_compute_multichannel.argtypes = [vp, dp, dp, dp, dp, ip, C.c_int, C.c_int, dp, ip, ip, dp, dp, vp]
        L.mg_compute_noalloc.argtypes = [vp, dp, dp, dp, dp, C.c_int, C.c_int, dp, ip, ip, vp]
        L.mg_compute_host.argtypes = [vp, dp, dp, dp, dp, C.c_int, C.c_int, dp, ip, ip, vp]
        L.mg_get_last_details.argtypes = [vp, C.c_int, dp, dp, vp]
        L.mg_measure_fma_peak.argtypes = [vp, C.c_int, C.c_double, C.POINTER(C.c_double)]
        L.mg_measure_fp64_pipes.argtypes = [vp, C.c_int, C.c_double, C.POINTER(C.c_double)]
        L.mg_launch_count.argtypes = [vp]
        L.mg_launch_count.restype = C.c_longlong
        L.mg_enable_kernel_timing.argtypes = [vp, C.c_int]
        L.mg_kernel_time_ms.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.mg_strerror.argtypes = [C.c_int]
        L.mg_strerror.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("mg_launch_count", "mg_strerror"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(code):
    if code != 0:
        raise MGError(code, lib().mg_strerror(code).decode())


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Context:
    """mg_ctx wrapper.  Tensors are torch CUDA tensors (float64 / int32) owned by the caller."""

    def __init__(self, process, sm_params, precision=MG_FP64, device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("mg5b200 needs a CUDA device (there is no CPU fallback)")
        self._h = C.c_void_p()
        self.sm = mg_sm_params(*sm_params)
        self.device = device
        torch.cuda.set_device(device)
        _check(lib().mg_create(C.byref(self._h), process, C.byref(self.sm), precision, device))
        self.process, self.precision = process, precision
        self.info = self.get_info()

    def close(self):
        if self._h:
            lib().mg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def get_info(self):
        i = mg_info()
        _check(lib().mg_get_info(self._h, C.byref(i)))
        return i

    def mom_shape(self, nevt, layout):
        npar = self.info.npar
        return (nevt, npar, 4) if layout == MG_LAYOUT_AOS else (nevt // MG_AOSOA_V, npar, 4, MG_AOSOA_V)

    def sample_rambo(self, seed, first_event, nevt, sqrt_s, layout=MG_LAYOUT_AOS, momenta=None, weight=None, want_weight=True):
        import torch
        dev = torch.device("cuda", self.device)
        if momenta is None:
            momenta = torch.empty(self.mom_shape(nevt, layout), dtype=torch.float64, device=dev)
        if weight is None and want_weight:
            weight = torch.empty(nevt, dtype=torch.float64, device=dev)
        _check(lib().mg_sample_rambo(self._h, seed, first_event, nevt, sqrt_s, layout, _ptr(momenta), _ptr(weight), _stream()))
        return momenta, weight

    def sample_uniforms(self, seed, first_event, nevt, rnd_hel=None, rnd_col=None):
        import torch
        dev = torch.device("cuda", self.device)
        if rnd_hel is None:
            rnd_hel = torch.empty(nevt, dtype=torch.float64, device=dev)
        if rnd_col is None:
            rnd_col = torch.empty(nevt, dtype=torch.float64, device=dev)
        _check(lib().mg_sample_uniforms(self._h, seed, first_event, nevt, _ptr(rnd_hel), _ptr(rnd_col), _stream()))
        return rnd_hel, rnd_col

    def filter_helicities(self, momenta, nevt, layout=MG_LAYOUT_AOS, gs=None, rel_threshold=0.0):
        ngood = C.c_int(0)
        buf = C.create_string_buffer(self.info.ncomb)
        _check(lib().mg_filter_helicities(self._h, _ptr(momenta), _ptr(gs), nevt, layout, rel_threshold, C.byref(ngood), buf, _stream()))
        self.info = self.get_info()
        return ngood.value, bytes(buf.raw)

    def set_good_helicities(self, mask):
        """Install a good-helicity mask (bytes of 0/1, length ncomb), e.g. the union over ranks."""
        mask = bytes(mask)
        assert len(mask) == self.info.ncomb
        _check(lib().mg_set_good_helicities(self._h, mask, _stream()))
        self.info = self.get_info()
        return self.info.ngood

    def compute(self, momenta, nevt, layout=MG_LAYOUT_AOS, gs=None, rnd_hel=None, rnd_col=None, me=None, sel_hel=None, sel_col=None):
        import torch
        dev = torch.device("cuda", self.device)
        if me is None:
            me = torch.empty(nevt, dtype=torch.float64, device=dev)
        if rnd_hel is not None and sel_hel is None:
            sel_hel = torch.empty(nevt, dtype=torch.int32, device=dev)
        if rnd_col is not None and sel_col is None:
            sel_col = torch.empty(nevt, dtype=torch.int32, device=dev)
        _check(lib().mg_compute(self._h, _ptr(momenta), _ptr(gs), _ptr(rnd_hel), _ptr(rnd_col), nevt, layout, _ptr(me),
                                _ptr(sel_hel), _ptr(sel_col), _stream()))
        return me, sel_hel, sel_col

    def compute_multichannel(self, momenta, nevt, channel, layout=MG_LAYOUT_AOS, gs=None, rnd_hel=None, rnd_col=None):
        """mg_compute_multichannel: (me, sel_hel, sel_col, numerator, denominator); channel = int32 tensor, one entry per 32 events."""
        import torch
        dev = torch.device("cuda", self.device)
        me, num, den = (torch.empty(nevt, dtype=torch.float64, device=dev) for _ in range(3))
        sel_hel = torch.empty(nevt, dtype=torch.int32, device=dev) if rnd_hel is not None else None
        sel_col = torch.empty(nevt, dtype=torch.int32, device=dev) if rnd_col is not None else None
        _check(lib().mg_compute_multichannel(self._h, _ptr(momenta), _ptr(gs), _ptr(rnd_hel), _ptr(rnd_col), _ptr(channel), nevt, layout,
                                             _ptr(me), _ptr(sel_hel), _ptr(sel_col), _ptr(num), _ptr(den), _stream()))
        return me, sel_hel, sel_col, num, den

    def compute_noalloc(self, momenta, nevt, me, layout=MG_LAYOUT_AOS, gs=None, rnd_hel=None, rnd_col=None, sel_hel=None, sel_col=None):
        """mg_compute_noalloc: as compute(), scratch in the library's static device array; the caller passes every output."""
        _check(lib().mg_compute_noalloc(self._h, _ptr(momenta), _ptr(gs), _ptr(rnd_hel), _ptr(rnd_col), nevt, layout, _ptr(me),
                                        _ptr(sel_hel), _ptr(sel_col), _stream()))
        return me, sel_hel, sel_col

    def noalloc_max_events(self):
        """Largest nevt mg_compute_noalloc accepts for this process (the formula of mg5b200.h)."""
        i = self.info
        f32 = self.precision in (MG_FP32, MG_FP32_ALL)      # rows of colour-flow partial sums per event (see mg5b200.h)
        w = {MG_GG_TTGG: 2, MG_GG_TTGGG: 4}.get(self.process, 1) if f32 else 1
        return (MG_NOALLOC_SCRATCH_BYTES - 256) // (8 * (i.ncomb + w * i.ncolor))

    def compute_host(self, momenta, nevt, layout=MG_LAYOUT_AOS, gs=None, rnd_hel=None, rnd_col=None, me=None, sel_hel=None, sel_col=None):
        """Host-buffer variant: all tensors are CPU tensors (pinned recommended); returns when the results are on the host."""
        import torch
        if me is None:
            me = torch.empty(nevt, dtype=torch.float64).pin_memory()
        if rnd_hel is not None and sel_hel is None:
            sel_hel = torch.empty(nevt, dtype=torch.int32).pin_memory()
        if rnd_col is not None and sel_col is None:
            sel_col = torch.empty(nevt, dtype=torch.int32).pin_memory()
        _check(lib().mg_compute_host(self._h, _ptr(momenta), _ptr(gs), _ptr(rnd_hel), _ptr(rnd_col), nevt, layout, _ptr(me),
                                     _ptr(sel_hel), _ptr(sel_col), _stream()))
        return me, sel_hel, sel_col

    def last_details(self, nevt):
        import torch
        dev = torch.device("cuda", self.device)
        mh2 = torch.empty((nevt, self.info.ncomb), dtype=torch.float64, device=dev)
        wcol = torch.empty((nevt, self.info.ncolor), dtype=torch.float64, device=dev)
        _check(lib().mg_get_last_details(self._h, nevt, _ptr(mh2), _ptr(wcol), _stream()))
        return mh2, wcol

    def measure_fma_peak(self, precision=MG_FP64, millis=50.0):
        out = C.c_double(0)
        _check(lib().mg_measure_fma_peak(self._h, precision, millis, C.byref(out)))
        return out.value

    def measure_fp64_pipes(self, mode, millis=30.0):
        """(plain-FMA TFLOP/s, tensor TFLOP/s, ms per iteration) of FP64 pipe microbenchmark `mode` (see mg5b200.h)."""
        out = (C.c_double * 3)()
        _check(lib().mg_measure_fp64_pipes(self._h, mode, millis, out))
        return out[0], out[1], out[2]

    def enable_kernel_timing(self, on=True):
        _check(lib().mg_enable_kernel_timing(self._h, 1 if on else 0))

    def kernel_time_ms(self):
        tot, n = C.c_double(0), C.c_longlong(0)
        _check(lib().mg_kernel_time_ms(self._h, C.byref(tot), C.byref(n)))
        return tot.value, n.value

    def launch_count(self):
        return int(lib().mg_launch_count(self._h))
