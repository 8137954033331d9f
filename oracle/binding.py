"""ctypes binding of oracle/libmg_oracle.so -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
Every function takes/returns numpy arrays in host memory; nothing here touches the CUDA path.
"""
import ctypes as C
import os

import numpy as np

from . import build_oracle

_lib = None

# SM inputs of BASELINE.json configs: MZ, WZ, MT, WT, 1/alpha_EW, G_F, alpha_s
SM_DEFAULT = (91.188, 2.441404, 173.0, 1.4915, 132.507, 1.16639e-5, 0.118)


def lib():
    global _lib
    if _lib is None:
        path = build_oracle.build()
        _lib = C.CDLL(path)
        _lib.orc_rambo_from_uniforms.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t))


def _sm(sm):
    return np.ascontiguousarray(np.array(sm if sm is not None else SM_DEFAULT, dtype=np.float64))


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(np.array(ctr, dtype=np.uint32))
    key = np.ascontiguousarray(np.array(key, dtype=np.uint32))
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(ctr, C.c_uint32), _p(key, C.c_uint32), _p(out, C.c_uint32))
    return out


def uniforms(seed, first_event, nevt, block, purpose):
    out = np.zeros((nevt, 2), dtype=np.float64)
    lib().orc_uniforms(C.c_uint64(seed), C.c_uint64(first_event), C.c_int(nevt), C.c_uint32(block), C.c_uint32(purpose), _p(out))
    return out


def rambo(seed, first_event, nevt, masses, sqrt_s):
    masses = np.ascontiguousarray(np.array(masses, dtype=np.float64))
    nf = len(masses)
    p = np.zeros((nevt, nf + 2, 4), dtype=np.float64)
    w = np.zeros(nevt, dtype=np.float64)
    lib().orc_rambo(C.c_uint64(seed), C.c_uint64(first_event), C.c_int(nevt), C.c_int(nf), _p(masses), C.c_double(sqrt_s), _p(p), _p(w))
    return p, w


def rambo_from_uniforms(r, masses, sqrt_s):
    r = np.ascontiguousarray(np.array(r, dtype=np.float64).ravel())
    masses = np.ascontiguousarray(np.array(masses, dtype=np.float64))
    nf = len(masses)
    p = np.zeros((nf + 2, 4), dtype=np.float64)
    w = lib().orc_rambo_from_uniforms(_p(r), C.c_int(nf), _p(masses), C.c_double(sqrt_s), _p(p))
    return p, w


def sm_derive(sm=None):
    out = np.zeros(8, dtype=np.float64)
    lib().orc_sm_derive(_p(_sm(sm)), _p(out))
    return dict(zip(["MW", "sw2", "ee", "gs", "gLZ", "gRZ", "gLA", "gRA"], out.tolist()))


def info(proc):
    out = np.zeros(8, dtype=np.int32)
    rc = lib().orc_info(C.c_int(proc), _p(out, C.c_int))
    assert rc == 0
    return dict(zip(["npar", "ndiag", "namp", "ncolor", "ncomb", "denom", "ntrees"], out.tolist()))


def colour_matrix(proc, full=True):
    nc = info(proc)["ncolor"]
    out = np.zeros((nc, nc), dtype=np.float64)
    rc = lib().orc_colour_matrix(C.c_int(proc), C.c_int(1 if full else 0), _p(out))
    assert rc == 0
    return out


def flows(proc):
    i = info(proc)
    ng = i["npar"] - 2
    out = np.zeros((i["ncolor"], ng), dtype=np.int32)
    rc = lib().orc_flows(C.c_int(proc), _p(out, C.c_int))
    assert rc == 0
    return out


def wavefunction(kind, p, m, lam):
    """kind: 'u','v','ubar','vbar','eps' -> complex[4]"""
    k = {"u": 0, "v": 1, "ubar": 2, "vbar": 3, "eps": 4}[kind]
    p = np.ascontiguousarray(np.array(p, dtype=np.float64))
    out = np.zeros(8, dtype=np.float64)
    lib().orc_wavefunction(C.c_int(k), _p(p), C.c_double(m), C.c_int(lam), _p(out))
    return out[0::2] + 1j * out[1::2]


def matrix_elements(proc, momenta, sm=None, gs=None, good=None, uncached=False, long_double=False):
    """momenta [nevt][npar][4] -> (me[nevt], mh2[nevt][ncomb], wcol[nevt][ncolor])"""
    i = info(proc)
    momenta = np.ascontiguousarray(momenta, dtype=np.float64)
    nevt = momenta.shape[0]
    assert momenta.shape[1:] == (i["npar"], 4)
    me = np.zeros(nevt)
    mh2 = np.zeros((nevt, i["ncomb"]))
    wcol = np.zeros((nevt, i["ncolor"]))
    gsp = None if gs is None else _p(np.ascontiguousarray(gs, dtype=np.float64))
    goodp = None
    if good is not None:
        good = np.ascontiguousarray(good, dtype=np.uint8)
        goodp = _p(good, C.c_ubyte)
    flags = (1 if uncached else 0) | (2 if long_double else 0)
    rc = lib().orc_matrix_elements(C.c_int(proc), _p(_sm(sm)), _p(momenta), gsp, C.c_int(nevt), goodp, C.c_int(flags), _p(me), _p(mh2), _p(wcol))
    assert rc == 0
    return me, mh2, wcol


def jamp(proc, p, h, sm=None, ward_gluon_leg=-1, uncached=False):
    i = info(proc)
    p = np.ascontiguousarray(p, dtype=np.float64)
    out = np.zeros(2 * i["ncolor"])
    scale = C.c_double(0)
    rc = lib().orc_jamp(C.c_int(proc), _p(_sm(sm)), _p(p), C.c_int(h), C.c_int(ward_gluon_leg), C.c_int(1 if uncached else 0), _p(out), C.byref(scale))
    assert rc == 0
    return out[0::2] + 1j * out[1::2], scale.value


def brute_colour(proc, p, h, sm=None):
    p = np.ascontiguousarray(p, dtype=np.float64)
    out = C.c_double(0)
    rc = lib().orc_brute_colour(C.c_int(proc), _p(_sm(sm)), _p(p), C.c_int(h), C.byref(out))
    assert rc == 0
    return out.value


def filter_helicities(mh2, rel_threshold=0.0):
    mh2 = np.ascontiguousarray(mh2, dtype=np.float64)
    nevt, ncomb = mh2.shape
    good = np.zeros(ncomb, dtype=np.uint8)
    lib().orc_filter(_p(mh2), C.c_int(nevt), C.c_int(ncomb), C.c_double(rel_threshold), _p(good, C.c_ubyte))
    return good


def select(rnd, w, mask=None):
    rnd = np.ascontiguousarray(rnd, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    nevt, n = w.shape
    out = np.zeros(nevt, dtype=np.int32)
    maskp = None
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        maskp = _p(mask, C.c_ubyte)
    lib().orc_select(_p(rnd), _p(w), C.c_int(nevt), C.c_int(n), maskp, _p(out, C.c_int))
    return out


def num_threads():
    return lib().orc_num_threads()


def channels(proc):
    """Names of the integration channels (diagrams without four-gluon vertices) in channel order (channel id = index + 1)."""
    n = lib().orc_channels(C.c_int(proc), None)
    assert n > 0
    buf = C.create_string_buffer(32 * n)
    lib().orc_channels(C.c_int(proc), buf)
    return [buf.raw[32 * k:32 * k + 32].split(b"\0")[0].decode() for k in range(n)]


def channel_flows(proc):
    """allowed[nchan][ncolor] (uint8): the colour flows the channel's diagram contributes to."""
    n, nc = lib().orc_channels(C.c_int(proc), None), info(proc)["ncolor"]
    out = np.zeros((n, nc), dtype=np.uint8)
    assert lib().orc_channel_flows(C.c_int(proc), _p(out, C.c_ubyte)) == 0
    return out


def channel_sums(proc, momenta, sm=None, gs=None, good=None):
    """chan2[nevt][nchan]: helicity-summed |A_k|^2 of every channel's diagram."""
    p = np.ascontiguousarray(momenta, dtype=np.float64)
    nevt = p.shape[0]
    n = lib().orc_channels(C.c_int(proc), None)
    out = np.zeros((nevt, n))
    gsp = None if gs is None else _p(np.ascontiguousarray(gs, dtype=np.float64))
    goodp = None if good is None else _p(np.ascontiguousarray(good, dtype=np.uint8), C.c_ubyte)
    assert lib().orc_channel_sums(C.c_int(proc), _p(_sm(sm)), _p(p), gsp, C.c_int(nevt), goodp, _p(out)) == 0
    return out


def count_flops(proc, p, sm=None):
    """(arithmetic operations, ME) of ONE event evaluated by the oracle on its counting scalar (SURVEY.md 8(d) cross-check)."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    ops, me = C.c_longlong(0), C.c_double(0)
    assert lib().orc_count_flops(C.c_int(proc), _p(_sm(sm)), _p(p), C.byref(ops), C.byref(me)) == 0
    return ops.value, me.value
