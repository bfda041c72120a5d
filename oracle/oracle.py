"""ORACLE binding (test infrastructure, NOT the product).

Builds oracle/me_oracle.cpp with g++ and exposes it through ctypes.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Nothing here imports the CUDA package (paper_2503_21935_b200) and nothing there imports this.

What it computes and the passages it follows are in the header of me_oracle.cpp.  The two host-side
steps below (good-helicity filter, helicity/colour selection) follow DESIGN.md readings R10/R11
(SURVEY.md 8(c) items 10-11); the paper does not describe them: "parity unpinned" against the paper.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "me_oracle.cpp")
_LIB = os.path.join(_HERE, "libme_oracle.so")
_LIB_COUNT = os.path.join(_HERE, "libme_oracle_count.so")   # same source, -DORC_COUNT (counted mode)
_LIB_QUAD = os.path.join(_HERE, "libme_oracle_quad.so")     # same source, -DORC_QUAD (113-bit scalar, libquadmath)
_lock = threading.Lock()
_lib = None
_lib_count = None
_lib_quad = None

PROC_ID = {"ee_mumu": 0, "gg_tt": 1, "gg_ttg": 2, "gg_ttgg": 3, "gg_ttggg": 4,
           "gux_taptamux": 5, "gux_taptamgux": 6, "gux_taptamggux": 7}
NGLUON = {"ee_mumu": 0, "gg_tt": 2, "gg_ttg": 3, "gg_ttgg": 4, "gg_ttggg": 5, "gux_taptamux": 1, "gux_taptamgux": 2, "gux_taptamggux": 3}
DEFAULT_PARAMS = dict(mt=173.0, wt=1.4915, mz=91.188, wz=2.441, aewm1=132.507, gf=1.16639e-5)


def build(force: bool = False) -> str:
    """Compile the oracle shared libraries (g++ -O2 -fopenmp) if missing or stale: the plain one and the
    operation-counting one (same source with -DORC_COUNT); and the quadruple-precision one (-DORC_QUAD)."""
    with _lock:
        for target, extra in ((_LIB, []), (_LIB_COUNT, ["-DORC_COUNT"]), (_LIB_QUAD, ["-DORC_QUAD"])):
            if force or not os.path.exists(target) or os.path.getmtime(target) < os.path.getmtime(_SRC):
                tmp = target + ".tmp%d" % os.getpid()
                cmd = ["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++14"] + extra + [_SRC, "-o", tmp] + (["-lquadmath"] if "-DORC_QUAD" in extra else [])
                subprocess.check_call(cmd)
                os.replace(tmp, target)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.orc_info.argtypes = [ctypes.c_int, ip, ip, ip, ip, ip]
        L.orc_counts.argtypes = [ctypes.c_int] + [ctypes.POINTER(ctypes.c_long)] * 3
        L.orc_helicity_table.argtypes = [ctypes.c_int, ctypes.c_void_p]
        L.orc_color_table.argtypes = [ctypes.c_int, ctypes.c_void_p]
        L.orc_color_matrix.argtypes = [ctypes.c_int, dp]
        L.orc_me_helicities.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_int64, ctypes.c_void_p, dp, dp, ctypes.c_int]
        L.orc_jamps.argtypes = [ctypes.c_int, dp, dp, ctypes.c_double, ctypes.c_int, ctypes.c_int, dp, dp]
        L.orc_census.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_long)]
        L.orc_brute_color.argtypes = [ctypes.c_int, dp, dp, ctypes.c_double, ctypes.c_int, dp]
        L.orc_wavefunction.argtypes = [ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp]
        L.orc_slash.argtypes = [dp, dp]
        L.orc_multichannel.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_int64, ctypes.c_void_p, dp, ctypes.c_int]
        L.orc_channel_keys.argtypes = [ctypes.c_int, ctypes.c_char_p, ctypes.c_int]
        L.orc_channel_flows.argtypes = [ctypes.c_int, ctypes.c_void_p]
        L.orc_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _params(params):
    d = dict(DEFAULT_PARAMS)
    if params:
        d.update(params)
    return np.array([d["mt"], d["wt"], d["mz"], d["wz"], d["aewm1"], d["gf"]], dtype=np.float64)


def info(process: str) -> dict:
    v = [ctypes.c_int() for _ in range(5)]
    rc = lib().orc_info(PROC_ID[process], *[ctypes.byref(x) for x in v])
    assert rc == 0
    return dict(zip(("npar", "ncomb", "ncol", "ndiag", "denom"), (x.value for x in v)))


def counts(process: str) -> dict:
    v = [ctypes.c_long() for _ in range(3)]
    assert lib().orc_counts(PROC_ID[process], *[ctypes.byref(x) for x in v]) == 0
    return dict(zip(("ntrees", "ntrie", "nsub"), (x.value for x in v)))


def helicity_table(process: str) -> np.ndarray:
    i = info(process)
    out = np.zeros((i["ncomb"], i["npar"]), dtype=np.int8)
    assert lib().orc_helicity_table(PROC_ID[process], out.ctypes.data) == 0
    return out


def color_table(process: str) -> np.ndarray:
    i = info(process)
    n = NGLUON[process]
    out = np.zeros((i["ncol"], n), dtype=np.int8)
    if n:
        assert lib().orc_color_table(PROC_ID[process], out.ctypes.data) == 0
    return out


def color_matrix(process: str) -> np.ndarray:
    i = info(process)
    out = np.zeros((i["ncol"], i["ncol"]), dtype=np.float64)
    assert lib().orc_color_matrix(PROC_ID[process], _dp(out)) == 0
    return out


def me_helicities(process, momenta, gs, params=None, mask=None, want_jamp2=False, nthreads=0):
    """Per-event per-helicity |M_h|^2 (not averaged) [nevt][ncomb] and optionally |J_c(h)|^2 [nevt][ncomb][ncol]."""
    i = info(process)
    mom = np.ascontiguousarray(momenta, dtype=np.float64)
    nevt = mom.shape[0]
    assert mom.shape == (nevt, i["npar"], 4)
    g = np.ascontiguousarray(np.broadcast_to(np.asarray(gs, dtype=np.float64), (nevt,)))
    mhel = np.zeros((nevt, i["ncomb"]), dtype=np.float64)
    j2 = np.zeros((nevt, i["ncomb"], i["ncol"]), dtype=np.float64) if want_jamp2 else None
    p = _params(params)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rc = lib().orc_me_helicities(PROC_ID[process], _dp(p), _dp(mom), _dp(g), nevt,
                                 None if m is None else m.ctypes.data, _dp(mhel),
                                 None if j2 is None else _dp(j2), int(nthreads))
    assert rc == 0
    return (mhel, j2) if want_jamp2 else mhel


def good_helicities(process, momenta, gs, params=None, nthreads=0) -> np.ndarray:
    """Reading R10: fp64, first min(nevt,16384) events; h is good iff max_e |M_h|^2 / sum_h' |M_h'|^2 > 1e-12."""
    n = min(len(momenta), 16384)
    g = np.broadcast_to(np.asarray(gs, dtype=np.float64), (len(momenta),))[:n]
    mh = me_helicities(process, momenta[:n], g, params, nthreads=nthreads)
    frac = mh / mh.sum(axis=1, keepdims=True)
    return (frac.max(axis=0) > 1e-12).astype(np.uint8)


def me(process, momenta, gs, params=None, mask=None, nthreads=0) -> np.ndarray:
    """ME[nevt] = (1/denom) sum over (good) helicities of |M_h|^2."""
    mh = me_helicities(process, momenta, gs, params, mask=mask, nthreads=nthreads)
    return mh.sum(axis=1) / info(process)["denom"]


def channel_keys(process) -> list:
    """Structural keys of the channels (= Feynman diagrams) in channel order (reading R17; see me_oracle.cpp)."""
    n = lib().orc_channel_keys(PROC_ID[process], None, 0)
    assert n > 0
    buf = ctypes.create_string_buffer(n + 1)
    assert lib().orc_channel_keys(PROC_ID[process], buf, n + 1) == n
    return buf.value.decode().split("\n")[:-1]


def channel_flows(process) -> np.ndarray:
    """allowed[ndiag][ncol] (bool): the colour flows a channel's diagram contributes to."""
    i = info(process)
    out = np.zeros((i["ndiag"], i["ncol"]), dtype=np.uint8)
    assert lib().orc_channel_flows(PROC_ID[process], out.ctypes.data) == i["ndiag"]
    return out.astype(bool)


def multichannel(process, momenta, gs, params=None, mask=None, nthreads=0) -> np.ndarray:
    """num[nevt][ndiag] = sum over (good) helicities and colour-structure terms of |A_d|^2 (reading R17); the
    single-diagram-enhancement weight of channel d is num[:, d] / num.sum(axis=1)."""
    i = info(process)
    mom = np.ascontiguousarray(momenta, dtype=np.float64)
    nevt = mom.shape[0]
    g = np.ascontiguousarray(np.broadcast_to(np.asarray(gs, dtype=np.float64), (nevt,)))
    num = np.zeros((nevt, i["ndiag"]), dtype=np.float64)
    p = _params(params)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rc = lib().orc_multichannel(PROC_ID[process], _dp(p), _dp(mom), _dp(g), nevt, None if m is None else m.ctypes.data,
                                _dp(num), int(nthreads))
    assert rc == 0
    return num


def select(process, momenta, gs, rndhel, rndcol, params=None, mask=None, nthreads=0, channel=None):
    """Reading R11.  Returns dict(me, selhel, selcol, cumhel [nevt][ncomb], cumcol [nevt][ncol]).

    helicity: scan helicities in table order, pick the first good h with r_hel * S < sum_{h'<=h} |M_h'|^2,
    fall back to the last good one; colour: weights w_c = sum_{h good} |J_c(h)|^2, same scan with r_col.
    With channel[nevt] (reading R17) the colour weights of the flows the event's channel does not contribute to
    are set to zero before the scan (fallback: the last allowed flow).
    """
    i = info(process)
    mh, j2 = me_helicities(process, momenta, gs, params, mask=mask, want_jamp2=True, nthreads=nthreads)
    nevt = mh.shape[0]
    good = np.ones(i["ncomb"], dtype=bool) if mask is None else np.asarray(mask).astype(bool)
    selhel = np.zeros(nevt, dtype=np.int32)
    selcol = np.zeros(nevt, dtype=np.int32)
    cumhel = np.zeros_like(mh)
    wcol = j2.sum(axis=1)
    allowed = None
    if channel is not None:
        allowed = channel_flows(process)[np.asarray(channel)]      # [nevt][ncol]
        wcol = np.where(allowed, wcol, 0.0)
    cumcol = np.zeros_like(wcol)
    last_good = int(np.nonzero(good)[0][-1])
    for e in range(nevt):
        tot = 0.0
        for h in range(i["ncomb"]):
            if good[h]:
                tot += mh[e, h]
            cumhel[e, h] = tot
        sel = last_good
        for h in range(i["ncomb"]):
            if good[h] and rndhel[e] * tot < cumhel[e, h]:
                sel = h
                break
        selhel[e] = sel
        totc = 0.0
        for c in range(i["ncol"]):
            totc += wcol[e, c]
            cumcol[e, c] = totc
        selc = i["ncol"] - 1 if allowed is None else int(np.nonzero(allowed[e])[0][-1])
        for c in range(i["ncol"]):
            if (allowed is None or allowed[e, c]) and rndcol[e] * totc < cumcol[e, c]:
                selc = c
                break
        selcol[e] = selc
    return dict(me=cumhel[:, -1] / i["denom"], selhel=selhel, selcol=selcol, cumhel=cumhel, cumcol=cumcol)


def jamps(process, momenta1, gs, h, ward_leg=-1, params=None, want_amps=False):
    """Colour-flow amplitudes J_sigma (complex [ncol]) of one event and helicity index h."""
    i = info(process)
    mom = np.ascontiguousarray(momenta1, dtype=np.float64).reshape(i["npar"], 4)
    out = np.zeros(2 * i["ncol"], dtype=np.float64)
    amps = np.zeros(2 * counts(process)["nsub"], dtype=np.float64) if want_amps else None
    p = _params(params)
    rc = lib().orc_jamps(PROC_ID[process], _dp(p), _dp(mom), float(gs), int(h), int(ward_leg), _dp(out),
                         None if amps is None else _dp(amps))
    assert rc == 0
    j = out[0::2] + 1j * out[1::2]
    if want_amps:
        return j, amps[0::2] + 1j * amps[1::2]
    return j


def census(process) -> dict:
    out = (ctypes.c_long * 5)()
    assert lib().orc_census(PROC_ID[process], out) == 0
    return dict(v3=out[0], v4=out[1], chain=out[2], closure=out[3], jamp_terms=out[4])


def brute_color(process, momenta1, gs, h, params=None) -> float:
    i = info(process)
    mom = np.ascontiguousarray(momenta1, dtype=np.float64).reshape(i["npar"], 4)
    out = ctypes.c_double()
    p = _params(params)
    assert lib().orc_brute_color(PROC_ID[process], _dp(p), _dp(mom), float(gs), int(h), ctypes.byref(out)) == 0
    return out.value


def wavefunction(kind: str, p, m: float, lam: int) -> np.ndarray:
    k = {"u": 0, "v": 1, "ubar": 2, "vbar": 3, "eps": 4}[kind]
    pp = np.ascontiguousarray(p, dtype=np.float64)
    out = np.zeros(8)
    lib().orc_wavefunction(k, _dp(pp), float(m), int(lam), _dp(out))
    return out[0::2] + 1j * out[1::2]


def slash(a) -> np.ndarray:
    a = np.asarray(a, dtype=np.complex128)
    a8 = np.ascontiguousarray(np.stack([a.real, a.imag], -1).reshape(-1))
    out = np.zeros(32)
    lib().orc_slash(_dp(a8), _dp(out))
    return (out[0::2] + 1j * out[1::2]).reshape(4, 4)


def count_ops(process, momenta1, gs, mask=None, params=None) -> dict:
    """Counted mode (north_star "FLOPs per ME counted by the instrumented oracle"): the arithmetic
    operations of the oracle for ONE event over the helicities of mask, from the -DORC_COUNT build of the same
    source (a double that counts its +,-,*,/ and sqrt).  flops = add + mul + div + sqrt, i.e. FMA = 2."""
    global _lib_count
    if _lib_count is None:
        build()
        L = ctypes.CDLL(_LIB_COUNT)
        dp = ctypes.POINTER(ctypes.c_double)
        L.orc_count_ops.argtypes = [ctypes.c_int, dp, dp, ctypes.c_double, ctypes.c_void_p, ctypes.POINTER(ctypes.c_long), dp]
        _lib_count = L
    i = info(process)
    mom = np.ascontiguousarray(momenta1, dtype=np.float64).reshape(i["npar"], 4)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    out = (ctypes.c_long * 4)()
    raw = ctypes.c_double()
    p = _params(params)
    rc = _lib_count.orc_count_ops(PROC_ID[process], _dp(p), _dp(mom), float(gs), None if m is None else m.ctypes.data,
                                  out, ctypes.byref(raw))
    assert rc == 0
    d = dict(add=out[0], mul=out[1], div=out[2], sqrt=out[3])
    d["flops"] = sum(d.values())
    d["me"] = raw.value / i["denom"]
    return d


def me_quad(process, momenta, gs, params=None, mask=None, nthreads=0) -> np.ndarray:
    """ME[nevt] like me(), from the quadruple-precision build of the same source (-DORC_QUAD: every amplitude operation
    in __float128, the result rounded to double at the end).  Some 50 times slower than me(): meant for the few events
    where the fp64 oracle and the fp64 CUDA path disagree beyond the tolerance, to say which of the two is off
    (tests/test_gpu_fullsize.py).  Pinned in tests/test_oracle_quad.py."""
    global _lib_quad
    if _lib_quad is None:
        build()
        L = ctypes.CDLL(_LIB_QUAD)
        dp = ctypes.POINTER(ctypes.c_double)
        L.orc_me_helicities.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_int64, ctypes.c_void_p, dp, dp, ctypes.c_int]
        _lib_quad = L
    i = info(process)
    mom = np.ascontiguousarray(momenta, dtype=np.float64)
    nevt = mom.shape[0]
    assert mom.shape == (nevt, i["npar"], 4)
    g = np.ascontiguousarray(np.broadcast_to(np.asarray(gs, dtype=np.float64), (nevt,)))
    mhel = np.zeros((nevt, i["ncomb"]), dtype=np.float64)
    p = _params(params)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rc = _lib_quad.orc_me_helicities(PROC_ID[process], _dp(p), _dp(mom), _dp(g), nevt, None if m is None else m.ctypes.data,
                                     _dp(mhel), None, int(nthreads))
    assert rc == 0
    return mhel.sum(axis=1) / i["denom"]


def num_threads() -> int:
    return lib().orc_num_threads()
