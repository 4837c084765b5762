"""ctypes front end of oracle/cdmt_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It imports nothing from paper_1607_00909_b200 (the CUDA path)
and the CUDA path imports nothing from here.

All arithmetic of the method lives in the C file (double precision, Algorithm 1 order,
PAPER.md:85-111); this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cdmt_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_cdmt.so")

IN_CF32, IN_CI8 = 0, 1
REF_CHANNEL, REF_SUBBAND = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("nsub", C.c_int), ("fcen_mhz", C.POINTER(C.c_double)), ("bw_mhz", C.c_double),
                ("nfft", C.c_int), ("noverlap", C.c_int), ("nchan", C.c_int), ("ndec", C.c_int),
                ("ndm", C.c_int), ("dm", C.POINTER(C.c_double)), ("in_dtype", C.c_int),
                ("chirp_ref", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_fft.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_fft.restype = C.c_int
        L.oracle_chirp_phase_cycles.argtypes = [C.c_double] * 3
        L.oracle_chirp_phase_cycles.restype = C.c_double
        L.oracle_sweep_seconds.argtypes = [C.c_double] * 3
        L.oracle_sweep_seconds.restype = C.c_double
        L.oracle_num_threads.restype = C.c_int
        L.oracle_sizes.argtypes = [C.POINTER(_Params), C.c_long] + [C.POINTER(C.c_int)] * 4
        L.oracle_block_spectrum.argtypes = [C.c_void_p, C.c_int, C.c_long, C.c_int, C.c_void_p]
        L.oracle_transfer_function.argtypes = [C.POINTER(_Params), C.c_double, C.c_int, C.c_double, C.c_void_p]
        L.oracle_transfer_function.restype = None
        L.oracle_unit.argtypes = [C.POINTER(_Params), C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_units.argtypes = [C.POINTER(_Params), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_run.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_long, C.c_void_p, C.c_void_p]
        L.oracle_channel_timeseries.argtypes = [C.POINTER(_Params), C.c_int, C.c_int, C.c_double,
                                                C.c_void_p, C.c_void_p]
        L.oracle_redigitize.argtypes = [C.c_void_p] + [C.c_long] * 4 + [C.c_double] * 2 + [C.c_void_p] * 6
        L.oracle_incoherent.argtypes = [C.c_void_p, C.c_long, C.c_long, C.c_void_p, C.c_double, C.c_long,
                                        C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_long), C.POINTER(C.c_long)]
        L.oracle_quantize.argtypes = [C.c_void_p] + [C.c_long] * 3 + [C.c_void_p] * 3
        _lib = L
    return _lib


class Params:
    """Owns the numpy arrays a C oracle_params points into."""

    def __init__(self, nsub, fcen_mhz, bw_mhz, nfft, noverlap, nchan, ndec, dm,
                 in_dtype=IN_CF32, chirp_ref=REF_CHANNEL):
        self.fcen = np.ascontiguousarray(fcen_mhz, dtype=np.float64).reshape(-1)
        self.dm = np.ascontiguousarray(dm, dtype=np.float64).reshape(-1)
        assert self.fcen.size == nsub
        self.nsub, self.bw_mhz = int(nsub), float(bw_mhz)
        self.nfft, self.noverlap, self.nchan, self.ndec = int(nfft), int(noverlap), int(nchan), int(ndec)
        self.ndm = int(self.dm.size)
        self.in_dtype, self.chirp_ref = int(in_dtype), int(chirp_ref)
        self.c = _Params(self.nsub, self.fcen.ctypes.data_as(C.POINTER(C.c_double)), self.bw_mhz,
                         self.nfft, self.noverlap, self.nchan, self.ndec, self.ndm,
                         self.dm.ctypes.data_as(C.POINTER(C.c_double)), self.in_dtype, self.chirp_ref)

    def sizes(self, nsamp):
        nb, m, h, vd = C.c_int(), C.c_int(), C.c_int(), C.c_int()
        rc = lib().oracle_sizes(C.byref(self.c), int(nsamp), C.byref(nb), C.byref(m), C.byref(h), C.byref(vd))
        if rc:
            raise ValueError("oracle_sizes: invalid parameters")
        return nb.value, m.value, h.value, vd.value


def _check_input(p: Params, x: np.ndarray) -> np.ndarray:
    if p.in_dtype == IN_CI8:
        assert x.dtype == np.int8 and x.shape[-1] == 2
    else:
        if x.dtype == np.complex64:
            x = x.view(np.float32).reshape(x.shape + (2,))
        assert x.dtype == np.float32 and x.shape[-1] == 2
    return np.ascontiguousarray(x)


def num_threads() -> int:
    return lib().oracle_num_threads()


def fft(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    rc = lib().oracle_fft(x.size, sign, x.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle_fft rc=%d" % rc)
    return out


def chirp_phase_cycles(dm, f0_mhz, f_off_mhz) -> float:
    return lib().oracle_chirp_phase_cycles(float(dm), float(f0_mhz), float(f_off_mhz))


def sweep_seconds(fcen_mhz, bw_mhz, dm) -> float:
    return lib().oracle_sweep_seconds(float(fcen_mhz), float(bw_mhz), float(dm))


def transfer_function(p: Params, fcen_mhz: float, c: int, dm: float) -> np.ndarray:
    H = np.empty(p.nfft // p.nchan, dtype=np.complex128)
    lib().oracle_transfer_function(C.byref(p.c), float(fcen_mhz), int(c), float(dm), H.ctypes.data)
    return H


def block_spectrum(p: Params, xpol: np.ndarray, first: int = 0) -> np.ndarray:
    """xpol: one polarisation, [T] complex64 or [T][2] int8. Returns the shifted spectrum Xs[N]."""
    xpol = _check_input(p, xpol)
    Xs = np.empty(p.nfft, dtype=np.complex128)
    rc = lib().oracle_block_spectrum(xpol.ctypes.data, p.in_dtype, int(first), p.nfft, Xs.ctypes.data)
    if rc:
        raise RuntimeError("oracle_block_spectrum rc=%d" % rc)
    return Xs


def channel_timeseries(p: Params, s: int, c: int, dm: float, xpol_block: np.ndarray) -> np.ndarray:
    xpol_block = _check_input(p, xpol_block)
    y = np.empty(p.nfft // p.nchan, dtype=np.complex128)
    rc = lib().oracle_channel_timeseries(C.byref(p.c), int(s), int(c), float(dm),
                                         xpol_block.ctypes.data, y.ctypes.data)
    if rc:
        raise RuntimeError("oracle_channel_timeseries rc=%d" % rc)
    return y


def units(p: Params, unit_s, xblocks: np.ndarray) -> np.ndarray:
    """xblocks [nunits][2][N] -> [nunits][ndm][Vd][C] float64, channels ASCENDING."""
    xblocks = _check_input(p, xblocks)
    nun = xblocks.shape[0]
    assert xblocks.shape[1] == 2 and xblocks.shape[2] == p.nfft
    us = np.ascontiguousarray(unit_s, dtype=np.int32)
    assert us.size == nun
    M = p.nfft // p.nchan
    vd = (M - p.noverlap // p.nchan) // p.ndec
    out = np.empty((nun, p.ndm, vd, p.nchan), dtype=np.float64)
    rc = lib().oracle_units(C.byref(p.c), nun, us.ctypes.data, xblocks.ctypes.data, out.ctypes.data)
    if rc:
        raise RuntimeError("oracle_units rc=%d" % rc)
    return out


def run(p: Params, x: np.ndarray, want64: bool = False):
    """x [nsub][2][T] -> filterbanks [ndm][nblock*Vd][nsub*nchan] float32 (and float64)."""
    x = _check_input(p, x)
    assert x.shape[0] == p.nsub and x.shape[1] == 2
    T = x.shape[2]
    nb, m, h, vd = p.sizes(T)
    shape = (p.ndm, nb * vd, p.nsub * p.nchan)
    out = np.empty(shape, dtype=np.float32)
    out64 = np.empty(shape, dtype=np.float64) if want64 else None
    rc = lib().oracle_run(C.byref(p.c), x.ctypes.data, T, out.ctypes.data,
                          out64.ctypes.data if want64 else None)
    if rc:
        raise RuntimeError("oracle_run rc=%d" % rc)
    return (out, out64) if want64 else out


QMEAN, QSTD = 64.0, 16.0   # reading Q22: code mean and standard deviation of a redigitised channel


def redigitize(fb: np.ndarray, nblock: int, qmean: float = QMEAN, qstd: float = QSTD) -> dict:
    """Alg. 1 l.104-106 on one batch: fb [ndm][nblock*vd][nch] float32 ->
    dict(segsum [ndm][nblock][nch][2], mean, std [ndm][nch] float64, offset, scale float32, codes uint8)."""
    fb = np.ascontiguousarray(fb, dtype=np.float32)
    ndm, nt, nch = fb.shape
    assert nt % nblock == 0
    vd = nt // nblock
    r = dict(segsum=np.empty((ndm, nblock, nch, 2)), mean=np.empty((ndm, nch)), std=np.empty((ndm, nch)),
             offset=np.empty((ndm, nch), np.float32), scale=np.empty((ndm, nch), np.float32),
             codes=np.empty((ndm, nt, nch), np.uint8))
    rc = lib().oracle_redigitize(fb.ctypes.data, ndm, nblock, vd, nch, float(qmean), float(qstd),
                                 *[r[k].ctypes.data for k in ("segsum", "mean", "std", "offset", "scale", "codes")])
    if rc:
        raise ValueError("oracle_redigitize rc=%d" % rc)
    return r


def quantize(fb: np.ndarray, offset: np.ndarray, scale: np.ndarray) -> np.ndarray:
    """The float32 decision of l.106 with given per-(DM, channel) offset and scale."""
    fb = np.ascontiguousarray(fb, dtype=np.float32)
    ndm, nt, nch = fb.shape
    offset = np.ascontiguousarray(offset, dtype=np.float32).reshape(ndm, nch)
    scale = np.ascontiguousarray(scale, dtype=np.float32).reshape(ndm, nch)
    codes = np.empty((ndm, nt, nch), np.uint8)
    rc = lib().oracle_quantize(fb.ctypes.data, ndm, nt, nch, offset.ctypes.data, scale.ctypes.data, codes.ctypes.data)
    if rc:
        raise ValueError("oracle_quantize rc=%d" % rc)
    return codes


def channel_frequencies(p: Params) -> np.ndarray:
    """Centre frequencies (MHz) of the filterbank channels in OUTPUT order (descending)."""
    c = np.arange(p.nchan)
    f = (p.fcen[:, None] + (c[None, :] + 0.5 - p.nchan / 2) * p.bw_mhz / p.nchan).reshape(-1)
    return np.ascontiguousarray(f[::-1])


def incoherent(fb: np.ndarray, fch: np.ndarray, tsamp: float, ddm, want_ts: bool = True) -> dict:
    """Brute-force incoherent dedispersion of one filterbank fb [nt][nch] over fine DM offsets ddm
    (PAPER.md:141).  Returns dict(shifts [nfine][nch] int32, smin, range, ts [nfine][nt-range] float32)."""
    fb = np.ascontiguousarray(fb, dtype=np.float32)
    nt, nch = fb.shape
    fch = np.ascontiguousarray(fch, dtype=np.float64)
    ddm = np.ascontiguousarray(ddm, dtype=np.float64).reshape(-1)
    assert fch.size == nch
    shifts = np.empty((ddm.size, nch), np.int32)
    rng, smin = C.c_long(), C.c_long()
    rc = lib().oracle_incoherent(fb.ctypes.data, nt, nch, fch.ctypes.data, float(tsamp), ddm.size, ddm.ctypes.data,
                                 shifts.ctypes.data, None, C.byref(rng), C.byref(smin))
    if rc:
        raise ValueError("oracle_incoherent rc=%d" % rc)
    out = dict(shifts=shifts, smin=smin.value, range=rng.value, ts=None)
    if want_ts:
        ts = np.empty((ddm.size, nt - rng.value), np.float32)
        rc = lib().oracle_incoherent(fb.ctypes.data, nt, nch, fch.ctypes.data, float(tsamp), ddm.size, ddm.ctypes.data,
                                     shifts.ctypes.data, ts.ctypes.data, None, None)
        if rc:
            raise ValueError("oracle_incoherent rc=%d" % rc)
        out["ts"] = ts
    return out
