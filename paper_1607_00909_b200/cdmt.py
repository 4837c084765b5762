"""Thin ctypes binding of libcdmt.so (include/cdmt.h): argument marshalling only.

Every function has the name of the C entry point it calls.  Device buffers are torch CUDA
tensors (torch is used for device memory and streams only); pointers are passed as
``tensor.data_ptr()`` and the stream as ``torch.cuda.current_stream().cuda_stream``.
There is no fallback: if the shared library is missing, importing fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# CDMT_LIBRARY selects another build of the same library (e.g. one compiled with other flags)
LIB_PATH = os.environ.get("CDMT_LIBRARY") or os.path.join(_HERE, "libcdmt.so")

OK, ERR_ARG, ERR_SIZE, ERR_WORKSPACE, ERR_CUDA, ERR_ALLOC = range(6)
IN_CF32, IN_CI8, IN_PF32, IN_PI8 = 0, 1, 2, 3
REF_CHANNEL, REF_SUBBAND = 0, 1
OPT_CHUNK_UNITS, OPT_DM_TILE, OPT_ACCURATE_SINCOS, OPT_PROFILE, OPT_FORCE_GENERIC = 0, 1, 2, 3, 4
OPT_HOST_GROUP_BLOCKS = 5
OPT_KEEP_TABLES = 6
OUT_F32, OUT_U8 = 0, 1
OPT_FUSED_KERNEL = 4  # 0 auto, 1 general, 2 scalar fast, 3 packed half transforms + TMEM, 4 packed polarisations + TMEM

EXPORTS = [
    "cdmt_plan_create", "cdmt_plan_destroy", "cdmt_plan_set_option", "cdmt_plan_query",
    "cdmt_execute", "cdmt_execute_sums", "cdmt_execute_host", "cdmt_execute_host_async", "cdmt_host_layout",
    "cdmt_host_scratch_bytes", "cdmt_host_traffic_bytes", "cdmt_unpack",
    "cdmt_forward_spectrum", "cdmt_redigitize", "cdmt_redigitize_sums", "cdmt_redigitize_workspace_bytes",
    "cdmt_redigitize_static", "cdmt_redigitize_static_max_bytes",
    "cdmt_incoherent_query", "cdmt_incoherent_shifts", "cdmt_incoherent_dedisperse", "cdmt_incoherent_carry", "cdmt_incoherent_work",
    "cdmt_sweep_seconds", "cdmt_min_overlap", "cdmt_suggest_sizes",
    "cdmt_multiplan_create", "cdmt_multiplan_destroy", "cdmt_multiplan_query", "cdmt_multiplan_group",
    "cdmt_multiplan_execute", "cdmt_multiplan_last_launch_count",
    "cdmt_measure_fp32_peak", "cdmt_last_launch_count", "cdmt_profile_read", "cdmt_strerror",
    "cdmt_version",
]

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libcdmt.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
        "(nvcc, sm_100a). There is no CPU fallback.")

_lib = C.CDLL(LIB_PATH)

_vp, _ll, _sz, _i, _d = C.c_void_p, C.c_longlong, C.c_size_t, C.c_int, C.c_double
_lib.cdmt_plan_create.argtypes = [C.POINTER(_vp), _i, C.POINTER(_d), _d, _i, _i, _i, _i, _i,
                                  C.POINTER(_d), _i, _i]
_lib.cdmt_plan_destroy.argtypes = [_vp]
_lib.cdmt_plan_set_option.argtypes = [_vp, _i, _ll]
_lib.cdmt_plan_query.argtypes = [_vp, _ll, C.POINTER(_i), C.POINTER(_ll), C.POINTER(_ll),
                                 C.POINTER(_sz), C.POINTER(_sz)]
_lib.cdmt_execute.argtypes = [_vp, _vp, _ll, _ll, _vp, _ll, _vp, _sz, _vp]
_lib.cdmt_execute_sums.argtypes = [_vp, _vp, _ll, _ll, _vp, _ll, _vp, _vp, _sz, _vp]
_lib.cdmt_execute_host.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp, _sz, _vp]
_lib.cdmt_execute_host_async.argtypes = [_vp, _vp, _ll, _ll, _i, _vp, _vp, _vp, _d, _d, _vp, _sz, _vp]
_lib.cdmt_host_layout.argtypes = [_vp, _ll, _i, C.POINTER(_sz), C.POINTER(_i), C.POINTER(_i), C.POINTER(_sz),
                                  C.POINTER(_sz)]
_lib.cdmt_redigitize_sums.argtypes = [_vp, _vp, _ll, _ll, _d, _d, _vp, _vp, _ll, _vp, _vp, _vp]
_lib.cdmt_host_scratch_bytes.argtypes = [_vp, _ll, C.POINTER(_sz)]
_lib.cdmt_host_traffic_bytes.argtypes = [_vp, _ll, C.POINTER(_sz), C.POINTER(_sz)]
_lib.cdmt_unpack.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp]
_lib.cdmt_forward_spectrum.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp, _sz, _vp]
_lib.cdmt_redigitize.argtypes = [_vp, _vp, _ll, _ll, _d, _d, _vp, _ll, _vp, _vp, _vp, _sz, _vp]
_lib.cdmt_redigitize_workspace_bytes.argtypes = [_vp, _ll, C.POINTER(_sz)]
_lib.cdmt_redigitize_static.argtypes = [_vp, _vp, _ll, _ll, _d, _d, _vp, _ll, _vp, _vp, _vp]
_lib.cdmt_redigitize_static_max_bytes.argtypes = [C.POINTER(_sz)]
_lib.cdmt_incoherent_query.argtypes = [_vp, _i, C.POINTER(_d), _ll, C.POINTER(_i), C.POINTER(_i), C.POINTER(_ll),
                                       C.POINTER(_i), C.POINTER(_sz)]
_lib.cdmt_incoherent_shifts.argtypes = [_vp, _i, C.POINTER(_d), _vp]
_lib.cdmt_incoherent_dedisperse.argtypes = [_vp, _vp, _ll, _ll, _i, C.POINTER(_d), _vp, _ll, _ll, _vp, _sz, _vp]
_lib.cdmt_incoherent_carry.argtypes = [_vp, _vp, _ll, _ll, _i, _vp]
_lib.cdmt_incoherent_work.argtypes = [_vp, _i, C.POINTER(_d), _ll, C.POINTER(_d), C.POINTER(_d)]
_lib.cdmt_sweep_seconds.argtypes = [_d, _d, _d]
_lib.cdmt_sweep_seconds.restype = _d
_lib.cdmt_suggest_sizes.argtypes = [_i, C.POINTER(_d), _d, _i, _i, _d, _i, _d, C.POINTER(_i), C.POINTER(_i)]
_lib.cdmt_multiplan_create.argtypes = [C.POINTER(_vp), _i, C.POINTER(_d), _d, _i, _i, _i, C.POINTER(_d), _i, _i, _d, _i]
_lib.cdmt_multiplan_destroy.argtypes = [_vp]
_lib.cdmt_multiplan_query.argtypes = [_vp, _ll, C.POINTER(_i), C.POINTER(_ll), C.POINTER(_ll), C.POINTER(_sz),
                                      C.POINTER(_sz), C.POINTER(_d)]
_lib.cdmt_multiplan_group.argtypes = [_vp, _i, _ll, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i), C.POINTER(_i),
                                      C.POINTER(_ll), C.POINTER(_ll)]
_lib.cdmt_multiplan_execute.argtypes = [_vp, _vp, _ll, _ll, _vp, _ll, _vp, _sz, _vp]
_lib.cdmt_multiplan_last_launch_count.argtypes = [_vp]
_lib.cdmt_multiplan_last_launch_count.restype = _ll
_lib.cdmt_min_overlap.argtypes = [_vp]
_lib.cdmt_min_overlap.restype = _ll
_lib.cdmt_measure_fp32_peak.argtypes = [_vp, _sz, _i, C.POINTER(_d), _vp]
_lib.cdmt_last_launch_count.argtypes = [_vp]
_lib.cdmt_profile_read.argtypes = [_vp, C.POINTER(_d), C.POINTER(_d), C.POINTER(_ll), C.POINTER(_ll)]
_lib.cdmt_last_launch_count.restype = _ll
_lib.cdmt_strerror.argtypes = [_i]
_lib.cdmt_strerror.restype = C.c_char_p
_lib.cdmt_version.restype = C.c_char_p


class CdmtError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: %s (status %d)" % (where, cdmt_strerror(status), status))


def _check(status: int, where: str):
    if status != OK:
        raise CdmtError(status, where)


def cdmt_strerror(status: int) -> str:
    return _lib.cdmt_strerror(int(status)).decode()


def cdmt_version() -> str:
    return _lib.cdmt_version().decode()


def cdmt_sweep_seconds(fcen_mhz: float, bw_mhz: float, dm: float) -> float:
    return _lib.cdmt_sweep_seconds(fcen_mhz, bw_mhz, dm)


def _ptr(t) -> int:
    """torch tensor / numpy array / int -> raw address."""
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Plan:
    """Owner of a cdmt_plan* (host state only)."""

    def __init__(self, handle: int, nsub, nfft, noverlap, nchan, ndec, ndm, in_dtype, chirp_ref):
        self.handle = handle
        self.nsub, self.nfft, self.noverlap, self.nchan, self.ndec = nsub, nfft, noverlap, nchan, ndec
        self.ndm, self.in_dtype, self.chirp_ref = ndm, in_dtype, chirp_ref

    def __del__(self):
        if getattr(self, "handle", None) and _lib is not None:   # _lib is None during interpreter shutdown
            _lib.cdmt_plan_destroy(self.handle)
            self.handle = None


def cdmt_plan_create(nsub, fcen_mhz, bw_mhz, nfft, noverlap, nchan, ndec, dm,
                     in_dtype=IN_CF32, chirp_ref=REF_CHANNEL) -> Plan:
    fc = np.ascontiguousarray(fcen_mhz, dtype=np.float64).reshape(-1)
    dms = np.ascontiguousarray(dm, dtype=np.float64).reshape(-1)
    h = _vp()
    st = _lib.cdmt_plan_create(C.byref(h), int(nsub), fc.ctypes.data_as(C.POINTER(_d)), float(bw_mhz),
                               int(nfft), int(noverlap), int(nchan), int(ndec), int(dms.size),
                               dms.ctypes.data_as(C.POINTER(_d)), int(in_dtype), int(chirp_ref))
    _check(st, "cdmt_plan_create")
    return Plan(h.value, int(nsub), int(nfft), int(noverlap), int(nchan), int(ndec), int(dms.size),
                int(in_dtype), int(chirp_ref))


def cdmt_plan_destroy(plan: Plan):
    if plan.handle:
        _check(_lib.cdmt_plan_destroy(plan.handle), "cdmt_plan_destroy")
        plan.handle = None


def cdmt_plan_set_option(plan: Plan, key: int, value: int):
    _check(_lib.cdmt_plan_set_option(plan.handle, int(key), int(value)), "cdmt_plan_set_option")


def cdmt_plan_query(plan: Plan, nsamp: int) -> dict:
    nb, cons, nout, ob, wb = _i(), _ll(), _ll(), _sz(), _sz()
    st = _lib.cdmt_plan_query(plan.handle, int(nsamp), C.byref(nb), C.byref(cons), C.byref(nout),
                              C.byref(ob), C.byref(wb))
    _check(st, "cdmt_plan_query")
    return dict(nblock=nb.value, nsamp_consumed=cons.value, nout_per_chan=nout.value,
                out_bytes=ob.value, workspace_bytes=wb.value)


def cdmt_execute(plan: Plan, d_in, nsamp: int, in_stride_pol: int, d_out, out_stride_dm: int,
                 d_workspace, workspace_bytes: int, stream=None):
    st = _lib.cdmt_execute(plan.handle, _ptr(d_in), int(nsamp), int(in_stride_pol), _ptr(d_out),
                           int(out_stride_dm), _ptr(d_workspace), int(workspace_bytes), _stream(stream))
    _check(st, "cdmt_execute")


def cdmt_execute_sums(plan: Plan, d_in, nsamp: int, in_stride_pol: int, d_out, out_stride_dm: int, d_segsum,
                      d_workspace, workspace_bytes: int, stream=None):
    st = _lib.cdmt_execute_sums(plan.handle, _ptr(d_in), int(nsamp), int(in_stride_pol), _ptr(d_out),
                                int(out_stride_dm), _ptr(d_segsum), _ptr(d_workspace), int(workspace_bytes),
                                _stream(stream))
    _check(st, "cdmt_execute_sums")


def cdmt_host_layout(plan: Plan, nsamp: int, out_kind: int = OUT_F32) -> dict:
    sb, ng, gb, a, b = _sz(), _i(), _i(), _sz(), _sz()
    _check(_lib.cdmt_host_layout(plan.handle, int(nsamp), int(out_kind), C.byref(sb), C.byref(ng), C.byref(gb),
                                 C.byref(a), C.byref(b)), "cdmt_host_layout")
    return dict(scratch_bytes=sb.value, ngroups=ng.value, group_blocks=gb.value, h2d_bytes=a.value,
                d2h_bytes=b.value)


def cdmt_execute_host_async(plan: Plan, h_in, nsamp: int, in_stride_pol: int, out_kind: int, h_out, h_offset,
                            h_scale, qmean: float, qstd: float, d_scratch, scratch_bytes: int, stream=None):
    st = _lib.cdmt_execute_host_async(plan.handle, _ptr(h_in), int(nsamp), int(in_stride_pol), int(out_kind),
                                      _ptr(h_out), _ptr(h_offset), _ptr(h_scale), float(qmean), float(qstd),
                                      _ptr(d_scratch), int(scratch_bytes), _stream(stream))
    _check(st, "cdmt_execute_host_async")


def cdmt_host_scratch_bytes(plan: Plan, nsamp: int) -> int:
    n = _sz()
    _check(_lib.cdmt_host_scratch_bytes(plan.handle, int(nsamp), C.byref(n)), "cdmt_host_scratch_bytes")
    return n.value


def cdmt_host_traffic_bytes(plan: Plan, nsamp: int):
    a, b = _sz(), _sz()
    _check(_lib.cdmt_host_traffic_bytes(plan.handle, int(nsamp), C.byref(a), C.byref(b)), "cdmt_host_traffic_bytes")
    return a.value, b.value


def cdmt_execute_host(plan: Plan, h_in, nsamp: int, in_stride_pol: int, h_out, d_scratch,
                      scratch_bytes: int, stream=None):
    st = _lib.cdmt_execute_host(plan.handle, _ptr(h_in), int(nsamp), int(in_stride_pol), _ptr(h_out),
                                _ptr(d_scratch), int(scratch_bytes), _stream(stream))
    _check(st, "cdmt_execute_host")


def cdmt_unpack(plan: Plan, d_in, nsamp: int, in_stride_pol: int, d_blocks, stream=None):
    st = _lib.cdmt_unpack(plan.handle, _ptr(d_in), int(nsamp), int(in_stride_pol), _ptr(d_blocks),
                          _stream(stream))
    _check(st, "cdmt_unpack")


def cdmt_forward_spectrum(plan: Plan, d_in, nsamp: int, in_stride_pol: int, d_spec, d_workspace,
                          workspace_bytes: int, stream=None):
    st = _lib.cdmt_forward_spectrum(plan.handle, _ptr(d_in), int(nsamp), int(in_stride_pol), _ptr(d_spec),
                                    _ptr(d_workspace), int(workspace_bytes), _stream(stream))
    _check(st, "cdmt_forward_spectrum")


def cdmt_redigitize_workspace_bytes(plan: Plan, nblock: int) -> int:
    n = _sz()
    _check(_lib.cdmt_redigitize_workspace_bytes(plan.handle, int(nblock), C.byref(n)),
           "cdmt_redigitize_workspace_bytes")
    return n.value


def cdmt_redigitize(plan: Plan, d_fb, fb_stride_dm: int, nblock: int, qmean: float, qstd: float, d_codes,
                    codes_stride_dm: int, d_offset, d_scale, d_workspace, workspace_bytes: int, stream=None):
    st = _lib.cdmt_redigitize(plan.handle, _ptr(d_fb), int(fb_stride_dm), int(nblock), float(qmean), float(qstd),
                              _ptr(d_codes), int(codes_stride_dm), _ptr(d_offset), _ptr(d_scale),
                              _ptr(d_workspace), int(workspace_bytes), _stream(stream))
    _check(st, "cdmt_redigitize")


def cdmt_redigitize_static(plan: Plan, d_fb, fb_stride_dm: int, nblock: int, qmean: float, qstd: float, d_codes,
                           codes_stride_dm: int, d_offset, d_scale, stream=None):
    st = _lib.cdmt_redigitize_static(plan.handle, _ptr(d_fb), int(fb_stride_dm), int(nblock), float(qmean),
                                     float(qstd), _ptr(d_codes), int(codes_stride_dm), _ptr(d_offset),
                                     _ptr(d_scale), _stream(stream))
    _check(st, "cdmt_redigitize_static")


def cdmt_redigitize_static_max_bytes() -> int:
    n = _sz(0)
    _check(_lib.cdmt_redigitize_static_max_bytes(C.byref(n)), "cdmt_redigitize_static_max_bytes")
    return int(n.value)


def cdmt_redigitize_sums(plan: Plan, d_fb, fb_stride_dm: int, nblock: int, qmean: float, qstd: float, d_segsum,
                         d_codes, codes_stride_dm: int, d_offset, d_scale, stream=None):
    st = _lib.cdmt_redigitize_sums(plan.handle, _ptr(d_fb), int(fb_stride_dm), int(nblock), float(qmean),
                                   float(qstd), _ptr(d_segsum), _ptr(d_codes), int(codes_stride_dm),
                                   _ptr(d_offset), _ptr(d_scale), _stream(stream))
    _check(st, "cdmt_redigitize_sums")


def _ddm(ddm):
    a = np.ascontiguousarray(ddm, dtype=np.float64).reshape(-1)
    return a, a.ctypes.data_as(C.POINTER(_d))


def cdmt_incoherent_query(plan: Plan, ddm, nt_in: int) -> dict:
    a, pa = _ddm(ddm)
    smin, rng, ng, nout, nws = _i(), _i(), _i(), _ll(), _sz()
    _check(_lib.cdmt_incoherent_query(plan.handle, a.size, pa, int(nt_in), C.byref(smin), C.byref(rng),
                                      C.byref(nout), C.byref(ng), C.byref(nws)), "cdmt_incoherent_query")
    return dict(shift_min=smin.value, shift_range=rng.value, nt_out=nout.value, ngroups=ng.value,
                workspace_bytes=nws.value)


def cdmt_incoherent_shifts(plan: Plan, ddm) -> np.ndarray:
    a, pa = _ddm(ddm)
    out = np.empty((a.size, plan.nsub * plan.nchan), dtype=np.int32)
    _check(_lib.cdmt_incoherent_shifts(plan.handle, a.size, pa, out.ctypes.data), "cdmt_incoherent_shifts")
    return out


def cdmt_incoherent_dedisperse(plan: Plan, d_fb, fb_stride_dm: int, nt_in: int, ddm, d_ts, ts_stride_dm: int,
                               ts_pitch: int, d_workspace, workspace_bytes: int, stream=None):
    a, pa = _ddm(ddm)
    st = _lib.cdmt_incoherent_dedisperse(plan.handle, _ptr(d_fb), int(fb_stride_dm), int(nt_in), a.size, pa,
                                         _ptr(d_ts), int(ts_stride_dm), int(ts_pitch), _ptr(d_workspace),
                                         int(workspace_bytes), _stream(stream))
    _check(st, "cdmt_incoherent_dedisperse")


def cdmt_incoherent_carry(plan: Plan, d_fb, fb_stride_dm: int, nt_in: int, shift_range: int, stream=None):
    _check(_lib.cdmt_incoherent_carry(plan.handle, _ptr(d_fb), int(fb_stride_dm), int(nt_in), int(shift_range),
                                      _stream(stream)), "cdmt_incoherent_carry")


def cdmt_incoherent_work(plan: Plan, ddm, nt_in: int):
    a, pa = _ddm(ddm)
    x, y = _d(), _d()
    _check(_lib.cdmt_incoherent_work(plan.handle, a.size, pa, int(nt_in), C.byref(x), C.byref(y)), "cdmt_incoherent_work")
    return x.value, y.value


def cdmt_min_overlap(plan: Plan) -> int:
    return _lib.cdmt_min_overlap(plan.handle)


def cdmt_suggest_sizes(fcen_mhz, bw_mhz: float, nchan: int, ndec: int, dm_max_abs: float,
                       chirp_ref: int = REF_CHANNEL, min_efficiency: float = 0.75):
    """(nfft, noverlap) from the dispersion sweep of the lowest channel / subband."""
    f = np.ascontiguousarray(fcen_mhz, dtype=np.float64).reshape(-1)
    nfft, nov = _i(), _i()
    _check(_lib.cdmt_suggest_sizes(f.size, f.ctypes.data_as(C.POINTER(_d)), float(bw_mhz), int(nchan), int(ndec),
                                   float(dm_max_abs), int(chirp_ref), float(min_efficiency), C.byref(nfft),
                                   C.byref(nov)), "cdmt_suggest_sizes")
    return nfft.value, nov.value


class MultiPlan:
    """Owner of a cdmt_multiplan*."""

    def __init__(self, handle: int, nsub, nchan, ndec, ndm, in_dtype):
        self.handle = handle
        self.nsub, self.nchan, self.ndec, self.ndm, self.in_dtype = nsub, nchan, ndec, ndm, in_dtype

    def __del__(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.cdmt_multiplan_destroy(self.handle)
            self.handle = None


def cdmt_multiplan_create(nsub, fcen_mhz, bw_mhz, nchan, ndec, dm, in_dtype=IN_CF32, chirp_ref=REF_CHANNEL,
                          min_efficiency=0.9, max_groups=4) -> MultiPlan:
    fc = np.ascontiguousarray(fcen_mhz, dtype=np.float64).reshape(-1)
    dms = np.ascontiguousarray(dm, dtype=np.float64).reshape(-1)
    h = _vp()
    st = _lib.cdmt_multiplan_create(C.byref(h), int(nsub), fc.ctypes.data_as(C.POINTER(_d)), float(bw_mhz), int(nchan),
                                    int(ndec), int(dms.size), dms.ctypes.data_as(C.POINTER(_d)), int(in_dtype),
                                    int(chirp_ref), float(min_efficiency), int(max_groups))
    _check(st, "cdmt_multiplan_create")
    return MultiPlan(h.value, int(nsub), int(nchan), int(ndec), int(dms.size), int(in_dtype))


def cdmt_multiplan_destroy(mp: MultiPlan):
    if mp.handle:
        _check(_lib.cdmt_multiplan_destroy(mp.handle), "cdmt_multiplan_destroy")
        mp.handle = None


def cdmt_multiplan_query(mp: MultiPlan, nsamp: int) -> dict:
    ng, nv, na, ob, wb, kf = _i(), _ll(), _ll(), _sz(), _sz(), _d()
    _check(_lib.cdmt_multiplan_query(mp.handle, int(nsamp), C.byref(ng), C.byref(nv), C.byref(na), C.byref(ob),
                                     C.byref(wb), C.byref(kf)), "cdmt_multiplan_query")
    return dict(ngroups=ng.value, nout_valid=nv.value, nout_alloc=na.value, out_bytes=ob.value,
                workspace_bytes=wb.value, kept_fraction=kf.value)


def cdmt_multiplan_group(mp: MultiPlan, group: int, nsamp: int) -> dict:
    s0, ns, nf, no, fs, nr = _i(), _i(), _i(), _i(), _ll(), _ll()
    _check(_lib.cdmt_multiplan_group(mp.handle, int(group), int(nsamp), C.byref(s0), C.byref(ns), C.byref(nf),
                                     C.byref(no), C.byref(fs), C.byref(nr)), "cdmt_multiplan_group")
    return dict(first_subband=s0.value, nsub=ns.value, nfft=nf.value, noverlap=no.value, first_sample=fs.value,
                nout=nr.value)


def cdmt_multiplan_execute(mp: MultiPlan, d_in, nsamp: int, in_stride_pol: int, d_out, out_stride_dm: int,
                           d_workspace, workspace_bytes: int, stream=None):
    st = _lib.cdmt_multiplan_execute(mp.handle, _ptr(d_in), int(nsamp), int(in_stride_pol), _ptr(d_out),
                                     int(out_stride_dm), _ptr(d_workspace), int(workspace_bytes), _stream(stream))
    _check(st, "cdmt_multiplan_execute")


def cdmt_multiplan_last_launch_count(mp: MultiPlan) -> int:
    return _lib.cdmt_multiplan_last_launch_count(mp.handle)


def cdmt_last_launch_count(plan: Plan) -> int:
    return _lib.cdmt_last_launch_count(plan.handle)


def cdmt_profile_read(plan: Plan) -> dict:
    a, b, na, nb = _d(), _d(), _ll(), _ll()
    _check(_lib.cdmt_profile_read(plan.handle, C.byref(a), C.byref(b), C.byref(na), C.byref(nb)),
           "cdmt_profile_read")
    return dict(ms_forward=a.value, ms_fused=b.value, n_forward=na.value, n_fused=nb.value)


def cdmt_measure_fp32_peak(d_scratch, scratch_bytes: int, iters: int = 5, stream=None) -> float:
    tf = _d()
    st = _lib.cdmt_measure_fp32_peak(_ptr(d_scratch), int(scratch_bytes), int(iters), C.byref(tf),
                                     _stream(stream))
    _check(st, "cdmt_measure_fp32_peak")
    return tf.value


# ---------------------------------------------------------------------------------------
# Convenience for tests and bench: allocate with torch, call the ABI, return the tensor.
# ---------------------------------------------------------------------------------------
def run_on_device(plan: Plan, d_in, nsamp: int, stream=None, out=None, workspace=None):
    """d_in: CUDA tensor [nsub][2][T] complex64, [nsub][2][T][2] int8, or planar [nsub][2][2][T] float32 / int8. Returns
    out [ndm][nblock*Vd][nsub*nchan] float32 (CUDA)."""
    import torch
    q = cdmt_plan_query(plan, nsamp)
    nt = q["nout_per_chan"]
    nch = plan.nsub * plan.nchan
    if out is None:
        out = torch.empty((plan.ndm, nt, nch), dtype=torch.float32, device=d_in.device)
    if workspace is None:
        workspace = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device=d_in.device)
    if plan.in_dtype in (IN_PF32, IN_PI8):
        stride_pol = d_in.stride(2)          # [nsub][2][2 parts][T] real words
    else:
        stride_pol = d_in.stride(1) // (2 if plan.in_dtype == IN_CI8 else 1)
    cdmt_execute(plan, d_in, nsamp, stride_pol, out, nt * nch, workspace, workspace.numel(), stream)
    return out
