"""B200-native direct incoherent dedispersion (hot path of arxiv/paper_1112_0065).

Thin ctypes binding over the C ABI in ``include/dedisp.h`` -- same names, argument
marshalling only.  Every step of the path (delay table, unpack, gather-sum, output
conversion) runs in the CUDA kernels of ``libdedisp_b200.so``; PyTorch is used by
callers for device memory and streams only.  There is no CPU fallback: if the
library is not built or no CUDA device is usable, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from pathlib import Path

_PKG = Path(__file__).resolve().parent
# DEDISP_B200_LIB selects a tuning variant built by build.build(defs=..., out=...)
LIB_PATH = Path(os.environ.get("DEDISP_B200_LIB") or (_PKG / "libdedisp_b200.so"))

DEDISP_OK = 0
DEDISP_ERR_INVALID_ARG = 1
DEDISP_ERR_NO_DM_LIST = 2
DEDISP_ERR_UNSUPPORTED_NBITS = 3
DEDISP_ERR_UNSUPPORTED_DTYPE = 4
DEDISP_ERR_OVERFLOW = 5
DEDISP_ERR_ALLOC = 6
DEDISP_ERR_CUDA = 7
DEDISP_ERR_SCRATCH_LIMIT = 8
DEDISP_OUT_U32 = 0
DEDISP_OUT_F32 = 1
DEDISP_KERNEL_AUTO = 0
DEDISP_KERNEL_DIRECT = 1
DEDISP_KERNEL_BITSLICE = 2
DEDISP_KERNEL_PAIRS = 3
DEDISP_KERNEL_QUADS = 4

# every symbol include/dedisp.h declares: (restype, argtypes)
_vp, _i, _ll, _sz, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_size_t, ctypes.c_double
ABI = {
    "dedisp_plan_create": (_i, [ctypes.POINTER(_vp), _i, _d, _d, _d]),
    "dedisp_set_dm_list": (_i, [_vp, ctypes.POINTER(_d), _i]),
    "dedisp_execute": (_i, [_vp, _ll, _vp, _i, _vp, _i, _vp]),
    "dedisp_execute_batch": (_i, [_vp, _i, _ll, _vp, _sz, _i, _vp, _sz, _i, _vp]),
    "dedisp_execute_tscrunch": (_i, [_vp, _i, _i, _ll, _vp, _sz, _i, _vp, _sz, _i, _vp]),
    "dedisp_get_in_row_stride_bytes_tscrunch": (_sz, [_vp, _i, _ll, _i]),
    "dedisp_execute_host": (_i, [_vp, _i, _ll, _vp, _i, _vp, _i]),
    "dedisp_reserve": (_i, [_vp, _i, _ll, _i]),
    "dedisp_static_scratch_bytes": (_sz, []),
    "dedisp_execute_static": (_i, [_vp, _ll, _vp, _i, _vp, _i, _vp]),
    "dedisp_destroy": (_i, [_vp]),
    "dedisp_get_max_delay": (_i, [_vp]),
    "dedisp_get_nchans": (_i, [_vp]),
    "dedisp_get_ndm": (_i, [_vp]),
    "dedisp_get_in_row_stride_bytes": (_sz, [_vp, _ll, _i]),
    "dedisp_get_delay_table": (_i, [_vp, ctypes.POINTER(ctypes.c_int32)]),
    "dedisp_set_kernel": (_i, [_vp, _i]),
    "dedisp_get_last_kernel": (_i, [_vp]),
    "dedisp_set_timing": (_i, [_vp, _i]),
    "dedisp_get_last_kernel_ms": (_i, [_vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]),
    "dedisp_get_launch_count": (ctypes.c_ulonglong, []),
    "dedisp_debug_quad_tables": (_i, [_i, _i, _vp, _i, _vp, _vp, _vp, _vp, _vp, _vp]),
    "dedisp_debug_checks_compiled": (_i, []),
    "dedisp_debug_set_poison": (_i, [_vp, _i]),
    "dedisp_debug_inject_fault": (_i, [_vp, _i]),
    "dedisp_debug_check_errors": (_i, [_vp, ctypes.POINTER(ctypes.c_ulonglong)]),
    "dedisp_get_last_cuda_error": (_i, [_vp]),
    "dedisp_get_error_string": (ctypes.c_char_p, [_i]),
    "dedisp_matched_filter": (_i, [_vp, _i, _ll, _ll, _i, ctypes.POINTER(_i), _i, ctypes.c_uint, _vp, _vp]),
    "dedisp_matched_filter_rms_workspace_bytes": (_sz, [_ll, _ll, _i]),
    "dedisp_matched_filter_rms": (_i, [_vp, _i, _ll, _ll, _i, ctypes.POINTER(_i), _i, ctypes.c_uint, _vp, _vp, _vp, _vp,
                                       _sz, _vp]),
    "dedisp_matched_filter_hint_blocks": (_ll, [_ll, ctypes.POINTER(_i), _i, ctypes.POINTER(_i), ctypes.POINTER(_i)]),
    "dedisp_find_events_hinted": (_i, [_vp, _ll, _ll, _vp, ctypes.c_float, _vp, _i, _i, _vp, _sz, _vp, _ll, _vp, _vp]),
    "dedisp_find_events_workspace_bytes": (_sz, [_ll, _ll]),
    "dedisp_search_events_workspace_bytes": (_sz, [_ll, _ll, ctypes.POINTER(_i), _i, _ll]),
    "dedisp_search_events": (_i, [_vp, _i, _ll, _ll, _i, ctypes.POINTER(_i), _i, ctypes.c_uint, ctypes.c_float, _vp, _ll,
                                  _vp, _sz, _vp, _ll, _vp, _vp]),
    "dedisp_find_events": (_i, [_vp, _ll, _ll, _vp, ctypes.c_float, _vp, _sz, _vp, _ll, _vp, _vp]),
    "dedisp_series_rms": (_i, [_vp, _ll, _ll, _vp, _vp]),
    "dedisp_transpose_time_major": (_i, [_vp, _i, _ll, _i, _vp, _vp]),
    "dedisp_rfi_mask": (_i, [_vp, _i, _i, _ll, _ll, _sz, _vp, _vp, ctypes.c_float, _i, _vp, _vp]),
    "dedisp_rfi_beam_counts": (_i, [_vp, _i, _i, _ll, _ll, _sz, _vp, _vp, ctypes.c_float, _vp, _vp]),
    "dedisp_rfi_mask_from_counts": (_i, [_vp, _ll, _ll, _i, _vp, _vp]),
    "dedisp_veto_events": (_i, [_vp, _vp, _ll, _vp, _ll, _vp, _vp]),
}
DEDISP_MF_MAX_WIDTH = 8192
DEDISP_EVENT_BYTES = 20      # struct dedisp_event {int series, t_start, length, t_peak; float peak;}

_lib = None


class DedispError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = lib().dedisp_get_error_string(status).decode()
        super().__init__(f"{where}: {msg} (status {status}, cudaError {cuda_error})")


def lib() -> ctypes.CDLL:
    """Load libdedisp_b200.so (built in-tree by ``paper_1112_0065_b200.build``)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is not built: run `python -m paper_1112_0065_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(str(LIB_PATH))
        for name, (res, args) in ABI.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array or plain int."""
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return x.ctypes.data


def _check(plan, st: int, where: str):
    if st != DEDISP_OK:
        ce = lib().dedisp_get_last_cuda_error(plan) if plan else 0
        raise DedispError(st, where, ce)


def dedisp_plan_create(nchans: int, dt: float, f_top: float, df: float) -> int:
    h = _vp()
    st = lib().dedisp_plan_create(ctypes.byref(h), nchans, dt, f_top, df)
    _check(None, st, "dedisp_plan_create")
    return h.value


def dedisp_set_dm_list(plan: int, dms) -> None:
    arr = (ctypes.c_double * len(dms))(*[float(v) for v in dms])
    _check(plan, lib().dedisp_set_dm_list(plan, arr, len(dms)), "dedisp_set_dm_list")


def dedisp_execute(plan: int, nsamps_out: int, in_ptr, in_nbits: int, out_ptr, out_dtype: int,
                   stream: int = 0) -> None:
    st = lib().dedisp_execute(plan, nsamps_out, _ptr(in_ptr), in_nbits, _ptr(out_ptr), out_dtype,
                              stream or None)
    _check(plan, st, "dedisp_execute")


def dedisp_execute_batch(plan: int, nbeams: int, nsamps_out: int, in_ptr, in_beam_stride: int,
                         in_nbits: int, out_ptr, out_beam_stride: int, out_dtype: int,
                         stream: int = 0) -> None:
    st = lib().dedisp_execute_batch(plan, nbeams, nsamps_out, _ptr(in_ptr), in_beam_stride, in_nbits,
                                    _ptr(out_ptr), out_beam_stride, out_dtype, stream or None)
    _check(plan, st, "dedisp_execute_batch")


def dedisp_execute_tscrunch(plan: int, tscrunch: int, nbeams: int, nsamps_out: int, in_ptr, in_beam_stride: int,
                            in_nbits: int, out_ptr, out_beam_stride: int, out_dtype: int,
                            stream: int = 0) -> None:
    st = lib().dedisp_execute_tscrunch(plan, tscrunch, nbeams, nsamps_out, _ptr(in_ptr), in_beam_stride,
                                       in_nbits, _ptr(out_ptr), out_beam_stride, out_dtype, stream or None)
    _check(plan, st, "dedisp_execute_tscrunch")


def dedisp_get_in_row_stride_bytes_tscrunch(plan: int, tscrunch: int, nsamps_out: int, in_nbits: int) -> int:
    return lib().dedisp_get_in_row_stride_bytes_tscrunch(plan, tscrunch, nsamps_out, in_nbits)


def dedisp_execute_host(plan: int, nbeams: int, nsamps_out: int, in_host, in_nbits: int, out_host,
                        out_dtype: int) -> None:
    st = lib().dedisp_execute_host(plan, nbeams, nsamps_out, _ptr(in_host), in_nbits,
                                   _ptr(out_host), out_dtype)
    _check(plan, st, "dedisp_execute_host")


def dedisp_reserve(plan: int, nbeams: int, nsamps_out: int, in_nbits: int) -> None:
    _check(plan, lib().dedisp_reserve(plan, nbeams, nsamps_out, in_nbits), "dedisp_reserve")


def dedisp_static_scratch_bytes() -> int:
    return int(lib().dedisp_static_scratch_bytes())


def dedisp_execute_static(plan: int, nsamps_out: int, in_ptr, in_nbits: int, out_ptr, out_dtype: int,
                          stream: int = 0) -> None:
    """dedisp_execute with the bit planes in a fixed 32 MiB device array: allocates nothing (include/dedisp.h)."""
    st = lib().dedisp_execute_static(plan, nsamps_out, _ptr(in_ptr), in_nbits, _ptr(out_ptr), out_dtype, stream or None)
    _check(plan, st, "dedisp_execute_static")


def dedisp_destroy(plan: int) -> None:
    lib().dedisp_destroy(plan)


def dedisp_get_max_delay(plan: int) -> int:
    return lib().dedisp_get_max_delay(plan)


def dedisp_get_nchans(plan: int) -> int:
    return lib().dedisp_get_nchans(plan)


def dedisp_get_ndm(plan: int) -> int:
    return lib().dedisp_get_ndm(plan)


def dedisp_get_in_row_stride_bytes(plan: int, nsamps_out: int, in_nbits: int) -> int:
    return lib().dedisp_get_in_row_stride_bytes(plan, nsamps_out, in_nbits)


def dedisp_get_delay_table(plan: int):
    import numpy as np
    out = np.empty((dedisp_get_nchans(plan), dedisp_get_ndm(plan)), dtype=np.int32)
    st = lib().dedisp_get_delay_table(plan, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)))
    _check(plan, st, "dedisp_get_delay_table")
    return out


def dedisp_set_kernel(plan: int, which: int) -> None:
    _check(plan, lib().dedisp_set_kernel(plan, which), "dedisp_set_kernel")


def dedisp_get_last_kernel(plan: int) -> int:
    return lib().dedisp_get_last_kernel(plan)


class _QuadTableInfo(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int) for n in ("nv", "vslot_bytes", "plane_words", "tile_words", "nquads_pad", "nrows",
                                            "usable")]


def dedisp_debug_quad_tables(delay_host, lanes_host):
    """Host only (no GPU): (info dict, row0, trip, vlist, rel) -- the quad-row tables for a delay table
    int32 [nchans][ndm] and a lane order int32 [ngroups][32]; the arrays are None when info["usable"] is 0."""
    import numpy as np
    delay = np.ascontiguousarray(delay_host, dtype=np.int32)
    lanes = np.ascontiguousarray(lanes_host, dtype=np.int32)
    nchans, ndm = delay.shape
    ngroups = lanes.shape[0]
    info = _QuadTableInfo()
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p) if a is not None else None
    st = lib().dedisp_debug_quad_tables(nchans, ndm, p(delay), ngroups, p(lanes), ctypes.byref(info), None, None, None,
                                        None)
    _check(None, st, "dedisp_debug_quad_tables")
    d = {n: getattr(info, n) for n, _ in _QuadTableInfo._fields_}
    if not d["usable"]:
        return d, None, None, None, None
    row0 = np.empty(d["nquads_pad"] + 1, dtype=np.int32)
    trip = np.empty((d["nrows"], 4), dtype=np.int32)
    vlist = np.empty((ngroups, d["nquads_pad"], d["nv"], 2), dtype=np.int32)
    rel = np.empty((ngroups, d["nquads_pad"], 32), dtype=np.uint32)
    st = lib().dedisp_debug_quad_tables(nchans, ndm, p(delay), ngroups, p(lanes), ctypes.byref(info), p(row0), p(trip),
                                        p(vlist), p(rel))
    _check(None, st, "dedisp_debug_quad_tables")
    return d, row0, trip, vlist, rel


def dedisp_debug_checks_compiled() -> bool:
    return bool(lib().dedisp_debug_checks_compiled())


def dedisp_debug_set_poison(plan: int, byte_value: int) -> None:
    _check(plan, lib().dedisp_debug_set_poison(plan, byte_value), "dedisp_debug_set_poison")


def dedisp_debug_inject_fault(plan: int, kind: int) -> None:
    _check(plan, lib().dedisp_debug_inject_fault(plan, kind), "dedisp_debug_inject_fault")


def dedisp_debug_check_errors(plan: int) -> list:
    buf = (ctypes.c_ulonglong * 8)()
    _check(plan, lib().dedisp_debug_check_errors(plan, buf), "dedisp_debug_check_errors")
    return list(buf)


def dedisp_get_launch_count() -> int:
    return int(lib().dedisp_get_launch_count())


def dedisp_get_last_cuda_error(plan: int) -> int:
    return lib().dedisp_get_last_cuda_error(plan)


def dedisp_get_error_string(status: int) -> str:
    return lib().dedisp_get_error_string(status).decode()


def dedisp_set_timing(plan: int, enable: bool) -> None:
    _check(plan, lib().dedisp_set_timing(plan, int(enable)), "dedisp_set_timing")


def dedisp_get_last_kernel_ms(plan: int) -> tuple[float, float]:
    """(prepass_ms, main_ms) of the last execute; needs dedisp_set_timing(plan, True)."""
    a, b = ctypes.c_float(), ctypes.c_float()
    _check(plan, lib().dedisp_get_last_kernel_ms(plan, ctypes.byref(a), ctypes.byref(b)),
           "dedisp_get_last_kernel_ms")
    return a.value, b.value


def dedisp_matched_filter(x_ptr, x_dtype: int, nrows: int, nsamps: int, radius: int, widths,
                          x_max: int, z_ptr, stream: int = 0) -> None:
    """Baseline removal + boxcar matched filters (include/dedisp.h)."""
    w = (ctypes.c_int * len(widths))(*[int(v) for v in widths])
    st = lib().dedisp_matched_filter(_ptr(x_ptr), x_dtype, nrows, nsamps, radius, w, len(widths),
                                     x_max, _ptr(z_ptr) if z_ptr is not None else None, stream or None)
    _check(None, st, "dedisp_matched_filter")


def dedisp_matched_filter_rms_workspace_bytes(nrows: int, nsamps: int, nwidths: int) -> int:
    return int(lib().dedisp_matched_filter_rms_workspace_bytes(nrows, nsamps, nwidths))


def dedisp_matched_filter_rms(x_ptr, x_dtype: int, nrows: int, nsamps: int, radius: int, widths,
                              x_max: int, z_ptr, rms_ptr, workspace_ptr, workspace_bytes: int,
                              stream: int = 0, blockmax_ptr=None) -> None:
    """dedisp_matched_filter + the RMS of every filtered series (and, optionally, the block maxima that
    dedisp_find_events_hinted uses) in the same pass (include/dedisp.h)."""
    w = (ctypes.c_int * len(widths))(*[int(v) for v in widths])
    st = lib().dedisp_matched_filter_rms(_ptr(x_ptr), x_dtype, nrows, nsamps, radius, w, len(widths), x_max,
                                         _ptr(z_ptr) if z_ptr is not None else None,
                                         _ptr(rms_ptr) if rms_ptr is not None else None,
                                         _ptr(blockmax_ptr) if blockmax_ptr is not None else None,
                                         _ptr(workspace_ptr) if workspace_ptr is not None else None,
                                         workspace_bytes, stream or None)
    _check(None, st, "dedisp_matched_filter_rms")


def dedisp_search_events_workspace_bytes(nrows: int, nsamps: int, widths, max_blocks: int) -> int:
    w = (ctypes.c_int * len(widths))(*[int(v) for v in widths])
    return int(lib().dedisp_search_events_workspace_bytes(nrows, nsamps, w, len(widths), max_blocks))


def dedisp_search_events(x_ptr, x_dtype: int, nrows: int, nsamps: int, radius: int, widths, x_max: int,
                         nsigma: float, rms_ptr, max_blocks: int, workspace_ptr, workspace_bytes: int, events_ptr,
                         max_events: int, count_ptr, stream: int = 0) -> None:
    """Rows f1 + f2 chained without materialising z: x -> event list (include/dedisp.h)."""
    w = (ctypes.c_int * len(widths))(*[int(v) for v in widths])
    st = lib().dedisp_search_events(_ptr(x_ptr), x_dtype, nrows, nsamps, radius, w, len(widths), x_max, nsigma,
                                    _ptr(rms_ptr), max_blocks, _ptr(workspace_ptr), workspace_bytes,
                                    _ptr(events_ptr) if events_ptr is not None else None, max_events,
                                    _ptr(count_ptr), stream or None)
    _check(None, st, "dedisp_search_events")


def dedisp_matched_filter_hint_blocks(nsamps: int, widths) -> tuple[int, int, int]:
    """(blocks per series, hint_block, hint_offset) of the blockmax array for these widths."""
    w = (ctypes.c_int * len(widths))(*[int(v) for v in widths])
    hb, ho = ctypes.c_int(), ctypes.c_int()
    nb = lib().dedisp_matched_filter_hint_blocks(nsamps, w, len(widths), ctypes.byref(hb), ctypes.byref(ho))
    return int(nb), hb.value, ho.value


def dedisp_find_events_hinted(z_ptr, nseries: int, nsamps: int, sigma_ptr, nsigma: float, hint_ptr,
                              hint_block: int, hint_offset: int, workspace_ptr, workspace_bytes: int,
                              events_ptr, max_events: int, count_ptr, stream: int = 0) -> None:
    """dedisp_find_events that skips the chunks of z the hint rules out (include/dedisp.h)."""
    st = lib().dedisp_find_events_hinted(_ptr(z_ptr), nseries, nsamps, _ptr(sigma_ptr), nsigma,
                                         _ptr(hint_ptr) if hint_ptr is not None else None, hint_block, hint_offset,
                                         _ptr(workspace_ptr), workspace_bytes,
                                         _ptr(events_ptr) if events_ptr is not None else None, max_events,
                                         _ptr(count_ptr), stream or None)
    _check(None, st, "dedisp_find_events_hinted")


def dedisp_find_events_workspace_bytes(nseries: int, nsamps: int) -> int:
    return int(lib().dedisp_find_events_workspace_bytes(nseries, nsamps))


def dedisp_find_events(z_ptr, nseries: int, nsamps: int, sigma_ptr, nsigma: float, workspace_ptr,
                       workspace_bytes: int, events_ptr, max_events: int, count_ptr,
                       stream: int = 0) -> None:
    """Sigma-cut + grouping of contiguous regions into events (include/dedisp.h)."""
    st = lib().dedisp_find_events(_ptr(z_ptr), nseries, nsamps, _ptr(sigma_ptr), nsigma,
                                  _ptr(workspace_ptr), workspace_bytes,
                                  _ptr(events_ptr) if events_ptr is not None else None, max_events,
                                  _ptr(count_ptr), stream or None)
    _check(None, st, "dedisp_find_events")


def dedisp_series_rms(z_ptr, nseries: int, nsamps: int, rms_ptr, stream: int = 0) -> None:
    _check(None, lib().dedisp_series_rms(_ptr(z_ptr), nseries, nsamps, _ptr(rms_ptr), stream or None),
           "dedisp_series_rms")


def dedisp_rfi_mask(x_ptr, x_dtype: int, nbeams: int, nseries: int, nsamps: int, beam_stride_bytes: int,
                    mean_ptr, sigma_ptr, nsigma: float, min_beams: int, mask_ptr, stream: int = 0) -> None:
    """Multibeam coincidence RFI mask (include/dedisp.h)."""
    st = lib().dedisp_rfi_mask(_ptr(x_ptr), x_dtype, nbeams, nseries, nsamps, beam_stride_bytes,
                               _ptr(mean_ptr), _ptr(sigma_ptr), nsigma, min_beams, _ptr(mask_ptr),
                               stream or None)
    _check(None, st, "dedisp_rfi_mask")


def dedisp_rfi_beam_counts(x_ptr, x_dtype: int, nbeams: int, nseries: int, nsamps: int, beam_stride_bytes: int,
                           mean_ptr, sigma_ptr, nsigma: float, counts_ptr, stream: int = 0) -> None:
    """Per-sample number of LOCAL beams above threshold (uint8): the per-GPU half of the coincidence test."""
    st = lib().dedisp_rfi_beam_counts(_ptr(x_ptr), x_dtype, nbeams, nseries, nsamps, beam_stride_bytes,
                                      _ptr(mean_ptr), _ptr(sigma_ptr), nsigma, _ptr(counts_ptr), stream or None)
    _check(None, st, "dedisp_rfi_beam_counts")


def dedisp_rfi_mask_from_counts(counts_ptr, nseries: int, nsamps: int, min_beams: int, mask_ptr, stream: int = 0) -> None:
    st = lib().dedisp_rfi_mask_from_counts(_ptr(counts_ptr), nseries, nsamps, min_beams, _ptr(mask_ptr), stream or None)
    _check(None, st, "dedisp_rfi_mask_from_counts")


def dedisp_veto_events(events_ptr, count_ptr, max_events: int, mask_ptr, nsamps: int, kept_ptr, stream: int = 0) -> None:
    """Events whose peak sample is masked get series = -1 - series; *kept = events left (include/dedisp.h)."""
    st = lib().dedisp_veto_events(_ptr(events_ptr) if events_ptr is not None else None, _ptr(count_ptr), max_events,
                                  _ptr(mask_ptr), nsamps, _ptr(kept_ptr), stream or None)
    _check(None, st, "dedisp_veto_events")


def dedisp_transpose_time_major(in_ptr, nchans: int, nsamps: int, nbits: int, out_ptr, stream: int = 0) -> None:
    """Telescope-order stream -> channel-major tight rows (include/dedisp.h; row f4)."""
    st = lib().dedisp_transpose_time_major(_ptr(in_ptr), nchans, nsamps, nbits, _ptr(out_ptr), stream or None)
    _check(None, st, "dedisp_transpose_time_major")
