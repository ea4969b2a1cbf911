"""ctypes binding of libtno_mf.so -- argument marshalling only; every step of the search runs in
the library's CUDA kernels (include/tno_mf.h).  torch is used for device memory and streams.

The functions carry the names of the C ABI (tno_mf_create, tno_mf_search, tno_mf_inject,
tno_mf_plan, tno_mf_last_stats, tno_mf_destroy, tno_mf_last_error, tno_mf_version).  There is no
CPU fallback: loading fails loudly if the library is missing and tno_mf_create fails without an
sm_100 device.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtno_mf.so")

TNO_MF_OK, TNO_MF_EINVAL, TNO_MF_ENOMEM, TNO_MF_ECUDA, TNO_MF_EUNSUPPORTED = 0, -1, -2, -3, -4

TRAJ_DTYPE = np.dtype([("vx", np.float32), ("vy", np.float32), ("ax", np.float32), ("ay", np.float32)])
CAND_DTYPE = np.dtype([("snr", np.float32), ("x", np.int32), ("y", np.int32), ("k", np.int32)])
SOURCE_DTYPE = np.dtype([("vx", np.float32), ("vy", np.float32), ("ax", np.float32), ("ay", np.float32),
                         ("x", np.int32), ("y", np.int32), ("amplitude", np.float32)])
assert TRAJ_DTYPE.itemsize == 16 and CAND_DTYPE.itemsize == 16 and SOURCE_DTYPE.itemsize == 28


class tno_mf_config(ctypes.Structure):
    _fields_ = [("device", ctypes.c_int32), ("stream", ctypes.c_void_p), ("topk", ctypes.c_int32),
                ("snr_threshold", ctypes.c_float), ("force_generic", ctypes.c_int32),
                ("record_events", ctypes.c_int32), ("workspace_limit_mb", ctypes.c_int32),
                ("filter", ctypes.c_int32), ("sep_shape", ctypes.c_int32)]


class TnoMfError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__("tno_mf error %d: %s" % (code, text))
        self.code = code


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python paper_2209_09848_b200/build.py` "
            "(nvcc, sm_100a).  There is no CPU fallback." % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_float
    lib.tno_mf_create.restype = ctypes.c_int
    lib.tno_mf_create.argtypes = [ctypes.POINTER(tno_mf_config), ctypes.POINTER(vp)]
    lib.tno_mf_search.restype = ctypes.c_int
    lib.tno_mf_search.argtypes = [vp, vp, i32, i32, i32, vp, vp, i32, f32, f32, vp, vp]
    lib.tno_mf_search_ex.restype = ctypes.c_int
    lib.tno_mf_search_ex.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, vp, i32, f32, f32, vp, vp]
    lib.tno_mf_search_masked.restype = ctypes.c_int
    lib.tno_mf_search_masked.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, i32, f32, f32, vp, vp]
    lib.tno_mf_search_host.restype = ctypes.c_int
    lib.tno_mf_search_max.restype = i32
    lib.tno_mf_search_max.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, i32, f32, f32, vp, vp, vp, vp]
    lib.tno_mf_search_host.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, vp, i32, f32, f32, vp, vp]
    lib.tno_mf_search_host_max.restype = i32
    lib.tno_mf_search_host_max.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, i32, f32, f32, vp, vp, vp, vp]
    lib.tno_mf_background.restype = ctypes.c_int
    lib.tno_mf_background.argtypes = [vp, vp, i32, i32, i32, vp, f32, i32, vp, vp]
    lib.tno_mf_flux.restype = ctypes.c_int
    lib.tno_mf_flux.argtypes = [vp, vp, i32, i32, i32, vp]
    lib.tno_mf_best.restype = ctypes.c_int
    lib.tno_mf_best.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, vp]
    lib.tno_mf_local_z_static.restype = ctypes.c_int
    lib.tno_mf_local_z_static.argtypes = [vp, vp, i32, i32, i32, vp]
    lib.tno_mf_debug_poison_shared.restype = ctypes.c_int
    lib.tno_mf_debug_poison_shared.argtypes = [vp, ctypes.c_uint32]
    lib.tno_mf_inject.restype = ctypes.c_int
    lib.tno_mf_inject.argtypes = [vp, vp, i32, i32, i32, vp, i32, f32, f32]
    lib.tno_mf_inject_ex.restype = ctypes.c_int
    lib.tno_mf_inject_ex.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, i32, f32, f32]
    f64p = ctypes.POINTER(ctypes.c_double)
    i32p = ctypes.POINTER(i32)
    lib.tno_mf_scatter_lossgrad.restype = i32
    lib.tno_mf_scatter_lossgrad.argtypes = [vp, vp, i32, i32, i32, vp, f32, vp, vp, f64p, vp, vp]
    lib.tno_mf_scatter_fit.restype = i32
    lib.tno_mf_scatter_fit.argtypes = [vp, vp, i32, i32, i32, vp, f32, i32, f32, vp, vp, f64p, i32p, i32p]
    lib.tno_mf_downsample.restype = i32
    lib.tno_mf_downsample.argtypes = [vp, vp, i32, i32, i32, i32, vp]
    lib.tno_mf_scatter_subtract.restype = i32
    lib.tno_mf_scatter_subtract.argtypes = [vp, vp, i32, i32, i32, vp, i32]
    lib.tno_mf_peaks.restype = i32
    lib.tno_mf_peaks.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    lib.tno_mf_set_prf_table.restype = i32
    lib.tno_mf_set_prf_table.argtypes = [vp, vp, i32]
    lib.tno_mf_set_prf_table2d.restype = i32
    lib.tno_mf_set_prf_table2d.argtypes = [vp, vp, i32, i32]
    lib.tno_mf_plan.restype = ctypes.c_int
    lib.tno_mf_plan.argtypes = [vp, i32, i32, f32, i32, i32, vp, vp]
    lib.tno_mf_plan_slots.restype = ctypes.c_int
    lib.tno_mf_plan_slots.argtypes = [vp, i32, i32, f32, vp, vp, i32, i32, vp, vp, vp]
    lib.tno_mf_last_stats.restype = ctypes.c_int
    lib.tno_mf_last_stats.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i32)]
    lib.tno_mf_last_kernel_ms.restype = ctypes.c_int
    lib.tno_mf_last_kernel_ms.argtypes = [vp, ctypes.POINTER(f32)]
    lib.tno_mf_last_work.restype = ctypes.c_int
    lib.tno_mf_last_work.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                     ctypes.POINTER(ctypes.c_double)]
    lib.tno_mf_destroy.restype = ctypes.c_int
    lib.tno_mf_destroy.argtypes = [vp]
    lib.tno_mf_last_error.restype = ctypes.c_char_p
    lib.tno_mf_last_error.argtypes = [vp]
    lib.tno_mf_version.restype = ctypes.c_char_p
    lib.tno_mf_version.argtypes = []
    return lib


_lib = _load()
_CTX_TOPK = {}          # context handle -> its topk (create-time config), for the size checks of out_topk buffers


def _check(rc: int, ctx) -> None:
    if rc != 0:
        raise TnoMfError(rc, _lib.tno_mf_last_error(ctx).decode())


def tno_mf_version() -> str:
    return _lib.tno_mf_version().decode()


def tno_mf_last_error(ctx=None) -> str:
    return _lib.tno_mf_last_error(ctx).decode()


def tno_mf_create(device: int = 0, stream: Optional[int] = None, topk: int = 0,
                  snr_threshold: float = float("-inf"), force_generic: bool = False,
                  record_events: bool = False, workspace_limit_mb: int = 0, shift_stack: bool = False,
                  filter: int = 0, sep_shape: int = 0):
    """Returns an opaque context handle.  `stream` is a raw cudaStream_t (int) or None."""
    cfg = tno_mf_config(device=int(device), stream=ctypes.c_void_p(stream or 0), topk=int(topk),
                        snr_threshold=float(snr_threshold), force_generic=int(bool(force_generic)),
                        record_events=int(bool(record_events)), workspace_limit_mb=int(workspace_limit_mb),
                        filter=int(filter) if filter else int(bool(shift_stack)), sep_shape=int(sep_shape))
    ctx = ctypes.c_void_p()
    _check(_lib.tno_mf_create(ctypes.byref(cfg), ctypes.byref(ctx)), None)
    _CTX_TOPK[ctx.value] = int(topk)            # the binding checks the size of out_topk buffers against it
    return ctx


def tno_mf_destroy(ctx) -> None:
    _CTX_TOPK.pop(ctx.value, None)
    _check(_lib.tno_mf_destroy(ctx), None)


def _traj_array(trajectories) -> np.ndarray:
    a = np.ascontiguousarray(trajectories, dtype=np.float32)
    if a.ndim != 2 or a.shape[1] != 4:
        raise ValueError("trajectories must be [n, 4] (vx, vy, ax, ay)")
    return a


def tno_mf_search(ctx, frames, sigma_t, trajectories, prf_sigma: float, t0: float,
                  out_snr=None, out_topk=None) -> None:
    """frames: CUDA float32 tensor [T, H, W] (contiguous); sigma_t: host float32 [T];
    trajectories: host [n, 4]; out_snr: CUDA float32 tensor [n, H, W] or None; out_topk: CUDA
    uint8/int32 tensor with n*topk*16 bytes or None.  Enqueues on the context's stream."""
    tno_mf_search_ex(ctx, frames, sigma_t, None, None, trajectories, prf_sigma, t0, out_snr, out_topk,
                     _plain=True)


def tno_mf_search_masked(ctx, frames, valid, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma: float,
                         t0: float, out_snr=None, out_topk=None) -> None:
    """tno_mf_search_ex with per-pixel validity weights (CUDA float32 tensor shaped like frames, or None)."""
    tno_mf_search_ex(ctx, frames, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma, t0, out_snr, out_topk,
                     _valid=valid)


def tno_mf_search_max(ctx, frames, valid, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma: float, t0: float,
                      out_max, out_argk=None, out_snr=None, out_topk=None) -> None:
    """The search with the max over the bank fused in: out_max CUDA float32 [H, W] (required), out_argk CUDA int32
    [H, W] or None; valid, out_snr, out_topk optional."""
    T, H, W = frames.shape
    assert out_max.is_cuda and out_max.is_contiguous() and tuple(out_max.shape) == (H, W) and out_max.element_size() == 4
    assert out_argk is None or (out_argk.is_cuda and out_argk.is_contiguous() and tuple(out_argk.shape) == (H, W)
                                and out_argk.element_size() == 4)
    tno_mf_search_ex(ctx, frames, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma, t0, out_snr, out_topk,
                     _valid=valid, _max=(out_max, out_argk))


def tno_mf_search_ex(ctx, frames, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma: float, t0: float,
                     out_snr=None, out_topk=None, _plain: bool = False, _valid=None, _max=None) -> None:
    """tno_mf_search with frame times (host float32 [T] or None) and pointing jitter (host float32
    [T, 2] px or None) in the track."""
    assert frames.is_cuda and frames.dtype.is_floating_point and frames.element_size() == 4
    assert frames.is_contiguous() and frames.dim() == 3
    T, H, W = frames.shape
    sig = np.ascontiguousarray(sigma_t, dtype=np.float32)
    if sig.shape != (T,):
        raise ValueError("sigma_t must have shape [T]")
    tm = jt = None
    if frame_times is not None:
        tm = np.ascontiguousarray(frame_times, dtype=np.float32)
        if tm.shape != (T,):
            raise ValueError("frame_times must have shape [T]")
    if jitter_xy is not None:
        jt = np.ascontiguousarray(jitter_xy, dtype=np.float32)
        if jt.shape != (T, 2):
            raise ValueError("jitter_xy must have shape [T, 2]")
    tr = _traj_array(trajectories)
    n = tr.shape[0]
    p_snr = None
    if out_snr is not None:
        assert out_snr.is_cuda and out_snr.is_contiguous() and out_snr.element_size() == 4
        assert out_snr.numel() == n * H * W
        p_snr = out_snr.data_ptr()
    p_top = None
    if out_topk is not None:
        assert out_topk.is_cuda and out_topk.is_contiguous()
        assert out_topk.numel() * out_topk.element_size() >= n * _CTX_TOPK.get(ctx.value, 0) * 16, \
            "out_topk is smaller than [n][topk] records of 16 bytes"
        p_top = out_topk.data_ptr()
    if _valid is not None:
        assert _valid.is_cuda and _valid.is_contiguous() and _valid.shape == frames.shape
        assert _valid.element_size() == 4 and _valid.dtype.is_floating_point
    if _max is not None:
        rc = _lib.tno_mf_search_max(ctx, frames.data_ptr(), _valid.data_ptr() if _valid is not None else None, T, H, W,
                                    sig.ctypes.data, tm.ctypes.data if tm is not None else None,
                                    jt.ctypes.data if jt is not None else None, tr.ctypes.data, n,
                                    float(prf_sigma), float(t0), _max[0].data_ptr(),
                                    _max[1].data_ptr() if _max[1] is not None else None, p_snr, p_top)
    elif _valid is not None:
        rc = _lib.tno_mf_search_masked(ctx, frames.data_ptr(), _valid.data_ptr(), T, H, W, sig.ctypes.data,
                                       tm.ctypes.data if tm is not None else None,
                                       jt.ctypes.data if jt is not None else None, tr.ctypes.data, n,
                                       float(prf_sigma), float(t0), p_snr, p_top)
    elif _plain:
        rc = _lib.tno_mf_search(ctx, frames.data_ptr(), T, H, W, sig.ctypes.data, tr.ctypes.data, n,
                                float(prf_sigma), float(t0), p_snr, p_top)
    else:
        rc = _lib.tno_mf_search_ex(ctx, frames.data_ptr(), T, H, W, sig.ctypes.data,
                                   tm.ctypes.data if tm is not None else None,
                                   jt.ctypes.data if jt is not None else None, tr.ctypes.data, n,
                                   float(prf_sigma), float(t0), p_snr, p_top)
    _check(rc, ctx)


def _host_ptr(a, shape, dtype_size, what):
    """Address of a HOST buffer (torch CPU tensor or ndarray) after checking contiguity, placement and size."""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):
        assert not a.is_cuda, what + " must be in host memory"
        assert a.is_contiguous(), what + " must be contiguous"
        nbytes, ptr = a.numel() * a.element_size(), a.data_ptr()
    else:
        assert a.flags.c_contiguous, what + " must be contiguous"
        nbytes, ptr = a.nbytes, a.ctypes.data
    need = int(np.prod(shape)) * dtype_size
    assert nbytes >= need, "%s holds %d bytes, %d needed" % (what, nbytes, need)
    return ptr


def tno_mf_search_host_max(ctx, frames, valid, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma: float,
                           t0: float, out_max=None, out_argk=None, out_snr=None, out_topk=None) -> None:
    """frames (and valid or None): HOST float32 tensors or ndarrays [T, H, W] (contiguous; pinned for overlap);
    out_max float32 / out_argk int32: HOST [H, W] or None; out_snr: HOST float32 [n, H, W] or None; out_topk: HOST
    buffer of n*topk*16 bytes or None.  Returns when the results are in the host buffers."""
    T, H, W = frames.shape
    sig = np.ascontiguousarray(sigma_t, dtype=np.float32)
    tm = None if frame_times is None else np.ascontiguousarray(frame_times, dtype=np.float32)
    jt = None if jitter_xy is None else np.ascontiguousarray(jitter_xy, dtype=np.float32)
    assert sig.shape == (T,) and (tm is None or tm.shape == (T,)) and (jt is None or jt.shape == (T, 2))
    tr = _traj_array(trajectories)
    n = tr.shape[0]
    assert valid is None or tuple(valid.shape) == (T, H, W)
    for a in (frames, valid, out_max, out_snr):
        assert a is None or (a.element_size() if hasattr(a, "element_size") else a.itemsize) == 4
    _check(_lib.tno_mf_search_host_max(
        ctx, _host_ptr(frames, (T, H, W), 4, "frames"), _host_ptr(valid, (T, H, W), 4, "valid"), T, H, W,
        sig.ctypes.data, tm.ctypes.data if tm is not None else None, jt.ctypes.data if jt is not None else None,
        tr.ctypes.data, n, float(prf_sigma), float(t0),
        _host_ptr(out_max, (H, W), 4, "out_max"), _host_ptr(out_argk, (H, W), 4, "out_argk"),
        _host_ptr(out_snr, (n, H, W), 4, "out_snr"),
        _host_ptr(out_topk, (n, _CTX_TOPK.get(ctx.value, 0)), 16, "out_topk")), ctx)


def tno_mf_search_host(ctx, frames, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma: float, t0: float,
                       out_snr=None, out_topk=None) -> None:
    """frames: HOST float32 tensor or ndarray [T, H, W] (contiguous; pinned for overlap); out_snr: HOST float32
    [n, H, W] or None; out_topk: HOST buffer of n*topk*16 bytes or None.  Returns when the results are in."""
    T, H, W = frames.shape
    sig = np.ascontiguousarray(sigma_t, dtype=np.float32)
    tm = None if frame_times is None else np.ascontiguousarray(frame_times, dtype=np.float32)
    jt = None if jitter_xy is None else np.ascontiguousarray(jitter_xy, dtype=np.float32)
    assert sig.shape == (T,) and (tm is None or tm.shape == (T,)) and (jt is None or jt.shape == (T, 2))
    tr = _traj_array(trajectories)
    n = tr.shape[0]
    assert (frames.element_size() if hasattr(frames, "element_size") else frames.itemsize) == 4
    _check(_lib.tno_mf_search_host(ctx, _host_ptr(frames, (T, H, W), 4, "frames"), T, H, W, sig.ctypes.data,
                                   tm.ctypes.data if tm is not None else None,
                                   jt.ctypes.data if jt is not None else None, tr.ctypes.data, n,
                                   float(prf_sigma), float(t0), _host_ptr(out_snr, (n, H, W), 4, "out_snr"),
                                   _host_ptr(out_topk, (n, _CTX_TOPK.get(ctx.value, 0)), 16, "out_topk")), ctx)


def tno_mf_background(ctx, frames, jitter_xy, delta: float, n_iter: int, out_coef=None, out_resid=None) -> None:
    """frames: CUDA float32 [T, H, W]; jitter_xy: host [T, 2]; out_coef: CUDA float32 [6, H, W] or None;
    out_resid: CUDA float32 [T, H, W] (may be `frames`) or None.  PAPER.md section 3.1."""
    assert frames.is_cuda and frames.is_contiguous() and frames.dim() == 3 and frames.element_size() == 4
    T, H, W = frames.shape
    jt = np.ascontiguousarray(jitter_xy, dtype=np.float32)
    assert jt.shape == (T, 2)
    for t, shp in ((out_coef, (6, H, W)), (out_resid, (T, H, W))):
        assert t is None or (t.is_cuda and t.is_contiguous() and tuple(t.shape) == shp and t.element_size() == 4)
    _check(_lib.tno_mf_background(ctx, frames.data_ptr(), T, H, W, jt.ctypes.data, float(delta), int(n_iter),
                                  out_coef.data_ptr() if out_coef is not None else None,
                                  out_resid.data_ptr() if out_resid is not None else None), ctx)


def tno_mf_flux(ctx, snr, out_flux) -> None:
    """snr, out_flux: CUDA float32 tensors [n, H, W]; flux estimate N / D of the last search's maps."""
    assert snr.is_cuda and snr.is_contiguous() and snr.dim() == 3 and snr.element_size() == 4
    assert out_flux.is_cuda and out_flux.is_contiguous() and out_flux.shape == snr.shape
    n, H, W = snr.shape
    _check(_lib.tno_mf_flux(ctx, snr.data_ptr(), n, H, W, out_flux.data_ptr()), ctx)


def tno_mf_best(ctx, snr, box: int, out_max, out_argk=None, out_z=None, out_topk=None) -> None:
    """snr: CUDA float32 tensor [n, H, W]; out_max / out_z: CUDA float32 [H, W]; out_argk: CUDA int32
    [H, W]; out_topk: CUDA tensor with topk*16 bytes.  Enqueues on the context's stream."""
    assert snr.is_cuda and snr.is_contiguous() and snr.dim() == 3 and snr.element_size() == 4
    n, H, W = snr.shape
    ptrs = []
    for t, es in ((out_max, 4), (out_argk, 4), (out_z, 4)):
        if t is None:
            ptrs.append(None)
            continue
        assert t.is_cuda and t.is_contiguous() and t.element_size() == es and t.numel() == H * W
        ptrs.append(t.data_ptr())
    p_top = None
    if out_topk is not None:
        assert out_topk.is_cuda and out_topk.is_contiguous()
        assert out_topk.numel() * out_topk.element_size() >= 1 * _CTX_TOPK.get(ctx.value, 0) * 16, \
            "out_topk is smaller than [n][topk] records of 16 bytes"
        p_top = out_topk.data_ptr()
    _check(_lib.tno_mf_best(ctx, snr.data_ptr(), n, H, W, int(box), ptrs[0], ptrs[1], ptrs[2], p_top), ctx)


def tno_mf_local_z_static(ctx, score, box: int, out_z) -> None:
    """score, out_z: CUDA float32 tensors [H, W] with H * W <= 2**20 (the library's static scratch).  No device
    allocation; enqueues on the context's stream.  Calls that overlap on the GPU share the scratch and race."""
    assert score.is_cuda and score.is_contiguous() and score.dim() == 2 and score.element_size() == 4
    H, W = score.shape
    assert out_z.is_cuda and out_z.is_contiguous() and out_z.element_size() == 4 and out_z.numel() == H * W
    _check(_lib.tno_mf_local_z_static(ctx, score.data_ptr(), H, W, int(box), out_z.data_ptr()), ctx)


def tno_mf_debug_poison_shared(ctx, pattern: int = 0xFFFFFFFF) -> None:
    """Fill the shared memory of every SM with `pattern` (default: a NaN as a float); see include/tno_mf.h."""
    _check(_lib.tno_mf_debug_poison_shared(ctx, int(pattern) & 0xFFFFFFFF), ctx)


def tno_mf_inject(ctx, frames, sources: np.ndarray, prf_sigma: float, t0: float) -> None:
    """frames: CUDA float32 tensor [T, H, W], modified in place; sources: SOURCE_DTYPE array."""
    assert frames.is_cuda and frames.is_contiguous() and frames.dim() == 3 and frames.element_size() == 4
    T, H, W = frames.shape
    src = np.ascontiguousarray(sources, dtype=SOURCE_DTYPE)
    _check(_lib.tno_mf_inject(ctx, frames.data_ptr(), T, H, W, src.ctypes.data, src.shape[0],
                              float(prf_sigma), float(t0)), ctx)


def tno_mf_inject_ex(ctx, frames, frame_times, jitter_xy, sources: np.ndarray, prf_sigma: float, t0: float) -> None:
    """tno_mf_inject with frame times (host [T] or None) and pointing jitter (host [T, 2] or None) in the track."""
    assert frames.is_cuda and frames.is_contiguous() and frames.dim() == 3 and frames.element_size() == 4
    T, H, W = frames.shape
    src = np.ascontiguousarray(sources, dtype=SOURCE_DTYPE)
    tm = None if frame_times is None else np.ascontiguousarray(frame_times, dtype=np.float32)
    jt = None if jitter_xy is None else np.ascontiguousarray(jitter_xy, dtype=np.float32)
    assert (tm is None or tm.shape == (T,)) and (jt is None or jt.shape == (T, 2))
    _check(_lib.tno_mf_inject_ex(ctx, frames.data_ptr(), T, H, W, tm.ctypes.data if tm is not None else None,
                                 jt.ctypes.data if jt is not None else None, src.ctypes.data, src.shape[0],
                                 float(prf_sigma), float(t0)), ctx)


def _dev3(t, shape=None):
    assert t.is_cuda and t.is_contiguous() and t.dim() == 3 and t.element_size() == 4 and t.dtype.is_floating_point
    assert shape is None or tuple(t.shape) == tuple(shape), (tuple(t.shape), shape)
    return t.data_ptr()


def _jitter(jitter_xy, T):
    jt = np.ascontiguousarray(jitter_xy, dtype=np.float32)
    if jt.shape != (T, 2):
        raise ValueError("jitter_xy must have shape [T, 2]")
    return jt


def tno_mf_scatter_lossgrad(ctx, D, jitter_xy, delta: float, beta, S, g_beta, g_S) -> float:
    """D [T, N, N], beta / g_beta [6, N, N], S / g_S [T, n, n]: CUDA float32 tensors.  Returns the loss."""
    T, N, _ = D.shape
    n = S.shape[-1]
    jt = _jitter(jitter_xy, T)
    loss = ctypes.c_double()
    _check(_lib.tno_mf_scatter_lossgrad(ctx, _dev3(D, (T, N, N)), T, N, n, jt.ctypes.data, float(delta),
                                        _dev3(beta, (6, N, N)), _dev3(S, (T, n, n)), ctypes.byref(loss),
                                        _dev3(g_beta, (6, N, N)), _dev3(g_S, (T, n, n))), ctx)
    return loss.value


def tno_mf_scatter_fit(ctx, D, jitter_xy, delta: float, max_iter: int, gtol: float, beta, S) -> Tuple[float, int, int]:
    """L-BFGS from (beta, S), overwritten with the minimiser.  Returns (loss, iterations, loss evaluations)."""
    T, N, _ = D.shape
    n = S.shape[-1]
    jt = _jitter(jitter_xy, T)
    loss, iters, evals = ctypes.c_double(), ctypes.c_int32(), ctypes.c_int32()
    _check(_lib.tno_mf_scatter_fit(ctx, _dev3(D, (T, N, N)), T, N, n, jt.ctypes.data, float(delta), int(max_iter),
                                   float(gtol), _dev3(beta, (6, N, N)), _dev3(S, (T, n, n)), ctypes.byref(loss),
                                   ctypes.byref(iters), ctypes.byref(evals)), ctx)
    return loss.value, iters.value, evals.value


def tno_mf_downsample(ctx, frames, factor: int, out) -> None:
    T, H, W = frames.shape
    _check(_lib.tno_mf_downsample(ctx, _dev3(frames), T, H, W, int(factor),
                                  _dev3(out, (T, H // factor, W // factor))), ctx)


def tno_mf_scatter_subtract(ctx, frames, S) -> None:
    T, H, W = frames.shape
    n = S.shape[-1]
    _check(_lib.tno_mf_scatter_subtract(ctx, _dev3(frames), T, H, W, _dev3(S, (T, n, n)), n), ctx)


def tno_mf_peaks(ctx, score, argk, radius: int, out_peaks, out_topk) -> None:
    """score: CUDA float32 [H, W]; argk: CUDA int32 [H, W] or None; out_peaks: CUDA float32 [H, W] or None;
    out_topk: CUDA int32 [topk, 4] or None."""
    assert score.is_cuda and score.is_contiguous() and score.dim() == 2 and score.element_size() == 4
    H, W = score.shape
    for t in (argk, out_peaks):
        assert t is None or (t.is_cuda and t.is_contiguous() and tuple(t.shape) == (H, W) and t.element_size() == 4)
    assert out_topk is None or (out_topk.is_cuda and out_topk.is_contiguous() and
                                out_topk.numel() * out_topk.element_size() >= _CTX_TOPK.get(ctx.value, 0) * 16)
    _check(_lib.tno_mf_peaks(ctx, score.data_ptr(), argk.data_ptr() if argk is not None else None, H, W, int(radius),
                             out_peaks.data_ptr() if out_peaks is not None else None,
                             out_topk.data_ptr() if out_topk is not None else None), ctx)


def tno_mf_set_prf_table(ctx, table) -> None:
    """table: [n_phase, 5] flux fractions (host array) for filter 3; None or an empty table removes it."""
    if table is None or len(table) == 0:
        _check(_lib.tno_mf_set_prf_table(ctx, None, 0), ctx)
        return
    tab = np.ascontiguousarray(table, dtype=np.float32)
    if tab.ndim != 2 or tab.shape[1] != 5:
        raise ValueError("prf table must have shape [n_phase, 5]")
    _check(_lib.tno_mf_set_prf_table(ctx, tab.ctypes.data, tab.shape[0]), ctx)


def tno_mf_set_prf_table2d(ctx, table) -> None:
    """table: [n_phase_y, n_phase_x, 5, 5] responses (host array) for filter 4; None removes it."""
    if table is None or len(table) == 0:
        _check(_lib.tno_mf_set_prf_table2d(ctx, None, 0, 0), ctx)
        return
    tab = np.ascontiguousarray(table, dtype=np.float32)
    if tab.ndim != 4 or tab.shape[2:] != (5, 5):
        raise ValueError("prf table must have shape [n_phase_y, n_phase_x, 5, 5]")
    _check(_lib.tno_mf_set_prf_table2d(ctx, tab.ctypes.data, tab.shape[0], tab.shape[1]), ctx)


def tno_mf_plan(trajectories, T: int, t0: float, max_entries: int, max_spread: int
                ) -> Tuple[int, np.ndarray, np.ndarray]:
    """Host-only: (n_batches, batch index per trajectory, slot per trajectory)."""
    tr = _traj_array(trajectories)
    n = tr.shape[0]
    ob = np.full(n, -1, dtype=np.int32)
    os_ = np.full(n, -1, dtype=np.int32)
    rc = _lib.tno_mf_plan(tr.ctypes.data, n, int(T), float(t0), int(max_entries), int(max_spread),
                          ob.ctypes.data, os_.ctypes.data)
    if rc < 0:
        raise TnoMfError(rc, "tno_mf_plan: invalid argument")
    return rc, ob, os_


def tno_mf_plan_slots(trajectories, T: int, t0: float, max_slots: int = 5, symmetric_filter: bool = True,
                      frame_times=None, jitter_xy=None) -> Tuple[int, np.ndarray, np.ndarray, np.ndarray]:
    """(number of batches, batch [n], slot [n], member [n]) of the separable kernel's slot packing (host only)."""
    tr = _traj_array(trajectories)
    n = tr.shape[0]
    tm = None if frame_times is None else np.ascontiguousarray(frame_times, dtype=np.float32)
    jt = None if jitter_xy is None else np.ascontiguousarray(jitter_xy, dtype=np.float32)
    assert (tm is None or tm.shape == (T,)) and (jt is None or jt.shape == (T, 2))
    batch, slot, member = (np.full(n, -1, dtype=np.int32) for _ in range(3))
    rc = _lib.tno_mf_plan_slots(tr.ctypes.data, n, int(T), float(t0), tm.ctypes.data if tm is not None else None,
                                jt.ctypes.data if jt is not None else None, int(max_slots),
                                int(bool(symmetric_filter)), batch.ctypes.data, slot.ctypes.data, member.ctypes.data)
    if rc < 0:
        raise TnoMfError(rc, "tno_mf_plan_slots: invalid arguments")
    return rc, batch, slot, member


def tno_mf_last_stats(ctx) -> Tuple[int, int]:
    """(kernel launches of the last search, 1 if the separable TMA kernel was used else 0)."""
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(_lib.tno_mf_last_stats(ctx, ctypes.byref(a), ctypes.byref(b)), None)
    return a.value, b.value


def tno_mf_last_kernel_ms(ctx) -> float:
    """Duration (ms) of the main search kernel of the last search (needs record_events)."""
    ms = ctypes.c_float()
    _check(_lib.tno_mf_last_kernel_ms(ctx, ctypes.byref(ms)), ctx)
    return ms.value


def tno_mf_last_work(ctx) -> Tuple[float, float, float]:
    """(x-pass multiply-adds, y-pass multiply-adds, y-pass additions) of the formulation the last search executed."""
    a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(_lib.tno_mf_last_work(ctx, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), None)
    return a.value, b.value, c.value


def make_sources(trajs, xs, ys, amps) -> np.ndarray:
    """Pack per-source arrays into SOURCE_DTYPE records."""
    tr = _traj_array(trajs)
    out = np.zeros(tr.shape[0], dtype=SOURCE_DTYPE)
    out["vx"], out["vy"], out["ax"], out["ay"] = tr[:, 0], tr[:, 1], tr[:, 2], tr[:, 3]
    out["x"], out["y"], out["amplitude"] = xs, ys, amps
    return out
