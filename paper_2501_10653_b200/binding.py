"""ctypes binding over libiqa_tiles.so (include/iqa_tiles.h) -- argument marshalling only.

Two layers, both without any arithmetic of the method:
  * ``iqa_*`` functions with the C names and argument order of the header.  Pointer
    arguments accept a torch tensor (its ``data_ptr()``), a numpy array (host entry points),
    an int address or None; ``stream`` accepts a ``torch.cuda.Stream``, an int handle or None.
    They return the ``iqa_status`` code.
  * convenience wrappers (``fused_tiles``, ``lisi_tiles``, ``auglisi_tiles``, ``aggregate``,
    ``merge_tiles``, ``pyramid``, ``fused_host``) that allocate the output tensors with torch,
    use torch's current stream, and raise ``IqaError`` on a non-zero status.

Importing this module FAILS when the library is missing and cannot be built with nvcc:
there is no CPU fallback (the CPU oracle under ``oracle/`` is test infrastructure only and
is never imported from here).
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

IQA_OK, IQA_ERR_NULL, IQA_ERR_SHAPE, IQA_ERR_PARAM, IQA_ERR_ALIGN, IQA_ERR_WORKSPACE, IQA_ERR_CUDA = range(7)
IQA_ERR_STATIC_LIMIT = 7
IQA_STATIC_WORKSPACE_BYTES = 1 << 20     # include/iqa_tiles.h; tests/test_zz_no_alloc.py checks the two agree

EXPORTS = ("iqa_status_string", "iqa_version", "iqa_debug_knob", "iqa_workspace_bytes", "iqa_lisi_tiles",
           "iqa_auglisi_tiles", "iqa_fused_tiles", "iqa_fused_tiles_static", "iqa_batch_workspace_bytes", "iqa_fused_batch",
           "iqa_query_plan", "iqa_query_plan_n", "iqa_workspace_bytes_2d", "iqa_fused_tiles_2d", "iqa_fused_tiles_2d_typed",
           "iqa_fused_batch_2d", "iqa_fused_batch_2d_typed", "iqa_series_tiles_2d", "iqa_series_tiles_2d_typed",
           "iqa_series_workspace_bytes", "iqa_series_tiles", "iqa_series_find", "iqa_series_find_2d_typed", "iqa_tiles_below", "iqa_tiles_bottom_k",
           "iqa_aggregate", "iqa_aggregate_partial", "iqa_aggregate_finish", "iqa_merge_tiles", "iqa_merge_tiles_batch",
           "iqa_pyramid_levels", "iqa_pyramid_tiles", "iqa_pyramid",
           "iqa_host_scratch_bytes", "iqa_fused_host", "iqa_fused_host_async",
           "iqa_host_scratch_bytes_typed", "iqa_fused_host_typed", "iqa_fused_host_typed_async")

IQA_SERIES_REFERENCE, IQA_SERIES_CONSECUTIVE = 0, 1
IQA_PIXEL_F32, IQA_PIXEL_F64, IQA_PIXEL_F16, IQA_PIXEL_I16, IQA_PIXEL_I32, IQA_PIXEL_U8 = range(6)
SERIES_MODES = {"reference": IQA_SERIES_REFERENCE, "consecutive": IQA_SERIES_CONSECUTIVE}


class IqaError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        super().__init__(f"{where}: iqa_status {status} ({iqa_status_string(status)})")


STALE = False      # True when an out-of-date libiqa_tiles.so had to be loaded because no nvcc is available


def _load() -> ctypes.CDLL:
    global STALE
    try:
        path = _build.build()
    except _build.NoCompiler as exc:   # no nvcc on this machine: a prebuilt library may stand in, and says so
        if not os.path.exists(_build.LIB):
            raise ImportError(
                "libiqa_tiles.so is not built and nvcc could not build it "
                f"({exc}); run `python -m paper_2501_10653_b200.build`. There is no CPU fallback.") from exc
        import warnings
        warnings.warn("libiqa_tiles.so is older than its sources and nvcc is not available: loading the stale library")
        STALE = True
        path = _build.LIB
    # a compile error is never swallowed: results must describe the sources in the tree
    lib = ctypes.CDLL(path)
    vp, f, i, sz = ctypes.c_void_p, ctypes.c_float, ctypes.c_int, ctypes.c_size_t
    lib.iqa_status_string.restype = ctypes.c_char_p
    lib.iqa_status_string.argtypes = [i]
    lib.iqa_version.restype = ctypes.c_char_p
    lib.iqa_version.argtypes = []
    lib.iqa_workspace_bytes.restype = sz
    lib.iqa_workspace_bytes.argtypes = [i, i]
    lib.iqa_host_scratch_bytes.restype = sz
    lib.iqa_host_scratch_bytes.argtypes = [i, i]
    lib.iqa_lisi_tiles.restype = i
    lib.iqa_lisi_tiles.argtypes = [vp, vp, i, i, f, f, f, vp, vp, sz, vp]
    lib.iqa_auglisi_tiles.restype = i
    lib.iqa_auglisi_tiles.argtypes = [vp, vp, i, i, f, vp, vp, sz, vp]
    lib.iqa_fused_tiles.restype = i
    lib.iqa_fused_tiles.argtypes = [vp, vp, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_fused_tiles_static.restype = i
    lib.iqa_fused_tiles_static.argtypes = [vp, vp, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, vp]
    lib.iqa_batch_workspace_bytes.restype = sz
    lib.iqa_batch_workspace_bytes.argtypes = [i, i, i]
    lib.iqa_fused_batch.restype = i
    lib.iqa_fused_batch.argtypes = [vp, vp, i, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_series_workspace_bytes.restype = sz
    lib.iqa_series_workspace_bytes.argtypes = [i, i, i]
    lib.iqa_series_tiles.restype = i
    lib.iqa_series_tiles.argtypes = [vp, i, i, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_series_find.restype = i
    lib.iqa_series_find.argtypes = [vp, i, i, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, vp, vp, sz,
                                    i, i, vp, vp, f, vp, i, vp, vp]
    lib.iqa_series_find_2d_typed.restype = i
    lib.iqa_series_find_2d_typed.argtypes = [vp, i, i, i, i, i, ctypes.c_longlong, i, f, f, f, f,
                                             vp, vp, vp, vp, vp, vp, vp, vp, sz, i, i, vp, vp, f, vp, i, vp, vp]
    lib.iqa_query_plan.restype = i
    lib.iqa_query_plan.argtypes = [vp, i, i, i, ctypes.c_longlong, i, i]
    lib.iqa_query_plan_n.restype = i
    lib.iqa_query_plan_n.argtypes = [vp, i, i, i, ctypes.c_longlong, i, i, i]
    lib.iqa_debug_knob.restype = i
    lib.iqa_debug_knob.argtypes = [ctypes.c_char_p, i]
    lib.iqa_fused_batch_2d_typed.restype = i
    lib.iqa_fused_batch_2d_typed.argtypes = [vp, vp, i, i, i, i, ctypes.c_longlong, i, f, f, f, f,
                                             vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_series_tiles_2d_typed.restype = i
    lib.iqa_series_tiles_2d_typed.argtypes = [vp, i, i, i, i, i, ctypes.c_longlong, i, f, f, f, f,
                                              vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_workspace_bytes_2d.restype = sz
    lib.iqa_workspace_bytes_2d.argtypes = [i, i, i]
    lib.iqa_fused_tiles_2d.restype = i
    lib.iqa_fused_tiles_2d.argtypes = [vp, vp, i, i, ctypes.c_longlong, ctypes.c_longlong, i, f, f, f, f,
                                       vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_aggregate_partial.restype = i
    lib.iqa_aggregate_partial.argtypes = [vp, vp, vp, vp, i, f, f, vp, vp]
    lib.iqa_aggregate_finish.restype = i
    lib.iqa_aggregate_finish.argtypes = [vp, ctypes.c_longlong, f, f, vp, vp]
    lib.iqa_fused_tiles_2d_typed.restype = i
    lib.iqa_fused_tiles_2d_typed.argtypes = [vp, vp, i, i, i, ctypes.c_longlong, ctypes.c_longlong, i, f, f, f, f,
                                             vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_fused_batch_2d.restype = i
    lib.iqa_fused_batch_2d.argtypes = [vp, vp, i, i, i, ctypes.c_longlong, i, f, f, f, f,
                                       vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_series_tiles_2d.restype = i
    lib.iqa_series_tiles_2d.argtypes = [vp, i, i, i, i, ctypes.c_longlong, i, f, f, f, f,
                                        vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_tiles_below.restype = i
    lib.iqa_tiles_below.argtypes = [vp, i, i, f, vp, i, vp, vp]
    lib.iqa_tiles_bottom_k.restype = i
    lib.iqa_tiles_bottom_k.argtypes = [vp, i, i, i, vp, vp, vp]
    lib.iqa_aggregate.restype = i
    lib.iqa_aggregate.argtypes = [vp, vp, vp, vp, i, f, f, vp, vp]
    lib.iqa_merge_tiles_batch.restype = i
    lib.iqa_merge_tiles_batch.argtypes = [vp, vp, vp, vp, i, i, i, f, f, vp, vp, vp, vp, vp]
    lib.iqa_merge_tiles.restype = i
    lib.iqa_merge_tiles.argtypes = [vp, vp, vp, vp, i, i, f, f, vp, vp, vp, vp, vp]
    lib.iqa_pyramid_levels.restype = i
    lib.iqa_pyramid_levels.argtypes = [i, i]
    lib.iqa_pyramid_tiles.restype = sz
    lib.iqa_pyramid_tiles.argtypes = [i, i]
    lib.iqa_pyramid.restype = i
    lib.iqa_pyramid.argtypes = [vp, vp, vp, vp, i, i, i, f, f, vp, vp, vp, vp, vp]
    lib.iqa_fused_host.restype = i
    lib.iqa_fused_host.argtypes = [vp, vp, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_fused_host_async.restype = i
    lib.iqa_fused_host_async.argtypes = [vp, vp, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_host_scratch_bytes_typed.restype = sz
    lib.iqa_host_scratch_bytes_typed.argtypes = [i, i, i]
    lib.iqa_fused_host_typed.restype = i
    lib.iqa_fused_host_typed.argtypes = [vp, vp, i, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.iqa_fused_host_typed_async.restype = i
    lib.iqa_fused_host_typed_async.argtypes = [vp, vp, i, i, i, f, f, f, f, vp, vp, vp, vp, vp, vp, sz, vp]
    return lib


lib = _load()
LIB_PATH = _build.LIB


# ----------------------------------------------------------------------------- marshalling
def _ptr(a):
    """Address of a tensor / array / int / None as c_void_p-compatible value."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    if hasattr(a, "ctypes"):
        return a.ctypes.data
    raise TypeError(f"cannot take the address of {type(a)!r}")


def _stream(s):
    if s is None:
        return None
    if isinstance(s, int):
        return s
    return s.cuda_stream


def _current_stream(device=None):
    import torch
    return torch.cuda.current_stream(device).cuda_stream


def _device_of(t):
    """Context manager making the device of tensor ``t`` (or a torch.device) current: the library launches on, and
    caches launch geometry for, the CURRENT device, so a call on tensors of another device must switch first."""
    import torch
    return torch.cuda.device(t.device if hasattr(t, "device") else t)


# ----------------------------------------------------------------------------- C names
def iqa_status_string(status: int) -> str:
    return lib.iqa_status_string(int(status)).decode()


def iqa_version() -> str:
    return lib.iqa_version().decode()


def iqa_workspace_bytes(N: int, N_T: int) -> int:
    return int(lib.iqa_workspace_bytes(int(N), int(N_T)))


def iqa_host_scratch_bytes(N: int, N_T: int) -> int:
    return int(lib.iqa_host_scratch_bytes(int(N), int(N_T)))


def iqa_lisi_tiles(x, y, N, N_T, C1, C2, D, lisi, workspace=None, workspace_bytes=0, stream=None) -> int:
    return lib.iqa_lisi_tiles(_ptr(x), _ptr(y), int(N), int(N_T), C1, C2, D, _ptr(lisi),
                              _ptr(workspace), int(workspace_bytes), _stream(stream))


def iqa_auglisi_tiles(x, y, N, N_T, C, auglisi, workspace=None, workspace_bytes=0, stream=None) -> int:
    return lib.iqa_auglisi_tiles(_ptr(x), _ptr(y), int(N), int(N_T), C, _ptr(auglisi),
                                 _ptr(workspace), int(workspace_bytes), _stream(stream))


def iqa_fused_tiles(x, y, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                    lisi_num=None, auglisi_num=None, workspace=None, workspace_bytes=0, stream=None) -> int:
    return lib.iqa_fused_tiles(_ptr(x), _ptr(y), int(N), int(N_T), C1, C2, C, D,
                               _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                               _ptr(lisi_num), _ptr(auglisi_num),
                               _ptr(workspace), int(workspace_bytes), _stream(stream))


def iqa_fused_tiles_static(x, y, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                           lisi_num=None, auglisi_num=None, stream=None) -> int:
    return lib.iqa_fused_tiles_static(_ptr(x), _ptr(y), int(N), int(N_T), C1, C2, C, D,
                                      _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                      _ptr(lisi_num), _ptr(auglisi_num), _stream(stream))


def iqa_batch_workspace_bytes(n_pairs: int, N: int, N_T: int) -> int:
    return int(lib.iqa_batch_workspace_bytes(int(n_pairs), int(N), int(N_T)))


def _ptr_table(images):
    """HOST array of device pointers (ctypes) from a sequence of tensors / addresses, or None."""
    if images is None:
        return None, 0
    if isinstance(images, ctypes.Array):
        return images, len(images)
    vals = [_ptr(a) or 0 for a in images]
    return (ctypes.c_void_p * len(vals))(*vals), len(vals)


def iqa_fused_batch(x_ptrs_host, y_ptrs_host, n_pairs, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                    lisi_num=None, auglisi_num=None, out2=None, workspace=None, workspace_bytes=0,
                    stream=None) -> int:
    """x_ptrs_host / y_ptrs_host: sequences of n_pairs CUDA tensors (or addresses), or ready ctypes arrays."""
    xt, _ = _ptr_table(x_ptrs_host)
    yt, _ = _ptr_table(y_ptrs_host)
    return lib.iqa_fused_batch(xt, yt, int(n_pairs), int(N), int(N_T), C1, C2, C, D,
                               _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                               _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2),
                               _ptr(workspace), int(workspace_bytes), _stream(stream))


IQA_PLAN_GENERIC, IQA_PLAN_TMA_ANY, IQA_PLAN_TMA = 0, 2, 16


def iqa_query_plan(x, pixel_type, H, W, pitch, N_T, series=0) -> int:
    return int(lib.iqa_query_plan(_ptr(x), int(pixel_type), int(H), int(W), int(pitch), int(N_T), int(series)))


def iqa_debug_knob(name: str, value: int) -> int:
    """Test / tuning hook (include/iqa_tiles.h): sets a knob, returns its previous value (-1: unknown name)."""
    return int(lib.iqa_debug_knob(name.encode(), int(value)))


class knob:
    """``with binding.knob("IQA_FORCE_ANY", 1): ...`` -- sets a library knob for the block and restores it."""

    def __init__(self, name: str, value: int):
        self.name, self.value = name, int(value)

    def __enter__(self):
        self.prev = iqa_debug_knob(self.name, self.value)
        return self

    def __exit__(self, *a):
        iqa_debug_knob(self.name, self.prev)


def _pixel_types():
    import torch
    return {torch.float32: IQA_PIXEL_F32, torch.float64: IQA_PIXEL_F64, torch.float16: IQA_PIXEL_F16,
            torch.int16: IQA_PIXEL_I16, torch.int32: IQA_PIXEL_I32, torch.uint8: IQA_PIXEL_U8}


def iqa_query_plan_n(x, pixel_type, H, W, pitch, N_T, series=0, n_cmp=0) -> int:
    return lib.iqa_query_plan_n(_ptr(x), int(pixel_type), int(H), int(W), int(pitch), int(N_T), int(series), int(n_cmp))


def plan_name(x, N_T, series=False, n=0) -> str:
    """Which kernel a call on the CUDA tensor ``x`` would take: 'tma:c<k>' (tma_kernel), 'tma_any' (any_kernel)
    or 'generic'.  ``n``: pairs / comparisons of the call (0: a job large enough to fill the GPU)."""
    with _device_of(x.device):
        p = iqa_query_plan_n(x, _pixel_types()[x.dtype], x.shape[0], x.shape[1], x.stride(0), N_T, 1 if series else 0, n)
    return f"tma:c{p - IQA_PLAN_TMA}" if p >= IQA_PLAN_TMA else {0: "generic", 2: "tma_any"}.get(p, "invalid")


def iqa_workspace_bytes_2d(H: int, W: int, N_T: int) -> int:
    return int(lib.iqa_workspace_bytes_2d(int(H), int(W), int(N_T)))


def iqa_fused_tiles_2d(x, y, H, W, pitch_x, pitch_y, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                       lisi_num=None, auglisi_num=None, workspace=None, workspace_bytes=0, stream=None) -> int:
    return lib.iqa_fused_tiles_2d(_ptr(x), _ptr(y), int(H), int(W), int(pitch_x), int(pitch_y), int(N_T),
                                  C1, C2, C, D, _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                  _ptr(lisi_num), _ptr(auglisi_num), _ptr(workspace), int(workspace_bytes),
                                  _stream(stream))


def iqa_fused_tiles_2d_typed(x, y, pixel_type, H, W, pitch_x, pitch_y, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                             lisi_num=None, auglisi_num=None, workspace=None, workspace_bytes=0, stream=None) -> int:
    return lib.iqa_fused_tiles_2d_typed(_ptr(x), _ptr(y), int(pixel_type), int(H), int(W), int(pitch_x), int(pitch_y),
                                        int(N_T), C1, C2, C, D, _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                        _ptr(lisi_num), _ptr(auglisi_num), _ptr(workspace), int(workspace_bytes),
                                        _stream(stream))


def iqa_fused_batch_2d(x_ptrs_host, y_ptrs_host, n_pairs, H, W, pitch, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                       lisi_num=None, auglisi_num=None, out2=None, workspace=None, workspace_bytes=0,
                       stream=None) -> int:
    xt, _ = _ptr_table(x_ptrs_host)
    yt, _ = _ptr_table(y_ptrs_host)
    return lib.iqa_fused_batch_2d(xt, yt, int(n_pairs), int(H), int(W), int(pitch), int(N_T), C1, C2, C, D,
                                  _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), _ptr(lisi_num),
                                  _ptr(auglisi_num), _ptr(out2), _ptr(workspace), int(workspace_bytes), _stream(stream))


def iqa_series_tiles_2d(img_ptrs_host, n_images, mode, H, W, pitch, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                        lisi_num=None, auglisi_num=None, out2=None, workspace=None, workspace_bytes=0,
                        stream=None) -> int:
    it, _ = _ptr_table(img_ptrs_host)
    return lib.iqa_series_tiles_2d(it, int(n_images), int(mode), int(H), int(W), int(pitch), int(N_T), C1, C2, C, D,
                                   _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), _ptr(lisi_num),
                                   _ptr(auglisi_num), _ptr(out2), _ptr(workspace), int(workspace_bytes), _stream(stream))


def iqa_fused_batch_2d_typed(x_ptrs_host, y_ptrs_host, n_pairs, pixel_type, H, W, pitch, N_T, C1, C2, C, D,
                             lisi, auglisi, sum_x, sum_y, lisi_num=None, auglisi_num=None, out2=None,
                             workspace=None, workspace_bytes=0, stream=None) -> int:
    xt, _ = _ptr_table(x_ptrs_host)
    yt, _ = _ptr_table(y_ptrs_host)
    return lib.iqa_fused_batch_2d_typed(xt, yt, int(n_pairs), int(pixel_type), int(H), int(W), int(pitch), int(N_T),
                                        C1, C2, C, D, _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                        _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2), _ptr(workspace),
                                        int(workspace_bytes), _stream(stream))


def iqa_series_tiles_2d_typed(img_ptrs_host, n_images, mode, pixel_type, H, W, pitch, N_T, C1, C2, C, D,
                              lisi, auglisi, sum_x, sum_y, lisi_num=None, auglisi_num=None, out2=None,
                              workspace=None, workspace_bytes=0, stream=None) -> int:
    it, _ = _ptr_table(img_ptrs_host)
    return lib.iqa_series_tiles_2d_typed(it, int(n_images), int(mode), int(pixel_type), int(H), int(W), int(pitch),
                                         int(N_T), C1, C2, C, D, _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                         _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2), _ptr(workspace),
                                         int(workspace_bytes), _stream(stream))


def iqa_series_workspace_bytes(n_images: int, N: int, N_T: int) -> int:
    return int(lib.iqa_series_workspace_bytes(int(n_images), int(N), int(N_T)))


def iqa_series_tiles(img_ptrs_host, n_images, mode, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                     lisi_num=None, auglisi_num=None, out2=None, workspace=None, workspace_bytes=0,
                     stream=None) -> int:
    """img_ptrs_host: sequence of n_images CUDA tensors (or addresses), or a ready ctypes array."""
    it, _ = _ptr_table(img_ptrs_host)
    return lib.iqa_series_tiles(it, int(n_images), int(mode), int(N), int(N_T), C1, C2, C, D,
                                _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2),
                                _ptr(workspace), int(workspace_bytes), _stream(stream))


IQA_FIND_LISI, IQA_FIND_AUGLISI = 0, 1


def iqa_series_find(img_ptrs_host, n_images, mode, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                    lisi_num, auglisi_num, out2, workspace, workspace_bytes,
                    index, k, bottom_idx, bottom_val, threshold, below_idx, capacity, below_counts, stream=None) -> int:
    it, _ = _ptr_table(img_ptrs_host)
    return lib.iqa_series_find(it, int(n_images), int(mode), int(N), int(N_T), C1, C2, C, D,
                               _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                               _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2), _ptr(workspace), int(workspace_bytes),
                               int(index), int(k), _ptr(bottom_idx), _ptr(bottom_val), float(threshold),
                               _ptr(below_idx), int(capacity), _ptr(below_counts), _stream(stream))


def iqa_series_find_2d_typed(img_ptrs_host, n_images, mode, pixel_type, H, W, pitch, N_T, C1, C2, C, D,
                             lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num, out2, workspace, workspace_bytes,
                             index, k, bottom_idx, bottom_val, threshold, below_idx, capacity, below_counts,
                             stream=None) -> int:
    it, _ = _ptr_table(img_ptrs_host)
    return lib.iqa_series_find_2d_typed(it, int(n_images), int(mode), int(pixel_type), int(H), int(W), int(pitch), int(N_T),
                                        C1, C2, C, D, _ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y),
                                        _ptr(lisi_num), _ptr(auglisi_num), _ptr(out2), _ptr(workspace),
                                        int(workspace_bytes), int(index), int(k), _ptr(bottom_idx), _ptr(bottom_val),
                                        float(threshold), _ptr(below_idx), int(capacity), _ptr(below_counts),
                                        _stream(stream))


def iqa_tiles_below(values, n_tiles, n_maps, threshold, indices, capacity, counts, stream=None) -> int:
    return lib.iqa_tiles_below(_ptr(values), int(n_tiles), int(n_maps), threshold, _ptr(indices), int(capacity),
                               _ptr(counts), _stream(stream))


def iqa_tiles_bottom_k(values, n_tiles, n_maps, k, indices, vals=None, stream=None) -> int:
    return lib.iqa_tiles_bottom_k(_ptr(values), int(n_tiles), int(n_maps), int(k), _ptr(indices), _ptr(vals),
                                  _stream(stream))


def iqa_aggregate(lisi, auglisi, sum_x, sum_y, n_tiles, C2, C, out2, stream=None) -> int:
    return lib.iqa_aggregate(_ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), int(n_tiles),
                             C2, C, _ptr(out2), _stream(stream))


def iqa_aggregate_partial(lisi, auglisi, sum_x, sum_y, n_tiles, C2, C, sums4, stream=None) -> int:
    return lib.iqa_aggregate_partial(_ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), int(n_tiles),
                                     C2, C, _ptr(sums4), _stream(stream))


def iqa_aggregate_finish(sums4, n_tiles_total, C2, C, out2, stream=None) -> int:
    return lib.iqa_aggregate_finish(_ptr(sums4), int(n_tiles_total), C2, C, _ptr(out2), _stream(stream))


def iqa_merge_tiles(lisi, auglisi, sum_x, sum_y, nt, g, C2, C,
                    lisi_out, auglisi_out, sum_x_out, sum_y_out, stream=None) -> int:
    return lib.iqa_merge_tiles(_ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), int(nt), int(g),
                               C2, C, _ptr(lisi_out), _ptr(auglisi_out), _ptr(sum_x_out),
                               _ptr(sum_y_out), _stream(stream))


def iqa_fused_host(x_host, y_host, N, N_T, C1, C2, C, D, lisi_host, auglisi_host,
                   sum_x_host, sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream=None) -> int:
    return lib.iqa_fused_host(_ptr(x_host), _ptr(y_host), int(N), int(N_T), C1, C2, C, D,
                              _ptr(lisi_host), _ptr(auglisi_host), _ptr(sum_x_host), _ptr(sum_y_host),
                              _ptr(out2_host), _ptr(dev_scratch), int(dev_scratch_bytes), _stream(stream))


def iqa_fused_host_async(x_host, y_host, N, N_T, C1, C2, C, D, lisi_host, auglisi_host,
                         sum_x_host, sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream=None) -> int:
    return lib.iqa_fused_host_async(_ptr(x_host), _ptr(y_host), int(N), int(N_T), C1, C2, C, D,
                                    _ptr(lisi_host), _ptr(auglisi_host), _ptr(sum_x_host), _ptr(sum_y_host),
                                    _ptr(out2_host), _ptr(dev_scratch), int(dev_scratch_bytes), _stream(stream))


def iqa_host_scratch_bytes_typed(N: int, N_T: int, pixel_type: int) -> int:
    return int(lib.iqa_host_scratch_bytes_typed(int(N), int(N_T), int(pixel_type)))


def iqa_fused_host_typed(x_host, y_host, pixel_type, N, N_T, C1, C2, C, D, lisi_host, auglisi_host,
                         sum_x_host, sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream=None) -> int:
    return lib.iqa_fused_host_typed(_ptr(x_host), _ptr(y_host), int(pixel_type), int(N), int(N_T), C1, C2, C, D,
                                    _ptr(lisi_host), _ptr(auglisi_host), _ptr(sum_x_host), _ptr(sum_y_host),
                                    _ptr(out2_host), _ptr(dev_scratch), int(dev_scratch_bytes), _stream(stream))


def iqa_fused_host_typed_async(x_host, y_host, pixel_type, N, N_T, C1, C2, C, D, lisi_host, auglisi_host,
                               sum_x_host, sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream=None) -> int:
    return lib.iqa_fused_host_typed_async(_ptr(x_host), _ptr(y_host), int(pixel_type), int(N), int(N_T), C1, C2, C, D,
                                          _ptr(lisi_host), _ptr(auglisi_host), _ptr(sum_x_host), _ptr(sum_y_host),
                                          _ptr(out2_host), _ptr(dev_scratch), int(dev_scratch_bytes), _stream(stream))


# ----------------------------------------------------------------------------- convenience
def _check_images(x, y):
    import torch
    if not (isinstance(x, torch.Tensor) and isinstance(y, torch.Tensor)):
        raise TypeError("x and y must be torch CUDA tensors")
    if not (x.is_cuda and y.is_cuda):
        raise ValueError("x and y must live on a CUDA device (no CPU fallback)")
    if x.dtype != torch.float32 or y.dtype != torch.float32:
        raise TypeError("x and y must be float32")
    if x.dim() != 2 or x.shape[0] != x.shape[1] or x.shape != y.shape:
        raise ValueError("x and y must be equally sized square 2-D images")
    if not (x.is_contiguous() and y.is_contiguous()):
        raise ValueError("x and y must be contiguous (row-major, no pitch)")
    return int(x.shape[0])


def make_workspace(N: int, N_T: int, device):
    """Device scratch for the *_tiles calls (None when none is needed)."""
    import torch
    nbytes = iqa_workspace_bytes(N, N_T)
    if nbytes == 0:
        return None, 0
    return torch.empty(nbytes, dtype=torch.uint8, device=device), nbytes


def fused_tiles(x, y, N_T, C1, C2, C, D, numerators: bool = False, workspace=None) -> dict:
    """Eqs. 1-2 per tile from one read of x and y.  Returns dict of (nt, nt) float32 CUDA
    tensors: lisi, auglisi, X, Y (+ L, A when ``numerators``)."""
    import torch
    N = _check_images(x, y)
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "fused_tiles")
    nt = N // N_T
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((nt, nt), dtype=torch.float32, device=x.device) for k in names}
    if workspace is None:
        workspace, _ = make_workspace(N, N_T, x.device)
    wsb = 0 if workspace is None else workspace.numel() * workspace.element_size()
    with _device_of(x.device):
        rc = iqa_fused_tiles(x, y, N, N_T, C1, C2, C, D, out["lisi"], out["auglisi"], out["X"], out["Y"],
                             out.get("L"), out.get("A"), workspace, wsb, _current_stream(x.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_fused_tiles")
    return out


def fused_tiles_static(x, y, N_T, C1, C2, C, D, out: dict) -> dict:
    """``fused_tiles`` for callers that may not allocate device memory: nothing is allocated here or in the
    library.  ``out`` holds the caller's own (nt, nt) float32 CUDA tensors ``lisi``, ``auglisi``, ``X``, ``Y`` and
    optionally ``L``, ``A``; the split-tile partial sums go to the library's built-in 1 MiB array
    (``IQA_STATIC_WORKSPACE_BYTES``; larger shapes raise ``IqaError`` with ``IQA_ERR_STATIC_LIMIT``).  All calls on
    a device share that array: keep them on one stream (overlapping calls race).  See include/iqa_tiles.h."""
    N = _check_images(x, y)
    with _device_of(x.device):
        rc = iqa_fused_tiles_static(x, y, N, N_T, C1, C2, C, D, out["lisi"], out["auglisi"], out["X"], out["Y"],
                                    out.get("L"), out.get("A"), _current_stream(x.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_fused_tiles_static")
    return out


def fused_batch(xs, ys, N_T, C1, C2, C, D, numerators: bool = False, aggregate: bool = True) -> dict:
    """The whole hot path over a batch of equally shaped pairs (lists of CUDA tensors).  Returns
    (P, nt, nt) float32 CUDA tensors lisi, auglisi, X, Y (+ L, A when ``numerators``) and, when
    ``aggregate``, ``whole`` of shape (P, 2): [LISI, augLISI] per pair (Eqs. 3-4)."""
    import torch
    if len(xs) != len(ys) or not xs:
        raise IqaError(IQA_ERR_SHAPE, "fused_batch")
    N = _check_images(xs[0], ys[0])
    for x, y in zip(xs, ys):
        if _check_images(x, y) != N or x.device != xs[0].device:
            raise ValueError("all pairs of a batch must have the same shape and device")
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "fused_batch")
    P, nt, dev = len(xs), N // N_T, xs[0].device
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((P, nt, nt), dtype=torch.float32, device=dev) for k in names}
    if aggregate:
        out["whole"] = torch.empty((P, 2), dtype=torch.float32, device=dev)
    nbytes = iqa_batch_workspace_bytes(P, N, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(dev):
        rc = iqa_fused_batch(xs, ys, P, N, N_T, C1, C2, C, D, out["lisi"], out["auglisi"], out["X"], out["Y"],
                             out.get("L"), out.get("A"), out.get("whole"), ws, nbytes, _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_fused_batch")
    return out


def fused_tiles_2d(x, y, N_T, C1, C2, C, D, numerators: bool = False) -> dict:
    """Eqs. 1-2 per tile of two H x W CUDA tensors with EDGE TILES; pixel types float32
    (TMA kernel), float64, float16, int16, int32, uint8 (generic kernels).  x and y
    may be row-pitched views (``stride(1) == 1``, e.g. a window ``big[r0:r1, c0:c1]``); nothing is copied.
    Returns dict of (ceil(H/N_T), ceil(W/N_T)) float32 CUDA tensors: lisi, auglisi, X, Y (+ L, A)."""
    import torch
    ptypes = _pixel_types()
    for t in (x, y):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype in ptypes and t.dim() == 2):
            raise TypeError("x and y must be 2-D CUDA tensors of a supported pixel type (no CPU fallback)")
        if t.dtype != x.dtype:
            raise TypeError("x and y must share their pixel type")
        if t.stride(1) != 1 or t.stride(0) < t.shape[1]:
            raise ValueError("rows must be contiguous (stride(1) == 1) and must not overlap")
    if x.shape != y.shape or x.device != y.device:
        raise ValueError("x and y must have the same shape and device")
    if N_T <= 0:
        raise IqaError(IQA_ERR_SHAPE, "fused_tiles_2d")
    H, W = int(x.shape[0]), int(x.shape[1])
    nty, ntx = -(-H // N_T), -(-W // N_T)
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((nty, ntx), dtype=torch.float32, device=x.device) for k in names}
    nbytes = iqa_workspace_bytes_2d(H, W, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=x.device) if nbytes else None
    with _device_of(x.device):
        rc = iqa_fused_tiles_2d_typed(x, y, ptypes[x.dtype], H, W, x.stride(0), y.stride(0), N_T, C1, C2, C, D,
                                      out["lisi"], out["auglisi"], out["X"], out["Y"], out.get("L"), out.get("A"),
                                      ws, nbytes, _current_stream(x.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_fused_tiles_2d_typed")
    return out


def _check_2d_list(images):
    """Shape, common row pitch and pixel type (IQA_PIXEL_*) of the images of a batch / series call."""
    import torch
    ptypes = _pixel_types()
    H, W = int(images[0].shape[0]), int(images[0].shape[1])
    pitch = int(images[0].stride(0))
    for t in images:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype in ptypes and t.dim() == 2):
            raise TypeError("images must be 2-D CUDA tensors of a supported pixel type (no CPU fallback)")
        if (tuple(t.shape) != (H, W) or t.stride(1) != 1 or int(t.stride(0)) != pitch or t.device != images[0].device
                or t.dtype != images[0].dtype):
            raise ValueError("all images of a call must share shape, row pitch, pixel type and device")
    return H, W, pitch, ptypes[images[0].dtype]


def series_tiles_2d(images, mode, N_T, C1, C2, C, D, numerators: bool = False, aggregate: bool = True) -> dict:
    """``series_tiles`` for H x W images with a common row pitch and edge tiles (SURVEY.md 8(f)-2 + 8(f)-4)."""
    import torch
    if mode not in SERIES_MODES:
        raise ValueError(f"mode must be one of {tuple(SERIES_MODES)}")
    if len(images) < 2 or N_T <= 0:
        raise IqaError(IQA_ERR_SHAPE, "series_tiles_2d")
    H, W, pitch, ptype = _check_2d_list(images)
    K, nty, ntx, dev = len(images) - 1, -(-H // N_T), -(-W // N_T), images[0].device
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((K, nty, ntx), dtype=torch.float32, device=dev) for k in names}
    if aggregate:
        out["whole"] = torch.empty((K, 2), dtype=torch.float32, device=dev)
    nbytes = K * iqa_workspace_bytes_2d(H, W, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(images[0]):
        rc = iqa_series_tiles_2d_typed(images, len(images), SERIES_MODES[mode], ptype, H, W, pitch, N_T, C1, C2, C, D,
                                       out["lisi"], out["auglisi"], out["X"], out["Y"], out.get("L"), out.get("A"),
                                       out.get("whole"), ws, nbytes, _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_series_tiles_2d_typed")
    return out


def fused_batch_2d(xs, ys, N_T, C1, C2, C, D, numerators: bool = False, aggregate: bool = True) -> dict:
    """``fused_batch`` for H x W images with a common row pitch and edge tiles."""
    import torch
    if len(xs) != len(ys) or not xs or N_T <= 0:
        raise IqaError(IQA_ERR_SHAPE, "fused_batch_2d")
    H, W, pitch, ptype = _check_2d_list(list(xs) + list(ys))
    P, nty, ntx, dev = len(xs), -(-H // N_T), -(-W // N_T), xs[0].device
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((P, nty, ntx), dtype=torch.float32, device=dev) for k in names}
    if aggregate:
        out["whole"] = torch.empty((P, 2), dtype=torch.float32, device=dev)
    nbytes = P * iqa_workspace_bytes_2d(H, W, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(xs[0]):
        rc = iqa_fused_batch_2d_typed(xs, ys, P, ptype, H, W, pitch, N_T, C1, C2, C, D, out["lisi"], out["auglisi"],
                                      out["X"], out["Y"], out.get("L"), out.get("A"), out.get("whole"), ws, nbytes,
                                      _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_fused_batch_2d_typed")
    return out


def series_tiles(images, mode, N_T, C1, C2, C, D, numerators: bool = False, aggregate: bool = True) -> dict:
    """Time series: K = len(images) - 1 comparisons, ``mode`` "reference"
    (I_0 vs I_k+1) or "consecutive" (I_k vs I_k+1).  Returns (K, nt, nt) float32 CUDA tensors lisi,
    auglisi, X, Y (+ L, A when ``numerators``) and, when ``aggregate``, ``whole`` (K, 2)."""
    import torch
    if mode not in SERIES_MODES:
        raise ValueError(f"mode must be one of {tuple(SERIES_MODES)}")
    if len(images) < 2:
        raise IqaError(IQA_ERR_SHAPE, "series_tiles")
    N = _check_images(images[0], images[1])
    for im in images:
        if _check_images(images[0], im) != N or im.device != images[0].device:
            raise ValueError("all images of a series must have the same shape and device")
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "series_tiles")
    K, nt, dev = len(images) - 1, N // N_T, images[0].device
    names = ["lisi", "auglisi", "X", "Y"] + (["L", "A"] if numerators else [])
    out = {k: torch.empty((K, nt, nt), dtype=torch.float32, device=dev) for k in names}
    if aggregate:
        out["whole"] = torch.empty((K, 2), dtype=torch.float32, device=dev)
    nbytes = iqa_series_workspace_bytes(len(images), N, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(dev):
        rc = iqa_series_tiles(images, len(images), SERIES_MODES[mode], N, N_T, C1, C2, C, D,
                              out["lisi"], out["auglisi"], out["X"], out["Y"], out.get("L"), out.get("A"),
                              out.get("whole"), ws, nbytes, _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_series_tiles")
    return out


def _check_maps(values):
    import torch
    if not (isinstance(values, torch.Tensor) and values.is_cuda and values.dtype == torch.float32
            and values.is_contiguous()):
        raise TypeError("values must be a contiguous float32 CUDA tensor (no CPU fallback)")
    if values.dim() == 2:                       # one (nt, nt) matrix
        return 1, values.numel()
    if values.dim() == 3:                       # (n_maps, nt, nt)
        return int(values.shape[0]), int(values.shape[1] * values.shape[2])
    raise ValueError("values must be (nt, nt) or (n_maps, nt, nt)")


def tiles_below(values, threshold, capacity=None):
    """Candidate tiles with value < threshold.  Returns (indices, counts): int32 CUDA
    tensors (n_maps, capacity) -- the first ``counts[m]`` entries of row m are valid, ascending -- and (n_maps,)."""
    import torch
    n_maps, n = _check_maps(values)
    capacity = n if capacity is None else int(capacity)
    idx = torch.full((n_maps, capacity), -1, dtype=torch.int32, device=values.device)
    cnt = torch.empty(n_maps, dtype=torch.int32, device=values.device)
    with _device_of(values.device):
        rc = iqa_tiles_below(values, n, n_maps, float(threshold), idx, capacity, cnt, _current_stream(values.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_tiles_below")
    return idx, cnt


def tiles_bottom_k(values, k):
    """The k tiles of lowest value per matrix, ascending by (value, index).  Returns (indices int32
    (n_maps, k), vals float32 (n_maps, k)) CUDA tensors."""
    import torch
    n_maps, n = _check_maps(values)
    idx = torch.empty((n_maps, k), dtype=torch.int32, device=values.device)
    val = torch.empty((n_maps, k), dtype=torch.float32, device=values.device)
    with _device_of(values.device):
        rc = iqa_tiles_bottom_k(values, n, n_maps, k, idx, val, _current_stream(values.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_tiles_bottom_k")
    return idx, val


def find_transients(images, mode, N_T, C1, C2, C, D, k: int = 16, index: str = "auglisi", threshold=None,
                    capacity=None) -> dict:
    """The finder end to end on the device in ONE library call (``iqa_series_find``): the K
    comparisons of a time series, then for every comparison the ``k`` tiles of lowest ``index`` ("auglisi" or "lisi";
    low = dissimilar) and, with ``threshold``, the tiles below it.  Returns the series outputs plus
    ``candidates`` (int32 (K, k) tile indices t = ty * nt + tx, ascending by (value, index)), ``candidate_values``
    (K, k) and, with ``threshold``, ``below`` (int32 (K, capacity), ascending) and ``below_counts`` (K,)."""
    import torch
    if index not in ("auglisi", "lisi"):
        raise ValueError("index must be 'auglisi' or 'lisi'")
    if mode not in SERIES_MODES:
        raise ValueError(f"mode must be one of {tuple(SERIES_MODES)}")
    if len(images) < 2:
        raise IqaError(IQA_ERR_SHAPE, "find_transients")
    N = _check_images(images[0], images[1])
    for im in images:
        if _check_images(images[0], im) != N or im.device != images[0].device:
            raise ValueError("all images of a series must have the same shape and device")
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "find_transients")
    K, nt, dev = len(images) - 1, N // N_T, images[0].device
    out = {nm: torch.empty((K, nt, nt), dtype=torch.float32, device=dev) for nm in ("lisi", "auglisi", "X", "Y")}
    out["whole"] = torch.empty((K, 2), dtype=torch.float32, device=dev)
    out["candidates"] = torch.empty((K, k), dtype=torch.int32, device=dev)
    out["candidate_values"] = torch.empty((K, k), dtype=torch.float32, device=dev)
    cap = 0
    if threshold is not None:
        cap = nt * nt if capacity is None else int(capacity)
        out["below"] = torch.full((K, cap), -1, dtype=torch.int32, device=dev)
        out["below_counts"] = torch.empty(K, dtype=torch.int32, device=dev)
    nbytes = iqa_series_workspace_bytes(len(images), N, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(dev):
        rc = iqa_series_find(images, len(images), SERIES_MODES[mode], N, N_T, C1, C2, C, D,
                             out["lisi"], out["auglisi"], out["X"], out["Y"], None, None, out["whole"], ws, nbytes,
                             IQA_FIND_AUGLISI if index == "auglisi" else IQA_FIND_LISI, k,
                             out["candidates"], out["candidate_values"],
                             0.0 if threshold is None else float(threshold), out.get("below"), cap,
                             out.get("below_counts"), _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_series_find")
    return out


def find_transients_2d(images, mode, N_T, C1, C2, C, D, k: int = 16, index: str = "auglisi", threshold=None,
                       capacity=None) -> dict:
    """``find_transients`` for H x W images of any supported pixel type with a common row pitch and edge tiles
    (``iqa_series_find_2d_typed``): the series outputs as (K, nty, ntx) tensors plus the candidate lists, tile index
    t = ty * ntx + tx."""
    import torch
    if index not in ("auglisi", "lisi"):
        raise ValueError("index must be 'auglisi' or 'lisi'")
    if mode not in SERIES_MODES:
        raise ValueError(f"mode must be one of {tuple(SERIES_MODES)}")
    if len(images) < 2 or N_T <= 0:
        raise IqaError(IQA_ERR_SHAPE, "find_transients_2d")
    H, W, pitch, ptype = _check_2d_list(images)
    K, nty, ntx, dev = len(images) - 1, -(-H // N_T), -(-W // N_T), images[0].device
    out = {nm: torch.empty((K, nty, ntx), dtype=torch.float32, device=dev) for nm in ("lisi", "auglisi", "X", "Y")}
    out["whole"] = torch.empty((K, 2), dtype=torch.float32, device=dev)
    out["candidates"] = torch.empty((K, k), dtype=torch.int32, device=dev)
    out["candidate_values"] = torch.empty((K, k), dtype=torch.float32, device=dev)
    cap = 0
    if threshold is not None:
        cap = nty * ntx if capacity is None else int(capacity)
        out["below"] = torch.full((K, cap), -1, dtype=torch.int32, device=dev)
        out["below_counts"] = torch.empty(K, dtype=torch.int32, device=dev)
    nbytes = K * iqa_workspace_bytes_2d(H, W, N_T)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev) if nbytes else None
    with _device_of(images[0]):
        rc = iqa_series_find_2d_typed(images, len(images), SERIES_MODES[mode], ptype, H, W, pitch, N_T, C1, C2, C, D,
                                      out["lisi"], out["auglisi"], out["X"], out["Y"], None, None, out["whole"], ws,
                                      nbytes, IQA_FIND_AUGLISI if index == "auglisi" else IQA_FIND_LISI, k,
                                      out["candidates"], out["candidate_values"],
                                      0.0 if threshold is None else float(threshold), out.get("below"), cap,
                                      out.get("below_counts"), _current_stream(dev))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_series_find_2d_typed")
    return out


def lisi_tiles(x, y, N_T, C1, C2, D, workspace=None):
    import torch
    N = _check_images(x, y)
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "lisi_tiles")
    nt = N // N_T
    out = torch.empty((nt, nt), dtype=torch.float32, device=x.device)
    if workspace is None:
        workspace, _ = make_workspace(N, N_T, x.device)
    wsb = 0 if workspace is None else workspace.numel() * workspace.element_size()
    with _device_of(x.device):
        rc = iqa_lisi_tiles(x, y, N, N_T, C1, C2, D, out, workspace, wsb, _current_stream(x.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_lisi_tiles")
    return out


def auglisi_tiles(x, y, N_T, C, workspace=None):
    import torch
    N = _check_images(x, y)
    if N_T <= 0 or N % N_T:
        raise IqaError(IQA_ERR_SHAPE, "auglisi_tiles")
    nt = N // N_T
    out = torch.empty((nt, nt), dtype=torch.float32, device=x.device)
    if workspace is None:
        workspace, _ = make_workspace(N, N_T, x.device)
    wsb = 0 if workspace is None else workspace.numel() * workspace.element_size()
    with _device_of(x.device):
        rc = iqa_auglisi_tiles(x, y, N, N_T, C, out, workspace, wsb, _current_stream(x.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_auglisi_tiles")
    return out


def aggregate(lisi, auglisi, X, Y, C2, C, out2=None):
    """Eqs. 3-4 over all given tiles -> float32 CUDA tensor [LISI, augLISI]."""
    import torch
    n = lisi.numel()
    if out2 is None:
        out2 = torch.empty(2, dtype=torch.float32, device=lisi.device)
    with _device_of(lisi.device):
        rc = iqa_aggregate(lisi, auglisi, X, Y, n, C2, C, out2, _current_stream(lisi.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_aggregate")
    return out2


def aggregate_partial(lisi, auglisi, X, Y, C2, C):
    """The four double sums of Eqs. 3-4 over the given tiles (one band of a sharded image) -> float64 CUDA tensor [4]."""
    import torch
    sums4 = torch.empty(4, dtype=torch.float64, device=lisi.device)
    with _device_of(lisi.device):
        rc = iqa_aggregate_partial(lisi, auglisi, X, Y, lisi.numel(), C2, C, sums4, _current_stream(lisi.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_aggregate_partial")
    return sums4


def aggregate_finish(sums4, n_tiles_total, C2, C):
    """Eqs. 3-4 from the all-reduced sums of every band -> float32 CUDA tensor [LISI, augLISI]."""
    import torch
    out2 = torch.empty(2, dtype=torch.float32, device=sums4.device)
    with _device_of(sums4.device):
        rc = iqa_aggregate_finish(sums4, n_tiles_total, C2, C, out2, _current_stream(sums4.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_aggregate_finish")
    return out2


def iqa_merge_tiles_batch(lisi, auglisi, sum_x, sum_y, nt, g, n_maps, C2, C,
                          lisi_out, auglisi_out, sum_x_out, sum_y_out, stream=None) -> int:
    return lib.iqa_merge_tiles_batch(_ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), int(nt), int(g), int(n_maps),
                                     C2, C, _ptr(lisi_out), _ptr(auglisi_out), _ptr(sum_x_out),
                                     _ptr(sum_y_out), _stream(stream))


def merge_tiles(lisi, auglisi, X, Y, g, C2, C) -> dict:
    """Eqs. 3-4 on every g x g block of the (nt, nt) matrices -> (nt/g, nt/g) matrices; (n_maps, nt, nt)
    stacks (the comparisons of a series, the pairs of a batch) are merged map by map in one launch."""
    import torch
    batched = lisi.dim() == 3
    nt = int(lisi.shape[-1])
    n_maps = int(lisi.shape[0]) if batched else 1
    if g <= 0 or nt % g or lisi.shape[-2] != nt or not lisi.is_contiguous():
        raise IqaError(IQA_ERR_SHAPE, "merge_tiles")
    no = nt // g
    shape = (n_maps, no, no) if batched else (no, no)
    out = {k: torch.empty(shape, dtype=torch.float32, device=lisi.device)
           for k in ("lisi", "auglisi", "X", "Y")}
    with _device_of(lisi.device):
        rc = iqa_merge_tiles_batch(lisi, auglisi, X, Y, nt, g, n_maps, C2, C, out["lisi"], out["auglisi"], out["X"],
                                   out["Y"], _current_stream(lisi.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_merge_tiles_batch")
    return out


def iqa_pyramid_levels(nty: int, ntx: int) -> int:
    return int(lib.iqa_pyramid_levels(int(nty), int(ntx)))


def iqa_pyramid_tiles(nty: int, ntx: int) -> int:
    return int(lib.iqa_pyramid_tiles(int(nty), int(ntx)))


def iqa_pyramid(lisi, auglisi, sum_x, sum_y, nty, ntx, n_maps, C2, C,
                lisi_out, auglisi_out, sum_x_out, sum_y_out, stream=None) -> int:
    return lib.iqa_pyramid(_ptr(lisi), _ptr(auglisi), _ptr(sum_x), _ptr(sum_y), int(nty), int(ntx), int(n_maps),
                           C2, C, _ptr(lisi_out), _ptr(auglisi_out), _ptr(sum_x_out), _ptr(sum_y_out), _stream(stream))


def pyramid(tiles: dict, C2, C) -> list:
    """all levels N_T, 2 N_T, 4 N_T, ... up to the whole image (a 1 x 1 matrix) from ONE ``iqa_pyramid`` launch.
    ``tiles``: dict of (nty, ntx) or (n_maps, nty, ntx) matrices lisi, auglisi, X, Y (any rectangle).  Returns
    ``[tiles, level 1, level 2, ...]``; level j holds (ceil(nty / 2^j), ceil(ntx / 2^j)) matrices (views of one buffer)."""
    import torch
    lisi = tiles["lisi"]
    batched = lisi.dim() == 3
    nty, ntx = int(lisi.shape[-2]), int(lisi.shape[-1])
    n_maps = int(lisi.shape[0]) if batched else 1
    src = [tiles[k] for k in ("lisi", "auglisi", "X", "Y")]
    if not all(t.is_contiguous() and t.dtype == torch.float32 and t.is_cuda for t in src):
        raise TypeError("pyramid needs contiguous float32 CUDA matrices (no CPU fallback)")
    L, total = iqa_pyramid_levels(nty, ntx), iqa_pyramid_tiles(nty, ntx)
    levels = [tiles]
    if L == 0:
        return levels
    out = [torch.empty((n_maps, total), dtype=torch.float32, device=lisi.device) for _ in range(4)]
    with _device_of(lisi.device):
        rc = iqa_pyramid(*src, nty, ntx, n_maps, C2, C, *out, _current_stream(lisi.device))
    if rc != IQA_OK:
        raise IqaError(rc, "iqa_pyramid")
    off = 0
    for j in range(1, L + 1):
        ny, nx = -(-nty // (1 << j)), -(-ntx // (1 << j))
        shape = (n_maps, ny, nx) if batched else (ny, nx)
        levels.append({k: (o[:, off:off + ny * nx] if batched else o[0, off:off + ny * nx]).reshape(shape)
                       for k, o in zip(("lisi", "auglisi", "X", "Y"), out)})
        off += ny * nx
    return levels


class HostRunner:
    """Reusable state for ``iqa_fused_host``: the device scratch and pinned result buffers."""

    def __init__(self, N: int, N_T: int, device="cuda:0", pixel_type: int = IQA_PIXEL_F32):
        import torch
        self.N, self.N_T = int(N), int(N_T)
        self.nt = self.N // self.N_T
        self.device = torch.device(device)
        self.pixel_type = int(pixel_type)        # IQA_PIXEL_*: the host images are uploaded and computed on as they are
        self.esize = {IQA_PIXEL_F32: 4, IQA_PIXEL_F64: 8, IQA_PIXEL_F16: 2, IQA_PIXEL_I16: 2, IQA_PIXEL_I32: 4,
                      IQA_PIXEL_U8: 1}.get(self.pixel_type, 0)
        self.scratch_bytes = iqa_host_scratch_bytes_typed(N, N_T, self.pixel_type)
        if self.scratch_bytes == 0:
            raise IqaError(IQA_ERR_SHAPE, "HostRunner")
        self.scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device=self.device)
        mk = lambda *s: torch.empty(*s, dtype=torch.float32).pin_memory()
        self.out = {k: mk(self.nt, self.nt) for k in ("lisi", "auglisi", "X", "Y")}
        self.out2 = mk(2)

    @property
    def h2d_bytes(self) -> int:
        return 2 * self.esize * self.N * self.N

    @property
    def d2h_bytes(self) -> int:
        return 4 * 4 * self.nt * self.nt + 8

    def __call__(self, x_host, y_host, C1, C2, C, D):
        with _device_of(self.device):
            args = (self.N, self.N_T, C1, C2, C, D, self.out["lisi"], self.out["auglisi"], self.out["X"], self.out["Y"],
                    self.out2, self.scratch, self.scratch_bytes, _current_stream(self.device))
            rc = (iqa_fused_host(x_host, y_host, *args) if self.pixel_type == IQA_PIXEL_F32
                  else iqa_fused_host_typed(x_host, y_host, self.pixel_type, *args))
        if rc != IQA_OK:
            raise IqaError(rc, "iqa_fused_host")
        return self.out, self.out2


class HostPipeline:
    """``depth`` HostRunners on ``depth`` streams: ``submit`` enqueues one host pair with
    ``iqa_fused_host_async`` on the next stream (after waiting for that stream's previous pair) and returns
    the slot whose pinned outputs will hold the result; ``wait(slot)`` / ``drain()`` synchronise.  The upload
    of pair i+1 overlaps the kernels, downloads and launch gaps of pair i."""

    def __init__(self, N: int, N_T: int, device="cuda:0", depth: int = 2, pixel_type: int = IQA_PIXEL_F32):
        import torch
        self.runners = [HostRunner(N, N_T, device, pixel_type) for _ in range(depth)]
        self.streams = [torch.cuda.Stream(device=self.runners[0].device) for _ in range(depth)]
        self.next = 0

    def submit(self, x_host, y_host, C1, C2, C, D) -> int:
        slot = self.next
        self.next = (self.next + 1) % len(self.runners)
        r, st = self.runners[slot], self.streams[slot]
        st.synchronize()                         # the slot's previous pair is complete: its buffers are free
        with _device_of(r.device):
            args = (r.N, r.N_T, C1, C2, C, D, r.out["lisi"], r.out["auglisi"], r.out["X"], r.out["Y"], r.out2, r.scratch,
                    r.scratch_bytes, st)
            rc = (iqa_fused_host_async(x_host, y_host, *args) if r.pixel_type == IQA_PIXEL_F32
                  else iqa_fused_host_typed_async(x_host, y_host, r.pixel_type, *args))
        if rc != IQA_OK:
            raise IqaError(rc, "iqa_fused_host_async")
        return slot

    def wait(self, slot: int):
        self.streams[slot].synchronize()
        return self.runners[slot].out, self.runners[slot].out2

    def drain(self):
        for st in self.streams:
            st.synchronize()


def fused_host(x_host, y_host, N_T, C1, C2, C, D, device="cuda:0"):
    """One-shot host call (allocates scratch each time; use HostRunner in loops).  x_host, y_host: square numpy arrays
    or CPU tensors of one supported pixel type (float32, float64, float16, int16, int32, uint8)."""
    N = int(x_host.shape[0])
    names = {"float32": IQA_PIXEL_F32, "float64": IQA_PIXEL_F64, "float16": IQA_PIXEL_F16, "int16": IQA_PIXEL_I16,
             "int32": IQA_PIXEL_I32, "uint8": IQA_PIXEL_U8}
    dt = str(x_host.dtype).replace("torch.", "")
    if dt not in names or str(y_host.dtype).replace("torch.", "") != dt:
        raise TypeError("x_host and y_host must share one supported pixel type")
    r = HostRunner(N, N_T, device, names[dt])
    out, out2 = r(x_host, y_host, C1, C2, C, D)
    return {k: v.clone() for k, v in out.items()}, out2.clone()
